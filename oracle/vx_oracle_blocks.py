"""Selection blocks finer than the physical page, for the oracle (test infrastructure only).

PAPER.md:518-519 (Listing 2: `block_size: 16` inside `page_size: 32`), :202 (cuda_mla "supporting ... finer blocks (down
to 16), so the block granularity can match the sparsity budget"), :85 (a block is b consecutive tokens).  The paper does
not say how blocks sit in pages; reading G28:

  G28  block_size b_s divides page_size b.  Request i has NB_i = ceil(n_i / b_s) blocks; logical block j covers the tokens
       [j b_s, min((j + 1) b_s, n_i)) -- b_s consecutive tokens that lie inside ONE physical page: logical page
       (j b_s) div b, token offset (j b_s) mod b.  Everything the method does per page it does per block: summaries
       (envelope of the block's valid tokens), scores, the budget and the forced sink / local counts (in blocks), the
       selection (ties to the lower logical block), attention over the tokens of the selected blocks.  With b_s = b
       this is the page-level method unchanged.
       Numbering used on both sides of the ABI: physical block id = physical page id * (b / b_s) + block within the page.

The oracle is the definition "a block is a page of b_s tokens": the pool is re-indexed (a pure gather, no arithmetic) into
a pool of blocks, the page table into a block table, and oracle/vx_oracle.c runs on that with page_size = b_s.
"""
import numpy as np

from oracle import vx_oracle as vo


def block_problem(pool: vo.Pool, pt: vo.PageTable, block_size: int, num_kv_heads: int, qk_dim: int, v_dim: int):
    """(Pool of blocks [N_pool * bpp, Hkv, b_s, d], PageTable of blocks with page_size = b_s).  Gathering only."""
    b = pt.page_size
    assert b % block_size == 0, "block_size must divide page_size"
    bpp = b // block_size

    def regather(a, width):
        if a is None:
            return None
        n = pool.num_pool_pages
        idx = (np.arange(n)[:, None, None, None] * pool.stride_page + np.arange(num_kv_heads)[None, :, None, None] * pool.stride_head
               + np.arange(b)[None, None, :, None] * pool.stride_token + np.arange(width)[None, None, None, :])
        flat = a.reshape(-1)[idx]                                   # [N, Hkv, b, width]
        blocks = flat.reshape(n, num_kv_heads, bpp, block_size, width).transpose(0, 2, 1, 3, 4)
        return np.ascontiguousarray(blocks.reshape(n * bpp, num_kv_heads, block_size, width))

    kv_shared = pool.v is None
    k = regather(pool.k, qk_dim)
    v = None if kv_shared else regather(pool.v, v_dim)
    bpool = vo.Pool(k=k, v=v, stride_page=num_kv_heads * block_size * qk_dim, stride_token=qk_dim,
                    stride_head=block_size * qk_dim, num_pool_pages=pool.num_pool_pages * bpp)
    if not kv_shared and v_dim != qk_dim:
        raise ValueError("separate V pools share K's strides: v_dim must equal qk_dim")
    indptr = pt.page_indptr.astype(np.int64) * bpp
    indices = (pt.page_indices.astype(np.int64)[:, None] * bpp + np.arange(bpp)[None, :]).reshape(-1)
    bpt = vo.PageTable(indptr.astype(np.int32), indices.astype(np.int32), pt.seq_lens, block_size)
    return bpool, bpt


def block_location(j: int, block_size: int, page_size: int):
    """(logical page, token offset inside the page) of logical block j (G28)"""
    return (j * block_size) // page_size, (j * block_size) % page_size
