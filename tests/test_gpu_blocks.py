"""Selection blocks finer than the page (-m gpu; NEXT-4 second half, PAPER.md:518-519 `block_size: 16` / `page_size: 32`,
:202 "finer blocks (down to 16)"; reading G28): vx_geom.block_size.  The caller's page table stays a PAGE table; summaries,
scores, budgets, forced counts and the selection are per BLOCK.  Against the block-level oracle (oracle/vx_oracle_blocks.py):
summaries bit-exact, scores 2e-5 of the score scale, selection by the comparator (physical BLOCK ids checked too),
attention within the bf16 tolerances, for GQA (block 16 in pages of 32 and 64: the mma decode kernel), MLA (block 16 in
pages of 64: the generic decode kernel), a ragged C5-like batch and an fp8 KV cache; block = page is the default path."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from oracle.workload_io import block_table, oracle_step
from tests.parity import check_attention, check_selection, oracle_attention_on

pytestmark = pytest.mark.gpu


def run(spec):
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload
    w = make_workload(spec, device="cuda:0")
    s = w.spec
    dev = w.q.device
    bpp = s.page_size // s.block_size if s.block_size else 1
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    assert summary.shape[0] == w.num_pool_pages * bpp
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    clean = summary.clone()
    out = torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev)
    lse = torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    sp = torch.full((s.batch, s.num_kv_heads, w.max_budget), -7, dtype=torch.int32, device=dev)
    sl, sc = torch.full_like(sp, -7), torch.full((s.batch, s.num_kv_heads), -7, dtype=torch.int32, device=dev)
    # poison the newest BLOCK's summary: the fused step must rebuild it (a1)
    indptr, indices = block_table(w)
    nb = -(-w.seq_lens.cpu().numpy() // (s.block_size or s.page_size))
    newest = torch.as_tensor(indices[indptr[:-1] + nb - 1], device=dev)
    summary[newest] = 0
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc, flags=vx.VX_STEP_UPDATE_SUMMARY)
    torch.cuda.synchronize()
    return vx, w, ctx, pool, pt, summary, clean, out, lse, sp, sl, sc, bpp


def spec_of(name, page, block, **kw):
    from paper_2606_06453_b200.workloads import SPECS, with_fp8
    fp8 = kw.pop("fp8", None)
    s = replace(SPECS[name], name=f"{name}-p{page}b{block}", page_size=page, block_size=block, **kw)
    return with_fp8(s, fp8) if fp8 else s


CASES = {
    "gqa-b16-p32": ("C2-small", 32, 16, {}),
    "gqa-b16-p64": ("C2-small", 64, 16, dict(seq_len=(2000, 4100))),
    "mla-b16-p64": ("C4-small", 64, 16, dict(budget=24)),
    "ragged-b16-p32": ("C5-small", 32, 16, {}),
    "gqa-b16-p32-fp8": ("C2-small", 32, 16, dict(fp8="e4m3")),
    "gqa-b32-p64-generic": ("C2-small", 64, 32, {}),
}


@pytest.mark.parametrize("case", list(CASES))
def test_blocks_finer_than_the_page_match_the_oracle(case):
    name, page, block, kw = CASES[case]
    vx, w, ctx, pool, pt, summary, clean, out, lse, sp, sl, sc, bpp = run(spec_of(name, page, block, **dict(kw)))
    s = w.spec
    ref = oracle_step(w)                                   # block-level oracle
    indptr, indices = block_table(w)
    nb = -(-w.seq_lens.cpu().numpy() // block)
    live = np.concatenate([indices[indptr[i]:indptr[i] + nb[i]] for i in range(s.batch)])
    got = clean.cpu()
    if s.kv_dtype:
        from oracle.vx_oracle_fp8 import dequantize
        got = dequantize(got.numpy(), s.kv_dtype, w.k_scale)
    else:
        got = got.float().numpy().astype(np.float64)
    assert np.array_equal(got[live], ref["summary"][live]), "block summaries differ from the oracle's"
    assert torch.equal(summary, clean), "the step rebuilds the newest block's summary, nothing else"
    total_blocks = w.total_pages * bpp
    scores = torch.empty(s.num_kv_heads, total_blocks, dtype=torch.float32, device="cuda:0")
    ctx.page_score(w.q, clean, pt, scores)
    torch.cuda.synchronize()
    g = scores.cpu().numpy().astype(np.float64) * (float(np.float32(w.k_scale)) if s.kv_dtype else 1.0)
    cols = np.concatenate([np.arange(indptr[i], indptr[i] + nb[i]) for i in range(s.batch)])
    assert np.abs(g[:, cols] - ref["scores"][:, cols]).max() <= 2e-5 * np.abs(ref["scores"][:, cols]).max()
    check_selection(w, sl.cpu().numpy(), sp.cpu().numpy(), sc.cpu().numpy(), ref, label=f"{case} fused step")
    sp2, sl2, sc2 = torch.full_like(sp, -7), torch.full_like(sl, -7), torch.full_like(sc, -7)
    ctx.topk_pages(scores, pt, w.budget, w.max_budget, sp2, sl2, sc2)
    torch.cuda.synchronize()
    assert torch.equal(sl, sl2) and torch.equal(sp, sp2) and torch.equal(sc, sc2)
    o_ref, l_ref = oracle_attention_on(w, sl.cpu().numpy(), sc.cpu().numpy())
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)
    out2, lse2 = torch.full_like(out, float("nan")), torch.full_like(lse, float("nan"))
    ctx.sparse_paged_decode(w.q, pool, pt, sp, sl, sc, w.max_budget, out2, lse2)
    torch.cuda.synchronize()
    check_attention(s.dtype, out2.float().cpu().numpy(), lse2.cpu().numpy(), o_ref, l_ref)
    ctx.close()


def test_block_equal_to_page_is_the_default_path_bit_for_bit():
    from paper_2606_06453_b200.workloads import SPECS
    a = run(SPECS["C2-small"])
    b = run(replace(SPECS["C2-small"], block_size=16))
    for x, y in zip(a[6:12], b[6:12]):                      # clean summaries, out, lse, sel_phys, sel_logical, sel_count
        assert torch.equal(x.view(torch.uint8) if x.dtype == torch.bfloat16 else x, y.view(torch.uint8) if y.dtype == torch.bfloat16 else y)
    a[2].close(); b[2].close()


def test_block_size_must_divide_the_page():
    import paper_2606_06453_b200 as vx
    kw = dict(dtype=torch.bfloat16, num_q_heads=32, num_kv_heads=8, qk_dim=128, v_dim=128, page_size=32, sm_scale=0.1,
              n_sink=1, n_local=2, max_batch=2, max_total_pages=64, max_pages_per_req=32, max_budget=8)
    vx.Context(block_size=16, **kw).close()
    for bad in (12, 64, -1):
        with pytest.raises(vx.VortexError):
            vx.Context(block_size=bad, **kw)
