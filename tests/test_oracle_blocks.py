"""Pins of the block-finer-than-page oracle (-m "not gpu"; reading G28 in oracle/vx_oracle_blocks.py).

The oracle is a re-indexing: blocks become pages of a pool of blocks.  What fixes it: a hand-worked map of blocks to
(page, offset); the gather puts every token's key where the definition says; block = page is the page-level oracle bit
for bit; selecting both halves of every selected page reproduces the page-level attention; block envelopes nest inside
the page envelope and their union is the page envelope; budgets that cover every block give dense attention."""
from dataclasses import replace

import numpy as np
import pytest

from oracle import vx_oracle as vo
from oracle.vx_oracle_blocks import block_location, block_problem
from oracle.workload_io import _to_oracle_pages, oracle_step, to_oracle
from paper_2606_06453_b200.workloads import SPECS, make_workload


def wl(name="C2-small", page=32, block=16, **kw):
    return make_workload(replace(SPECS[name], page_size=page, block_size=block, batch=2, **kw))


def test_hand_worked_block_locations():
    # page 32, block 16: blocks 0, 1 in page 0 (offsets 0, 16), block 2 in page 1 ...; page 64, block 16: four per page
    assert [block_location(j, 16, 32) for j in range(5)] == [(0, 0), (0, 16), (1, 0), (1, 16), (2, 0)]
    assert [block_location(j, 16, 64) for j in (0, 3, 4, 7, 9)] == [(0, 0), (0, 48), (1, 0), (1, 48), (2, 16)]


@pytest.mark.parametrize("name,page,block", [("C2-small", 32, 16), ("C4-small", 64, 16)])
def test_the_gather_puts_every_token_where_the_definition_says(name, page, block):
    w = wl(name, page, block)
    s = w.spec
    q, pool, pt = _to_oracle_pages(w)
    bpool, bpt = block_problem(pool, pt, block, s.num_kv_heads, s.qk_dim, s.v_dim)
    bpp = page // block
    assert bpt.page_size == block and np.array_equal(bpt.page_indptr, pt.page_indptr * bpp)
    k = pool.k.reshape(-1)
    rng = np.random.default_rng(0)
    for _ in range(200):
        i = int(rng.integers(s.batch))
        t = int(rng.integers(int(pt.seq_lens[i])))                    # token t of request i
        h, c = int(rng.integers(s.num_kv_heads)), int(rng.integers(s.qk_dim))
        phys = int(pt.page_indices[pt.page_indptr[i] + t // page])
        want = k[phys * pool.stride_page + (t % page) * pool.stride_token + h * pool.stride_head + c]
        j = t // block
        lp, off = block_location(j, block, page)
        assert lp == t // page and off <= t % page < off + block
        pb = int(bpt.page_indices[bpt.page_indptr[i] + j])
        assert pb == phys * bpp + off // block                        # physical block id = page id * bpp + block in page
        got = bpool.k.reshape(-1)[pb * bpool.stride_page + (t % block) * bpool.stride_token + h * bpool.stride_head + c]
        assert got == want


@pytest.mark.parametrize("name", ["C2-small", "C4-small"])
def test_block_equal_to_page_is_the_page_level_oracle(name):
    w = make_workload(replace(SPECS[name], batch=2))
    a = oracle_step(w)
    b = oracle_step(replace(w, spec=replace(w.spec, block_size=w.spec.page_size)))
    q, pool, pt = _to_oracle_pages(w)
    s = w.spec
    bpool, bpt = block_problem(pool, pt, s.page_size, s.num_kv_heads, s.qk_dim, s.v_dim)       # the gather with bpp = 1
    c = vo.decode_step(q, bpool, bpt, vo.as_np(w.budget), w.max_budget, s.num_q_heads, s.num_kv_heads, s.qk_dim, s.v_dim,
                       s.sm_scale, s.n_sink, s.n_local)
    for key in ("scores", "sel_logical", "sel_phys", "sel_count", "out", "lse"):
        assert np.array_equal(a[key], b[key]) and np.array_equal(a[key], c[key]), key


def test_both_halves_of_a_page_are_the_page():
    w = wl()
    s = w.spec
    pw = replace(w, spec=replace(s, block_size=0))
    ref = oracle_step(pw)                                             # page-level selection and attention (page 32)
    sl, sc = ref["sel_logical"], ref["sel_count"]
    bl = np.full((s.batch, s.num_kv_heads, 2 * w.max_budget), -1, dtype=np.int32)
    for i in range(s.batch):
        nb = -(-int(w.seq_lens[i]) // 16)
        for h in range(s.num_kv_heads):
            blocks = [b for p in sl[i, h, :sc[i, h]] for b in (2 * p, 2 * p + 1) if b < nb]
            bl[i, h, :len(blocks)] = blocks
    bc = (bl >= 0).sum(-1).astype(np.int32)
    q, bpool, bpt = to_oracle(w)
    o, l = vo.sparse_attention(q, bpool, bpt, bl, bc, s.num_q_heads, s.num_kv_heads, s.qk_dim, s.v_dim, s.sm_scale)
    np.testing.assert_allclose(o, ref["out"], rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(l, ref["lse"], rtol=1e-13)


def test_block_envelopes_nest_in_the_page_envelope():
    w = wl()
    s = w.spec
    q, pool, pt = _to_oracle_pages(w)
    page_sum = vo.page_summary(pool, pt, s.num_kv_heads, s.qk_dim)
    _, bpool, bpt = to_oracle(w)
    blk_sum = vo.page_summary(bpool, bpt, s.num_kv_heads, s.qk_dim)
    for i in range(s.batch):
        n = int(pt.seq_lens[i])
        for lp in range(-(-n // 32)):
            phys = int(pt.page_indices[pt.page_indptr[i] + lp])
            halves = [2 * phys + u for u in range(2) if (2 * lp + u) * 16 < n]
            lo = np.min([blk_sum[b, :, 0] for b in halves], axis=0)
            hi = np.max([blk_sum[b, :, 1] for b in halves], axis=0)
            assert np.array_equal(lo, page_sum[phys, :, 0]) and np.array_equal(hi, page_sum[phys, :, 1])
            for b in halves:
                assert (blk_sum[b, :, 0] >= page_sum[phys, :, 0]).all() and (blk_sum[b, :, 1] <= page_sum[phys, :, 1]).all()


def test_budget_over_all_blocks_is_dense_attention():
    w = wl(budget=100000)
    s = w.spec
    ref = oracle_step(w)
    q, pool, pt = _to_oracle_pages(w)
    o, l = vo.dense_attention(q, pool, pt, s.num_q_heads, s.num_kv_heads, s.qk_dim, s.v_dim, s.sm_scale)
    nb = -(-vo.as_np(w.seq_lens) // 16)
    assert np.array_equal(ref["sel_count"], np.repeat(nb[:, None], s.num_kv_heads, 1))
    np.testing.assert_allclose(ref["out"], o, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(ref["lse"], l, rtol=1e-13)


def test_finer_blocks_spend_the_budget_in_blocks_and_keep_forced_blocks():
    w = wl()
    s = w.spec
    ref = oracle_step(w)
    nb = -(-vo.as_np(w.seq_lens) // 16)
    for i in range(s.batch):
        for h in range(s.num_kv_heads):
            sel = ref["sel_logical"][i, h, :ref["sel_count"][i, h]]
            assert len(sel) == min(int(w.budget[i]), nb[i])
            assert set(range(s.n_sink)) <= set(sel) and set(range(nb[i] - s.n_local, nb[i])) <= set(sel)
