"""GPU parity: every C-ABI call against the fp64 oracle on the same seeded inputs (-m gpu).

Sizes: the reduced variants of BASELINE.json's configs (several tiles, ragged tails, partial
last pages) where the oracle runs in seconds; full-size sampled parity is in test_gpu_fullsize.py.
"""
from dataclasses import replace

import os

import numpy as np
import pytest
import torch

from oracle import vx_oracle as vo
from oracle.workload_io import bf16_bits_to_f64, oracle_step, to_oracle
from tests.parity import check_attention, check_selection, oracle_attention_on

pytestmark = pytest.mark.gpu

SMALL = ["C1", "C2-small", "C3-small", "C4-small", "C5-small"]


def setup(name_or_spec):
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload
    w = make_workload(name_or_spec, device="cuda:0")
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    return vx, w, ctx, pool, pt


def outputs(w):
    s = w.spec
    dev = w.q.device
    return dict(out=torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev),
                lse=torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev),
                sel_phys=torch.full((s.batch, s.num_kv_heads, w.max_budget), -7, dtype=torch.int32, device=dev),
                sel_logical=torch.full((s.batch, s.num_kv_heads, w.max_budget), -7, dtype=torch.int32, device=dev),
                sel_count=torch.full((s.batch, s.num_kv_heads), -7, dtype=torch.int32, device=dev))


def build_summary(vx, w, ctx, pool, pt):
    summary = vx.alloc_summary(w)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    return summary


@pytest.mark.parametrize("name", SMALL)
def test_summary_bulk_matches_oracle_exactly(name):
    vx, w, ctx, pool, pt = setup(name)
    # poison the stale slots of partial last pages: they must not leak into the envelope
    n = w.seq_lens.cpu(); b = w.spec.page_size
    for i in range(w.spec.batch):
        r = int(n[i]) % b
        if r:
            phys = int(w.page_indices[int(w.page_indptr[i + 1]) - 1])
            w.k_pool[phys, :, r:, ::2] = 1e30
            w.k_pool[phys, :, r:, 1::2] = -1e30
    summary = build_summary(vx, w, ctx, pool, pt)
    torch.cuda.synchronize()
    _, opool, opt = to_oracle(w)
    ref = vo.page_summary(opool, opt, w.spec.num_kv_heads, w.spec.qk_dim)
    got = bf16_bits_to_f64(vo.as_np(summary))
    used = np.unique(opt.page_indices)
    assert np.array_equal(got[used], ref[used])
    unused = np.setdiff1d(np.arange(w.num_pool_pages), used)
    assert (got[unused] == 0).all()               # pages outside the table are not written


@pytest.mark.parametrize("name", ["C2-small", "C4-small"])
def test_summary_append_mode_touches_only_last_page(name):
    vx, w, ctx, pool, pt = setup(name)
    summary = build_summary(vx, w, ctx, pool, pt)
    before = summary.clone()
    # a new token arrives in every request: overwrite the newest slot, then append-update
    b = w.spec.page_size
    lastp = [int(w.page_indices[int(w.page_indptr[i + 1]) - 1]) for i in range(w.spec.batch)]
    for i, phys in enumerate(lastp):
        slot = (int(w.seq_lens[i]) - 1) % b
        w.k_pool[phys, :, slot] = 100.0
    ctx.page_summary_update(pool, pt, summary, first_new_pos=None)
    torch.cuda.synchronize()
    _, opool, opt = to_oracle(w)
    ref = vo.page_summary(opool, opt, w.spec.num_kv_heads, w.spec.qk_dim)
    got = bf16_bits_to_f64(vo.as_np(summary))
    used = np.unique(opt.page_indices)
    assert np.array_equal(got[used], ref[used])
    others = np.setdiff1d(np.arange(w.num_pool_pages), lastp)
    assert torch.equal(summary[others], before[others])
    # mid-sequence first_new_pos: only pages from that position on are rebuilt
    summary2 = before.clone()
    w.k_pool[lastp[0]] = 0.0
    fnp = (w.seq_lens - 1).clamp(min=0)
    ctx.page_summary_update(pool, pt, summary2, first_new_pos=fnp)
    torch.cuda.synchronize()
    assert torch.equal(summary2[others], before[others]) and not torch.equal(summary2[lastp[0]], before[lastp[0]])


@pytest.mark.parametrize("name", SMALL)
def test_page_score_matches_oracle(name):
    vx, w, ctx, pool, pt = setup(name)
    summary = build_summary(vx, w, ctx, pool, pt)
    scores = torch.full((w.spec.num_kv_heads, w.total_pages), float("nan"), device="cuda:0")
    ctx.page_score(w.q, summary, pt, scores)
    torch.cuda.synchronize()
    ref = oracle_step(w)
    got = scores.cpu().numpy().astype(np.float64)
    # fp32 accumulation of d*g products of magnitude <= |q||k|: relative 1e-5 of the score scale
    scale = np.abs(ref["scores"]).max()
    assert np.abs(got - ref["scores"]).max() <= 2e-5 * scale


@pytest.mark.parametrize("name", SMALL)
def test_topk_on_oracle_scores_is_bit_exact(name):
    # feed the kernel the oracle's scores rounded to fp32, and the oracle the same fp32 values:
    # then both sides decide on identical numbers and the selection must match exactly
    vx, w, ctx, pool, pt = setup(name)
    ref = oracle_step(w)
    s32 = ref["scores"].astype(np.float32)
    _, _, opt = to_oracle(w)
    sl_r, sp_r, sc_r, _ = vo.topk_pages(s32.astype(np.float64), opt, vo.as_np(w.budget), w.spec.n_sink,
                                        w.spec.n_local, w.max_budget)
    o = outputs(w)
    ctx.topk_pages(torch.from_numpy(s32).cuda(), pt, w.budget, w.max_budget, o["sel_phys"], o["sel_logical"],
                   o["sel_count"])
    torch.cuda.synchronize()
    assert np.array_equal(o["sel_count"].cpu().numpy(), sc_r)
    assert np.array_equal(o["sel_logical"].cpu().numpy(), sl_r)
    assert np.array_equal(o["sel_phys"].cpu().numpy(), sp_r)


def test_topk_constructed_ties_and_edge_budgets():
    from paper_2606_06453_b200.workloads import SPECS
    spec = replace(SPECS["C2-small"], batch=4, seq_len=(700, 1400))
    vx, w, ctx, pool, pt = setup(spec)
    g = torch.Generator().manual_seed(5)
    s32 = (torch.randint(0, 6, (w.spec.num_kv_heads, w.total_pages), generator=g).float() - 2.5)  # heavy ties, +-
    s32[0] = 1.25                                                                                # all equal
    pages = (w.seq_lens.cpu() + 15) // 16
    budget = torch.tensor([3, int(pages[1]), int(pages[2]) + 5, 17], dtype=torch.int32)          # min, == P, > P
    mb = int(budget.max())
    ctx2 = vx.context_for(w, max_budget=mb)
    _, _, opt = to_oracle(w)
    sl_r, sp_r, sc_r, _ = vo.topk_pages(s32.numpy().astype(np.float64), opt, budget.numpy(), 1, 2, mb)
    dev = "cuda:0"
    sl = torch.empty(4, 8, mb, dtype=torch.int32, device=dev); sp = torch.empty_like(sl)
    sc = torch.empty(4, 8, dtype=torch.int32, device=dev)
    ctx2.topk_pages(s32.to(dev), pt, budget.to(dev), mb, sp, sl, sc)
    torch.cuda.synchronize()
    assert np.array_equal(sc.cpu().numpy(), sc_r)
    assert np.array_equal(sl.cpu().numpy(), sl_r) and np.array_equal(sp.cpu().numpy(), sp_r)


@pytest.mark.parametrize("name", SMALL)
def test_decode_on_oracle_selection(name):
    vx, w, ctx, pool, pt = setup(name)
    ref = oracle_step(w)
    o = outputs(w)
    dev = "cuda:0"
    ctx.sparse_paged_decode(w.q, pool, pt, torch.from_numpy(ref["sel_phys"]).to(dev),
                            torch.from_numpy(ref["sel_logical"]).to(dev), torch.from_numpy(ref["sel_count"]).to(dev),
                            w.max_budget, o["out"], o["lse"])
    torch.cuda.synchronize()
    check_attention(w.spec.dtype, o["out"].float().cpu().numpy(), o["lse"].cpu().numpy(), ref["out"], ref["lse"])


@pytest.mark.parametrize("name", SMALL)
@pytest.mark.parametrize("flags", [0, 1])
def test_fused_step_matches_oracle(name, flags):
    vx, w, ctx, pool, pt = setup(name)
    summary = build_summary(vx, w, ctx, pool, pt)
    if flags:                                     # stale last-page summaries: the step must refresh them
        lastp = [int(w.page_indices[int(w.page_indptr[i + 1]) - 1]) for i in range(w.spec.batch)]
        summary[lastp] = 0
    o = outputs(w)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, o["out"], o["lse"], o["sel_phys"],
                           o["sel_logical"], o["sel_count"], flags=flags)
    torch.cuda.synchronize()
    assert ctx.last_launch_count >= (1 if w.spec.kv_shared else 3)     # MLA, small batch: one fused kernel; else score, select, decode
    ref = oracle_step(w)
    sl, sc = o["sel_logical"].cpu().numpy(), o["sel_count"].cpu().numpy()
    check_selection(w, sl, o["sel_phys"].cpu().numpy(), sc, ref)
    o_ref, l_ref = oracle_attention_on(w, sl, sc)
    check_attention(w.spec.dtype, o["out"].float().cpu().numpy(), o["lse"].cpu().numpy(), o_ref, l_ref)
    if w.planted:                                 # C3: planted pages should be found (sanity, not parity)
        rec = np.mean([len(set(w.planted[i]) & set(sl[i, h, :sc[i, h]].tolist())) / len(w.planted[i])
                       for i in range(w.spec.batch) for h in range(w.spec.num_kv_heads)])
        assert rec >= 0.99


@pytest.mark.parametrize("name", ["C1", "C2-small", "C3-small", "C5-small", "C4-small"])
def test_max_aggregation_scores_and_step_match_oracle(name):
    """VX_AGG_MAX (the max_h envelope variant): scores and the fused step against the oracle."""
    import paper_2606_06453_b200 as vxm
    vx, w, _, pool, pt = setup(name)
    ctx = vxm.context_for(w, agg=vxm.binding.VX_AGG_MAX)
    summary = build_summary(vx, w, ctx, pool, pt)
    ref = oracle_step(w, agg=vo.AGG_MAX)
    scores = torch.full((w.spec.num_kv_heads, w.total_pages), float("nan"), device="cuda:0")
    ctx.page_score(w.q, summary, pt, scores)
    torch.cuda.synchronize()
    got = scores.cpu().numpy().astype(np.float64)
    assert np.abs(got - ref["scores"]).max() <= 2e-5 * np.abs(ref["scores"]).max()
    # the invariant that defines the variant: S_max[j] >= u[h, j] for every head, with equality for one of them
    grp = w.spec.num_q_heads // w.spec.num_kv_heads
    u = ref["u"].reshape(w.spec.num_kv_heads, grp, -1)
    assert (got[:, None, :] >= u - 2e-5 * np.abs(u).max()).all()
    o = outputs(w)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, o["out"], o["lse"], o["sel_phys"],
                           o["sel_logical"], o["sel_count"], flags=1)
    torch.cuda.synchronize()
    sl, sc = o["sel_logical"].cpu().numpy(), o["sel_count"].cpu().numpy()
    check_selection(w, sl, o["sel_phys"].cpu().numpy(), sc, ref)
    o_ref, l_ref = oracle_attention_on(w, sl, sc)
    check_attention(w.spec.dtype, o["out"].float().cpu().numpy(), o["lse"].cpu().numpy(), o_ref, l_ref)


def test_step_without_local_pages_runs_the_summary_kernel_first():
    """n_local = 0: the newest page is not forced, so its refreshed summary must be in place BEFORE scoring
    (the decode kernel cannot fold the update); stale summaries of the newest pages must not change the result."""
    from paper_2606_06453_b200.workloads import SPECS
    spec = replace(SPECS["C2-small"], n_local=0, n_sink=1)
    vx, w, ctx, pool, pt = setup(spec)
    summary = build_summary(vx, w, ctx, pool, pt)
    lastp = [int(w.page_indices[int(w.page_indptr[i + 1]) - 1]) for i in range(w.spec.batch)]
    summary[lastp] = 0
    o = outputs(w)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, o["out"], o["lse"], o["sel_phys"],
                           o["sel_logical"], o["sel_count"], flags=1)
    torch.cuda.synchronize()
    assert ctx.last_launch_count >= 4
    ref = oracle_step(w)
    sl, sc = o["sel_logical"].cpu().numpy(), o["sel_count"].cpu().numpy()
    check_selection(w, sl, o["sel_phys"].cpu().numpy(), sc, ref)
    o_ref, l_ref = oracle_attention_on(w, sl, sc)
    check_attention(w.spec.dtype, o["out"].float().cpu().numpy(), o["lse"].cpu().numpy(), o_ref, l_ref)


@pytest.mark.parametrize("name", ["C1", "C4-small", "C5-small"])
def test_host_step_equals_device_step(name):
    vx, w, ctx, pool, pt = setup(name)
    summary = build_summary(vx, w, ctx, pool, pt)
    o = outputs(w)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, o["out"], o["lse"])
    torch.cuda.synchronize()
    pin = lambda t: t.cpu().contiguous().pin_memory()
    h_out = torch.empty_like(o["out"], device="cpu").pin_memory()
    h_lse = torch.empty_like(o["lse"], device="cpu").pin_memory()
    ctx.sparse_decode_step_host(pin(w.q), pool, summary, pin(w.page_indptr), pin(w.page_indices), pin(w.seq_lens),
                                pin(w.budget), w.max_budget, h_out, h_lse)
    assert torch.equal(h_out, o["out"].cpu()) and torch.equal(h_lse, o["lse"].cpu())


def test_full_budget_equals_dense_attention():
    from paper_2606_06453_b200.workloads import SPECS
    spec = replace(SPECS["C2-small"], budget=300)          # >= every request's page count
    vx, w, ctx, pool, pt = setup(spec)
    summary = build_summary(vx, w, ctx, pool, pt)
    o = outputs(w)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, o["out"], o["lse"], o["sel_phys"],
                           o["sel_logical"], o["sel_count"])
    torch.cuda.synchronize()
    pages = ((w.seq_lens + 15) // 16).cpu().numpy()
    assert np.array_equal(o["sel_count"].cpu().numpy(), np.repeat(pages[:, None], 8, 1))
    q, opool, opt = to_oracle(w)
    od, ld = vo.dense_attention(q, opool, opt, 32, 8, 128, 128, spec.sm_scale)
    check_attention("bf16", o["out"].float().cpu().numpy(), o["lse"].cpu().numpy(), od, ld)


def test_empty_batch_and_bad_arguments():
    vx, w, ctx, pool, pt = setup("C1")
    empty = vx.PageTable(torch.zeros(1, dtype=torch.int32, device="cuda:0"),
                         torch.zeros(0, dtype=torch.int32, device="cuda:0"),
                         torch.zeros(0, dtype=torch.int32, device="cuda:0"), 0, 0)
    o = outputs(w)
    summary = vx.alloc_summary(w)
    ctx.sparse_decode_step(w.q, pool, summary, empty, w.budget, w.max_budget, o["out"], o["lse"])   # no-op
    assert ctx.last_launch_count == 0
    with pytest.raises(vx.VortexError) as e:
        ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget + 1, o["out"], o["lse"])
    assert e.value.status == 3
    with pytest.raises(vx.VortexError) as e:
        ctx.sparse_decode_step(None, pool, summary, pt, w.budget, w.max_budget, o["out"], o["lse"])
    assert e.value.status == 1
    with pytest.raises(vx.VortexError) as e:
        vx.context_for(w, qk_dim=80, v_dim=80)
    assert e.value.status == 2


def test_trace_attach_is_refused_by_the_product_library_and_works_in_the_trace_build():
    """vx_trace_attach (include/vortex_b200.h): the product library carries no stamps and says so; the -DVX_TRACE
    build records one timeline per CTA (paper_2606_06453_b200/trace.py, run here on a small config)."""
    import subprocess
    import sys
    import paper_2606_06453_b200 as vxm
    from paper_2606_06453_b200.binding import VortexError, VX_ERR_UNSUPPORTED, VX_TRACE_SCORE
    vx, w, ctx, pool, pt = setup("C2-small")
    buf = torch.zeros(64, 16, dtype=torch.int64, device="cuda:0")
    with pytest.raises(VortexError) as e:
        ctx.trace_attach(buf, VX_TRACE_SCORE)
    assert e.value.status == VX_ERR_UNSUPPORTED
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for kernel in ("score", "topk", "decode"):
        r = subprocess.run([sys.executable, "-m", "paper_2606_06453_b200.trace", "--config", "C2-small", "--kernel", kernel,
                            "--iters", "1"], cwd=root, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        assert "entry" in r.stdout and "CTAs on" in r.stdout, r.stdout
