"""The fused MLA step kernel (-m gpu): vx_sparse_decode_step on the MLA geometry runs score -> select -> decode -> merge of
a request in ONE kernel on the thread-block cluster that owns the request (csrc/vx_step_mla.cu; DESIGN.md
section 17).  Checked against the fp64 oracle by the stated tolerances, and -- because the kernel computes its scores in
vx_page_score's summation order and selects with the same device function as vx_topk_pages -- bit for bit against the
three separate C-ABI calls.  The cases drive the schedule's edges: every cluster size (8 / 4 / 2 / 1 CTAs per
request), requests shorter than one CTA's share (1 .. 7 pages on 8 CTAs), budgets >= P, budgets that are all forced
pages, partial last pages, long requests (several ring wraps of the summary stream)."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from oracle import vx_oracle as vo
from oracle.workload_io import oracle_step, to_oracle
from tests.parity import check_attention, check_selection, oracle_attention_on

pytestmark = pytest.mark.gpu


SCHEDULES = ["fused", "flat"]


def run_fused(spec, flags=None, schedule="fused"):
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload
    w = make_workload(spec, device="cuda:0")
    s = w.spec
    dev = w.q.device
    ctx = vx.context_for(w)
    ctx.set_option(vx.VX_OPT_MLA_STEP, vx.VX_MLA_STEP_FLAT if schedule == "flat" else vx.VX_MLA_STEP_FUSED)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    last = w.page_indices[(w.page_indptr[1:] - 1).long()].long()
    clean = summary.clone()
    summary[last] = 0                                   # the step must rebuild the newest page's summary (a1)
    out = torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev)
    lse = torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    sp = torch.full((s.batch, s.num_kv_heads, w.max_budget), -7, dtype=torch.int32, device=dev)
    sl = torch.full_like(sp, -7)
    sc = torch.full((s.batch, s.num_kv_heads), -7, dtype=torch.int32, device=dev)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc,
                           flags=vx.VX_STEP_UPDATE_SUMMARY if flags is None else flags)
    torch.cuda.synchronize()
    launches = ctx.last_launch_count
    return vx, w, ctx, pool, pt, summary, clean, out, lse, sp, sl, sc, launches


CASES = {
    # name: (batch, seq_len range, budget)  -> cluster size the launcher picks on 148 SMs
    "tiny-requests-on-8-ctas": (3, (1, 448), 6),          # 1..7 pages: shares of 0 or 1 page, budgets >= P
    "forced-only-budget": (5, (200, 3000), 2),            # budget = n_sink + n_local: nothing to rank
    "cluster8": (6, (3000, 40000), 12),
    "cluster4": (30, (500, 9000), 9),
    "cluster2": (70, (64, 6000), 8),
    "cluster1": (150, (1, 2500), 5),
    "long-requests": (2, (150000, 260000), 40),           # 2,344 .. 4,063 pages: the summary ring wraps many times
}


@pytest.mark.parametrize("schedule", SCHEDULES)
@pytest.mark.parametrize("case", list(CASES))
def test_fused_step_matches_oracle_and_the_separate_calls(case, schedule):
    from paper_2606_06453_b200.workloads import SPECS
    batch, seq, budget = CASES[case]
    spec = replace(SPECS["C4"], name=case, batch=batch, seq_len=seq, budget=budget, cfg_id=40 + list(CASES).index(case))
    vx, w, ctx, pool, pt, summary, clean, out, lse, sp, sl, sc, launches = run_fused(spec, schedule=schedule)
    s = w.spec
    assert launches == 1, "the MLA step is one kernel"
    ref = oracle_step(w)
    check_selection(w, sl.cpu().numpy(), sp.cpu().numpy(), sc.cpu().numpy(), ref)
    o_ref, l_ref = oracle_attention_on(w, sl.cpu().numpy(), sc.cpu().numpy())
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)
    assert torch.equal(summary, clean), "the newest page's summary is rebuilt inside the step (a1), nothing else is touched"
    # ---- the same selection, bit for bit, from the three separate calls ---------------------------------------
    scores = torch.empty(s.num_kv_heads, w.total_pages, dtype=torch.float32, device="cuda:0")
    ctx.page_score(w.q, clean, pt, scores)
    sp2, sl2, sc2 = torch.full_like(sp, -7), torch.full_like(sl, -7), torch.full_like(sc, -7)
    ctx.topk_pages(scores, pt, w.budget, w.max_budget, sp2, sl2, sc2)
    out2, lse2 = torch.empty_like(out), torch.empty_like(lse)
    ctx.sparse_paged_decode(w.q, pool, pt, sp2, sl2, sc2, w.max_budget, out2, lse2)
    torch.cuda.synchronize()
    assert torch.equal(sc, sc2) and torch.equal(sl, sl2) and torch.equal(sp, sp2)
    check_attention(s.dtype, out2.float().cpu().numpy(), lse2.cpu().numpy(), o_ref, l_ref)
    # ---- ... and from the step's other schedule (three chained kernels) ------------------------------------------
    ctx.set_option(vx.VX_OPT_MLA_STEP, vx.VX_MLA_STEP_CHAINED)
    sp3, sl3, sc3 = torch.full_like(sp, -7), torch.full_like(sl, -7), torch.full_like(sc, -7)
    out3, lse3 = torch.empty_like(out), torch.empty_like(lse)
    ctx.sparse_decode_step(w.q, pool, clean, pt, w.budget, w.max_budget, out3, lse3, sp3, sl3, sc3, flags=0)
    torch.cuda.synchronize()
    assert ctx.last_launch_count == 3
    assert torch.equal(sc, sc3) and torch.equal(sl, sl3) and torch.equal(sp, sp3)
    check_attention(s.dtype, out3.float().cpu().numpy(), lse3.cpu().numpy(), o_ref, l_ref)
    with pytest.raises(vx.VortexError):
        ctx.set_option(vx.VX_OPT_MLA_STEP, 7)
    ctx.close()


@pytest.mark.parametrize("schedule", SCHEDULES)
def test_fused_step_without_summary_update_leaves_the_pool_alone(schedule):
    from paper_2606_06453_b200.workloads import SPECS
    spec = replace(SPECS["C4"], name="no-update", batch=9, seq_len=(100, 5000), budget=7, cfg_id=48)
    vx, w, ctx, pool, pt, summary, clean, out, lse, sp, sl, sc, launches = run_fused(spec, flags=0, schedule=schedule)
    last = w.page_indices[(w.page_indptr[1:] - 1).long()].long()
    assert launches == 1 and bool((summary[last] == 0).all())          # poisoned rows stay as they were
    o_ref, l_ref = oracle_attention_on(w, sl.cpu().numpy(), sc.cpu().numpy())
    check_attention(w.spec.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)
    ctx.close()


@pytest.mark.parametrize("schedule", SCHEDULES)
def test_fused_step_centroid_flow(schedule):
    """block top-k summaries (Eq.1-2) through the fused kernel: 1,152-byte rows, [Qsum] query vector"""
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import SPECS, make_workload
    spec = replace(SPECS["C4"], name="centroid", batch=12, seq_len=(300, 20000), budget=10, cfg_id=49)
    w = make_workload(spec, device="cuda:0")
    s = w.spec
    kind = vx.binding.VX_SUMMARY_CENTROID
    ctx = vx.context_for(w, summary_kind=kind)
    ctx.set_option(vx.VX_OPT_MLA_STEP, vx.VX_MLA_STEP_FLAT if schedule == "flat" else vx.VX_MLA_STEP_FUSED)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w, kind)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    clean = summary.clone()
    last = w.page_indices[(w.page_indptr[1:] - 1).long()].long()
    summary[last] = 0
    dev = "cuda:0"
    out = torch.empty(s.batch, s.num_q_heads, s.v_dim, dtype=w.q.dtype, device=dev)
    lse = torch.empty(s.batch, s.num_q_heads, dtype=torch.float32, device=dev)
    sp = torch.full((s.batch, 1, w.max_budget), -7, dtype=torch.int32, device=dev)
    sl, sc = torch.full_like(sp, -7), torch.full((s.batch, 1), -7, dtype=torch.int32, device=dev)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc,
                           flags=vx.VX_STEP_UPDATE_SUMMARY)
    torch.cuda.synchronize()
    assert ctx.last_launch_count == 1 and torch.equal(summary, clean)
    scores = torch.empty(1, w.total_pages, dtype=torch.float32, device=dev)
    ctx.page_score(w.q, clean, pt, scores)
    sp2, sl2, sc2 = torch.full_like(sp, -7), torch.full_like(sl, -7), torch.full_like(sc, -7)
    ctx.topk_pages(scores, pt, w.budget, w.max_budget, sp2, sl2, sc2)
    torch.cuda.synchronize()
    assert torch.equal(sl, sl2) and torch.equal(sp, sp2) and torch.equal(sc, sc2)
    o_ref, l_ref = oracle_attention_on(w, sl.cpu().numpy(), sc.cpu().numpy())
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)
    ctx.close()
