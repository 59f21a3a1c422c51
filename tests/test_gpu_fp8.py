"""fp8 KV cache (-m gpu; NEXT-2, PAPER.md:200 / :520 / :525): pools and summaries as fp8_e4m3 / fp8_e5m2 codes with one
scale per pool tensor (G25-G27), bf16 queries and outputs.  Every call against the fp64 oracle on the values
the codes stand for (oracle/vx_oracle_fp8.py): summaries bit-exact, scores to 2e-5 of the score scale, selections by the
parity comparator, attention within the bf16 tolerances on the GPU's own selection -- at reduced sizes element by
element and at full size (C2, C4) on sampled requests."""
import numpy as np
import pytest
import torch

from oracle import vx_oracle as vo
from oracle.vx_oracle_fp8 import dequantize
from oracle.workload_io import oracle_step, to_oracle
from tests.parity import check_attention, check_selection, oracle_attention_on

pytestmark = pytest.mark.gpu


def run(spec, poison_newest=True):
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload
    w = make_workload(spec, device="cuda:0")
    s = w.spec
    dev = w.q.device
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    assert summary.dtype == torch.uint8
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    clean = summary.clone()
    if poison_newest:                                   # the fused step must rebuild the newest page's summary (a1)
        last = w.page_indices[(w.page_indptr[1:] - 1).long()].long()
        summary[last] = 0x55
    out = torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev)
    lse = torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    sp = torch.full((s.batch, s.num_kv_heads, w.max_budget), -7, dtype=torch.int32, device=dev)
    sl, sc = torch.full_like(sp, -7), torch.full((s.batch, s.num_kv_heads), -7, dtype=torch.int32, device=dev)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc,
                           flags=vx.VX_STEP_UPDATE_SUMMARY)
    torch.cuda.synchronize()
    return vx, w, ctx, pool, pt, summary, clean, out, lse, sp, sl, sc


CASES = [("C2-small", "e4m3"), ("C4-small", "e4m3"), ("C5-small", "e4m3"), ("C3-small", "e4m3"), ("C2-small", "e5m2"),
         ("C4-small", "e5m2")]


@pytest.mark.parametrize("name,fmt", CASES)
def test_fp8_calls_and_fused_step_match_the_oracle(name, fmt):
    from paper_2606_06453_b200.workloads import with_fp8
    vx, w, ctx, pool, pt, summary, clean, out, lse, sp, sl, sc = run(with_fp8(name, fmt))
    s = w.spec
    ref = oracle_step(w)
    # (a1) summaries: the min / max CODES, exact -- compared as the values they stand for, on every page of the table
    phys = w.page_indices.cpu().long().numpy()
    got = dequantize(clean.cpu().numpy(), fmt, w.k_scale)[phys]
    assert np.array_equal(got, ref["summary"][phys]), "fp8 summaries differ from the oracle's envelope"
    assert torch.equal(summary, clean), "the step rebuilds the newest page's summary, nothing else changes"
    # (a2) scores: computed without k_scale (G27)
    scores = torch.empty(s.num_kv_heads, w.total_pages, dtype=torch.float32, device="cuda:0")
    ctx.page_score(w.q, clean, pt, scores)
    torch.cuda.synchronize()
    g = scores.cpu().numpy().astype(np.float64) * float(np.float32(w.k_scale))
    scale = np.abs(ref["scores"]).max()
    assert np.abs(g - ref["scores"]).max() <= 2e-5 * scale
    # (a3) + (a6) selection of the fused step; the separate calls give the same one
    check_selection(w, sl.cpu().numpy(), sp.cpu().numpy(), sc.cpu().numpy(), ref, label=f"{s.name} fused step")
    sp2, sl2, sc2 = torch.full_like(sp, -7), torch.full_like(sl, -7), torch.full_like(sc, -7)
    ctx.topk_pages(scores, pt, w.budget, w.max_budget, sp2, sl2, sc2)
    torch.cuda.synchronize()
    assert torch.equal(sl, sl2) and torch.equal(sp, sp2) and torch.equal(sc, sc2)
    # (a4) + (a5) attention on the GPU's selection, scaled values
    o_ref, l_ref = oracle_attention_on(w, sl.cpu().numpy(), sc.cpu().numpy())
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)
    out2, lse2 = torch.full_like(out, float("nan")), torch.full_like(lse, float("nan"))
    ctx.sparse_paged_decode(w.q, pool, pt, sp, sl, sc, w.max_budget, out2, lse2)
    torch.cuda.synchronize()
    check_attention(s.dtype, out2.float().cpu().numpy(), lse2.cpu().numpy(), o_ref, l_ref)
    ctx.close()


def test_fp8_scales_are_used_once():
    """doubling v_scale doubles the output and leaves lse; a power-of-two k_scale with sm_scale halved changes nothing"""
    from dataclasses import replace
    from paper_2606_06453_b200.workloads import with_fp8
    vx, w, ctx, pool, pt, summary, clean, out, lse, sp, sl, sc = run(with_fp8("C2-small"))
    sp_, st_, sh_ = w.strides
    pool2 = vx.KvPool(w.k_pool, w.v_pool, sp_, st_, sh_, w.k_scale, 2.0 * w.v_scale)
    out2, lse2 = torch.empty_like(out), torch.empty_like(lse)
    ctx.sparse_paged_decode(w.q, pool2, pt, sp, sl, sc, w.max_budget, out2, lse2)
    out1, lse1 = torch.empty_like(out), torch.empty_like(lse)
    ctx.sparse_paged_decode(w.q, pool, pt, sp, sl, sc, w.max_budget, out1, lse1)
    torch.cuda.synchronize()
    assert torch.equal(lse1, lse2)
    assert float((out2.float() - 2.0 * out1.float()).abs().max()) <= 2.0 ** -7 * float(out2.float().abs().max())
    with pytest.raises(vx.VortexError):                  # a missing scale is refused, not silently read as zero
        ctx.sparse_paged_decode(w.q, vx.KvPool(w.k_pool, w.v_pool, sp_, st_, sh_, 0.0, 1.0), pt, sp, sl, sc, w.max_budget, out1, lse1)
    ctx.close()


def test_fp8_rejects_what_it_does_not_build():
    import paper_2606_06453_b200 as vx
    kw = dict(dtype=torch.bfloat16, num_q_heads=32, num_kv_heads=8, qk_dim=128, v_dim=128, page_size=16, sm_scale=0.1,
              n_sink=1, n_local=2, max_batch=2, max_total_pages=64, max_pages_per_req=32, max_budget=8)
    vx.Context(kv_format=vx.binding.VX_KV_FP8_E4M3, **kw).close()
    for bad in (dict(kv_format=3), dict(kv_format=1, summary_kind=vx.binding.VX_SUMMARY_CENTROID),
                dict(kv_format=1, agg=vx.binding.VX_AGG_MAX), dict(kv_format=2, dtype=torch.float32)):
        with pytest.raises(vx.VortexError):
            vx.Context(**{**kw, **bad})


@pytest.mark.parametrize("name,samples", [("C2", [3, 20]), ("C4", [5, 31, 60])])
def test_fp8_fullsize_sampled(name, samples):
    from paper_2606_06453_b200.workloads import subproblem, with_fp8
    vx, w, ctx, pool, pt, summary, clean, out, lse, sp, sl, sc = run(with_fp8(name))
    s = w.spec
    n = w.seq_lens.cpu().long()
    P = (n + s.page_size - 1) // s.page_size
    assert torch.equal(sc.cpu().long(), torch.minimum(w.budget.cpu().long(), P)[:, None].expand(-1, s.num_kv_heads))
    assert bool(torch.isfinite(out.float()).all()) and bool(torch.isfinite(lse).all())
    for r in samples:
        sub = subproblem(w, [r])
        ref = oracle_step(sub)
        check_selection(sub, sl[r:r + 1].cpu().numpy(), sl[r:r + 1].cpu().numpy(), sc[r:r + 1].cpu().numpy(), ref,
                        label=f"{s.name} full size, request {r}")
        q, opool, opt = to_oracle(sub)
        o_ref, l_ref = vo.sparse_attention(q, opool, opt, sl[r:r + 1].cpu().numpy(), sc[r:r + 1].cpu().numpy(),
                                           s.num_q_heads, s.num_kv_heads, s.qk_dim, s.v_dim, s.sm_scale)
        check_attention(s.dtype, out[r:r + 1].float().cpu().numpy(), lse[r:r + 1].cpu().numpy(), o_ref, l_ref)
    ctx.close()
