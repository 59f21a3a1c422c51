"""GPU parity of the block top-k flow: VX_SUMMARY_CENTROID summaries,
scores, and the fused step against the oracle (-m gpu).  Same bars as the envelope flow: summaries bit-exact,
selections exact up to the 1e-3 near-tie rule, attention within the bf16 tolerances on the GPU's selected set."""
import numpy as np
import pytest
import torch

from oracle import vx_oracle as vo
from oracle.workload_io import bf16_bits_to_f64, to_oracle
from tests.parity import check_attention, check_selection, oracle_attention_on

pytestmark = pytest.mark.gpu

SMALL = ["C1", "C2-small", "C3-small", "C4-small", "C5-small"]


def setup(name):
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200 import binding
    from paper_2606_06453_b200.workloads import make_workload
    w = make_workload(name, device="cuda:0")
    ctx = vx.context_for(w, summary_kind=binding.VX_SUMMARY_CENTROID)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w, binding.VX_SUMMARY_CENTROID)
    return vx, w, ctx, pool, pt, summary


def oracle_centroid_step(w):
    q, pool, pt = to_oracle(w)
    s = w.spec
    return vo.decode_step(q, pool, pt, vo.as_np(w.budget), w.max_budget, s.num_q_heads, s.num_kv_heads, s.qk_dim,
                          s.v_dim, s.sm_scale, s.n_sink, s.n_local, kind="centroid")


def as_f64(t):
    a = vo.as_np(t)
    return bf16_bits_to_f64(a)


@pytest.mark.parametrize("name", SMALL)
def test_centroid_summaries_are_bit_exact_bulk_and_append(name):
    vx, w, ctx, pool, pt, summary = setup(name)
    n = w.seq_lens.cpu(); b = w.spec.page_size
    for i in range(w.spec.batch):                  # poison stale slots of partial last pages
        r = int(n[i]) % b
        if r:
            phys = int(w.page_indices[int(w.page_indptr[i + 1]) - 1])
            w.k_pool[phys, :, r:, :] = 1e30
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    torch.cuda.synchronize()
    _, opool, opt = to_oracle(w)
    ref = vo.page_centroid(opool, opt, w.spec.num_kv_heads, w.spec.qk_dim)
    got = as_f64(summary)
    used = np.unique(vo.as_np(w.page_indices))
    assert np.array_equal(got[used], ref[used]), "centroids must match the oracle bit for bit"
    # append mode: only each request's newest page is rebuilt
    last = w.page_indices[(w.page_indptr[1:] - 1).long()].long()
    summary.zero_()
    ctx.page_summary_update(pool, pt, summary, first_new_pos=None)
    torch.cuda.synchronize()
    got = as_f64(summary)
    lastn = last.cpu().numpy()
    assert np.array_equal(got[lastn], ref[lastn])
    mask = np.ones(got.shape[0], bool); mask[lastn] = False
    assert (got[mask] == 0).all()


@pytest.mark.parametrize("name", SMALL)
def test_centroid_scores_and_fused_step_match_oracle(name):
    vx, w, ctx, pool, pt, summary = setup(name)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    ref = oracle_centroid_step(w)
    scores = torch.full((w.spec.num_kv_heads, w.total_pages), float("nan"), device="cuda:0")
    ctx.page_score(w.q, summary, pt, scores)
    torch.cuda.synchronize()
    got = scores.cpu().numpy().astype(np.float64)
    assert np.abs(got - ref["scores"]).max() <= 2e-5 * max(np.abs(ref["scores"]).max(), np.abs(ref["u"]).max())
    # stale newest-page centroids: the step (flag) must refresh them before scoring (no fold for this kind)
    s = w.spec
    dev = "cuda:0"
    last = w.page_indices[(w.page_indptr[1:] - 1).long()].long()
    summary[last] = 0
    out = torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev)
    lse = torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    sp = torch.full((s.batch, s.num_kv_heads, w.max_budget), -7, dtype=torch.int32, device=dev)
    sl = torch.full_like(sp, -7)
    sc = torch.full((s.batch, s.num_kv_heads), -7, dtype=torch.int32, device=dev)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc, flags=1)
    torch.cuda.synchronize()
    sln, scn = sl.cpu().numpy(), sc.cpu().numpy()
    check_selection(w, sln, sp.cpu().numpy(), scn, ref)
    o_ref, l_ref = oracle_attention_on(w, sln, scn)
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)
    lastn = last.cpu().numpy()
    assert np.array_equal(as_f64(summary)[lastn], ref["summary"][lastn])


def test_centroid_rejects_max_aggregation():
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200 import binding
    from paper_2606_06453_b200.workloads import make_workload
    w = make_workload("C2-small", device="cuda:0")
    with pytest.raises(vx.VortexError):
        vx.context_for(w, summary_kind=binding.VX_SUMMARY_CENTROID, agg=binding.VX_AGG_MAX)
