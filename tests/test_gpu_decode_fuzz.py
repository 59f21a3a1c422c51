"""vx_sparse_paged_decode on arbitrary selection lists (-m gpu): random subsets of each request's pages in RANDOM
order (the call does not require the ascending order vx_topk_pages emits), counts from 1 page up to the budget,
fewer pages than split CTAs, the partial last page anywhere in the list -- against the oracle on the same lists."""
import numpy as np
import pytest
import torch

from oracle.workload_io import to_oracle
from tests.parity import check_attention
from oracle import vx_oracle as vo

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name", ["C2-small", "C3-small", "C4-small", "C5-small"])
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_decode_on_random_unordered_selections(name, seed):
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload
    w = make_workload(name, device="cuda:0")
    s = w.spec
    mb = w.max_budget
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    rng = np.random.default_rng(seed)
    P = ((w.seq_lens.cpu().numpy() + s.page_size - 1) // s.page_size)
    indptr, indices = w.page_indptr.cpu().numpy(), w.page_indices.cpu().numpy()
    sl = np.full((s.batch, s.num_kv_heads, mb), -1, np.int32)
    sp = np.full_like(sl, -1)
    sc = np.zeros((s.batch, s.num_kv_heads), np.int32)
    for i in range(s.batch):
        for h in range(s.num_kv_heads):
            hi = min(mb, int(P[i]))
            cnt = int(rng.choice([1, 2, 3, hi // 2 + 1, hi]))
            cnt = max(1, min(cnt, hi))
            pick = rng.permutation(int(P[i]))[:cnt]              # random subset, random order
            if seed == 0 and cnt >= 2:                           # the partial last page in the middle of the list
                pick[cnt // 2] = P[i] - 1 if (P[i] - 1) not in pick else pick[cnt // 2]
            sl[i, h, :cnt] = pick
            sp[i, h, :cnt] = indices[indptr[i] + pick]
            sc[i, h] = cnt
    dev = "cuda:0"
    out = torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev)
    lse = torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    ctx.sparse_paged_decode(w.q, pool, pt, torch.from_numpy(sp).to(dev), torch.from_numpy(sl).to(dev),
                            torch.from_numpy(sc).to(dev), mb, out, lse)
    torch.cuda.synchronize()
    q, opool, opt = to_oracle(w)
    o_ref, l_ref = vo.sparse_attention(q, opool, opt, sl, sc, s.num_q_heads, s.num_kv_heads, s.qk_dim, s.v_dim, s.sm_scale)
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)


@pytest.mark.parametrize("batch,splits", [(3, 8), (20, 4), (40, 3), (50, 2)])
def test_mla_decode_cluster_merge_at_every_cluster_size(batch, splits):
    """The MLA decode merges the splits of a request inside a thread-block cluster (2, 4 or 8 CTAs, DESIGN.md 7;
    any other count goes through global partials and an arrival counter):
    batches chosen so that the split heuristic picks each size, selections shorter than the split count included
    (empty splits), the fused step against the oracle."""
    from dataclasses import replace
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload, SPECS
    from oracle.workload_io import oracle_step
    from tests.parity import check_selection, oracle_attention_on
    w = make_workload(replace(SPECS["C4-small"], name=f"C4-small-b{batch}", batch=batch, seq_len=(200, 3000)), device="cuda:0")
    s = w.spec
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    dev = "cuda:0"
    out = torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev)
    lse = torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    sp = torch.empty(s.batch, s.num_kv_heads, w.max_budget, dtype=torch.int32, device=dev)
    sl = torch.empty_like(sp)
    sc = torch.empty(s.batch, s.num_kv_heads, dtype=torch.int32, device=dev)
    for _ in range(2):                            # twice: the kernel leaves no state behind
        out.fill_(float("nan"))
        ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc)
    torch.cuda.synchronize()
    # the split count the library picks for this batch (its heuristic, restated): whole waves of equal CTAs
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    cost = lambda sp: -(-s.batch * sp // sms) * (-(-w.max_budget // sp) + 2)
    assert min(range(1, min(32, w.max_budget, s.num_q_heads) + 1), key=lambda sp: (cost(sp), sp)) == splits
    ref = oracle_step(w)
    sl_h, sc_h = sl.cpu().numpy(), sc.cpu().numpy()
    check_selection(w, sl_h, sp.cpu().numpy(), sc_h, ref)
    o_ref, l_ref = oracle_attention_on(w, sl_h, sc_h)
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)


def _gqa_splits(units, budget, sms, fp8):
    """the GQA decode kernels' split heuristics, restated (vx_decode_gqa.cu: decode_gqa_splits; vx_decode_gqa_fp8.cu)"""
    slots = sms * (3 if fp8 else 2)
    fixed = 30 if fp8 else 3
    cost = lambda sp: -(-units * sp // slots) * (-(-(-(-budget // sp)) // 4) + fixed)
    return min(range(1, min(32, budget) + 1), key=lambda sp: (cost(sp), sp))


@pytest.mark.parametrize("fmt", ["bf16", "e4m3"])
@pytest.mark.parametrize("batch,budget,splits", [(1, 32, 8), (8, 64, 4), (12, 64, None), (16, 64, 2), (20, 64, None)])
def test_gqa_decode_cluster_merge_at_every_cluster_size(fmt, batch, budget, splits):
    """The GQA decode kernels (bf16 and fp8 KV cache) merge 2, 4 or 8 splits of a (request, KV head) inside a thread-block
    cluster over distributed shared memory, any other count through global partials and an arrival counter:
    batches chosen so that the heuristics pick cluster sizes 8, 4 and 2 and a non-cluster count, requests with fewer pages
    than split warps included (empty splits), run twice (no state left behind), the fused step against the oracle."""
    from dataclasses import replace
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload, SPECS, with_fp8
    from oracle.workload_io import oracle_step
    from tests.parity import check_selection, oracle_attention_on
    spec = replace(SPECS["C3-small"], name=f"C3-small-b{batch}k{budget}", batch=batch, seq_len=(300, 4000), budget=budget)
    if fmt != "bf16":
        spec = with_fp8(spec, fmt)
    w = make_workload(spec, device="cuda:0")
    s = w.spec
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    got = _gqa_splits(s.batch * s.num_kv_heads, w.max_budget, sms, fmt != "bf16")
    if fmt == "bf16" and splits is not None:
        assert got == splits                      # (the bf16 rows are built to hit each cluster size)
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    dev = "cuda:0"
    out = torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev)
    lse = torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    sp = torch.empty(s.batch, s.num_kv_heads, w.max_budget, dtype=torch.int32, device=dev)
    sl = torch.empty_like(sp)
    sc = torch.empty(s.batch, s.num_kv_heads, dtype=torch.int32, device=dev)
    for _ in range(2):
        out.fill_(float("nan"))
        ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc)
    torch.cuda.synchronize()
    ref = oracle_step(w)
    sl_h, sc_h = sl.cpu().numpy(), sc.cpu().numpy()
    check_selection(w, sl_h, sp.cpu().numpy(), sc_h, ref)
    o_ref, l_ref = oracle_attention_on(w, sl_h, sc_h)
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)
    print(f"[gqa cluster merge] {fmt} batch {batch} budget {w.max_budget}: {got} splits")
