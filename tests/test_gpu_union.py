"""vx_union_pages against oracle/vx_oracle_union.py (-m gpu): bit-exact ids, order, counts, padding."""
import numpy as np
import pytest
import torch

from oracle import vx_oracle as vo
from oracle import vx_oracle_union as vu

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed", [0, 1, 2])
@pytest.mark.parametrize("hkv,k", [(8, 128), (1, 32), (2, 300)])
def test_union_matches_the_oracle(seed, hkv, k):
    import paper_2606_06453_b200 as vx
    rng = np.random.default_rng(seed)
    pages = [int(x) for x in rng.choice([1, 5, 40, 300, 2048, 5000, 20000], size=5)]
    b = 16
    seq = [p * b - int(rng.integers(0, b)) for p in pages]
    indptr = np.concatenate([[0], np.cumsum(pages)]).astype(np.int32)
    T = int(indptr[-1])
    indices = rng.permutation(T + 11)[:T].astype(np.int32)
    budget = np.array([max(3, int(rng.integers(3, k + 1))) for _ in pages], np.int32)
    scores = rng.standard_normal((hkv, T)).astype(np.float32)
    if seed == 2:
        scores[1:] = scores[:1]                       # identical heads: the union is one head's set
    dev = "cuda:0"
    ctx = vx.Context(dtype=torch.bfloat16, num_q_heads=4 * hkv, num_kv_heads=hkv, qk_dim=128, v_dim=128, page_size=b,
                     sm_scale=1.0, n_sink=1, n_local=2, max_batch=len(pages), max_total_pages=T,
                     max_pages_per_req=max(pages), max_budget=k, device=dev)
    pt = vx.PageTable(torch.from_numpy(indptr).to(dev), torch.from_numpy(indices).to(dev),
                      torch.tensor(seq, dtype=torch.int32, device=dev), T, max(pages))
    sl = torch.full((len(pages), hkv, k), -7, dtype=torch.int32, device=dev)
    sp = torch.full_like(sl, -7)
    sc = torch.full((len(pages), hkv), -7, dtype=torch.int32, device=dev)
    ctx.topk_pages(torch.from_numpy(scores).to(dev), pt, torch.from_numpy(budget).to(dev), k, sp, sl, sc)
    mu = min(hkv * k, max(pages))
    ul = torch.full((len(pages), mu), -7, dtype=torch.int32, device=dev)
    up = torch.full_like(ul, -7)
    uc = torch.full((len(pages),), -7, dtype=torch.int32, device=dev)
    ctx.union_pages(pt, sl, sc, k, mu, up, ul, uc)
    torch.cuda.synchronize()
    ul_r, up_r, uc_r = vu.union_pages(sl.cpu().numpy(), sc.cpu().numpy(), indptr, indices, np.array(seq), b, mu)
    assert np.array_equal(uc.cpu().numpy(), uc_r)
    assert np.array_equal(ul.cpu().numpy(), ul_r)
    assert np.array_equal(up.cpu().numpy(), up_r)
    if seed == 2:
        assert np.array_equal(uc.cpu().numpy(), sc.cpu().numpy()[:, 0])
    with pytest.raises(vx.VortexError):               # max_union below the largest possible union
        ctx.union_pages(pt, sl, sc, k, mu - 1, up, ul, uc)
    ctx.union_pages(pt, sl, sc, k, mu, up, None, uc)  # union_logical is optional
    torch.cuda.synchronize()
    assert np.array_equal(up.cpu().numpy(), up_r)
    ctx.close()


@pytest.mark.parametrize("name", ["C2-small", "C5-small"])
def test_decode_over_the_union_table(name):
    """The use the paper names for Union (:538, :200): one block table per request for the decode backend.  The union
    table, broadcast to every KV head, drives vx_sparse_paged_decode; outputs match the oracle's attention over the
    union set within the bf16 tolerances."""
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload
    from oracle.workload_io import oracle_step
    from tests.parity import check_attention, oracle_attention_on
    w = make_workload(name, device="cuda:0")
    s = w.spec
    ref = oracle_step(w)
    dev = "cuda:0"
    mu = min(s.num_kv_heads * w.max_budget, w.max_pages_per_req)
    ctx = vx.context_for(w, max_budget=mu)
    pool, pt = vx.tables_for(w)
    sl = torch.from_numpy(ref["sel_logical"]).to(dev)
    sc = torch.from_numpy(ref["sel_count"]).to(dev)
    ul = torch.empty(s.batch, mu, dtype=torch.int32, device=dev)
    up = torch.empty_like(ul)
    uc = torch.empty(s.batch, dtype=torch.int32, device=dev)
    ctx.union_pages(pt, sl, sc, w.max_budget, mu, up, ul, uc)
    ul_r, up_r, uc_r = vu.union_pages(ref["sel_logical"], ref["sel_count"], w.page_indptr.cpu().numpy(),
                                      w.page_indices.cpu().numpy(), w.seq_lens.cpu().numpy(), s.page_size, mu)
    assert np.array_equal(ul.cpu().numpy(), ul_r) and np.array_equal(up.cpu().numpy(), up_r)
    assert np.array_equal(uc.cpu().numpy(), uc_r)
    bl = ul[:, None, :].expand(-1, s.num_kv_heads, -1).contiguous()        # the same table for every KV head
    bp = up[:, None, :].expand(-1, s.num_kv_heads, -1).contiguous()
    bc = uc[:, None].expand(-1, s.num_kv_heads).contiguous()
    out = torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev)
    lse = torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    ctx.sparse_paged_decode(w.q, pool, pt, bp, bl, bc, mu, out, lse)
    torch.cuda.synchronize()
    o_ref, l_ref = oracle_attention_on(w, bl.cpu().numpy(), bc.cpu().numpy())
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)
    ctx.close()
