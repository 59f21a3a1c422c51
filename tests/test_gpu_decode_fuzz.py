"""vx_sparse_paged_decode on arbitrary selection lists (-m gpu): random subsets of each request's pages in RANDOM
order (the call does not require the ascending order vx_topk_pages emits), counts from 1 page up to the budget,
fewer pages than split CTAs, the partial last page anywhere in the list -- against the oracle on the same lists."""
import numpy as np
import pytest
import torch

from tests.oracle_io import to_oracle
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
