"""Hand-written selection cases (tests/golden/topk_cases.txt) against the oracle, and (gpu) against
vx_topk_pages.  The expected ids were worked out by hand from PAPER.md:280 / :92 Eq.3 and readings G4-G6."""
import os

import numpy as np
import pytest

from oracle import vx_oracle as vo

HERE = os.path.dirname(os.path.abspath(__file__))


def cases():
    out = []
    for line in open(os.path.join(HERE, "golden", "topk_cases.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        head, scores, want = (part.split() for part in line.split("|"))
        b, n, k, n_sink, n_local = (int(x) for x in head)
        out.append((b, n, k, n_sink, n_local, [float(x) for x in scores], [int(x) for x in want]))
    return out


CASES = cases()


def table_for(b, n, scores):
    P = (n + b - 1) // b
    assert P == len(scores), "fixture: one score per logical page"
    perm = np.arange(P, dtype=np.int32)[::-1].copy() + 3          # physical id = P + 2 - logical
    return P, vo.PageTable(np.array([0, P], np.int32), perm, np.array([n], np.int32), b)


@pytest.mark.parametrize("case", CASES, ids=[f"case{i}" for i in range(len(CASES))])
def test_oracle_topk_matches_hand_worked_cases(case):
    b, n, k, n_sink, n_local, scores, want = case
    P, pt = table_for(b, n, scores)
    sl, sp, sc, _ = vo.topk_pages(np.array([scores]), pt, [k], n_sink, n_local, max(k, 1))
    assert sc[0, 0] == len(want) == min(k, P)
    assert sl[0, 0, :len(want)].tolist() == want
    assert sp[0, 0, :len(want)].tolist() == [P + 2 - j for j in want]
    assert (sl[0, 0, len(want):] == -1).all()


@pytest.mark.gpu
@pytest.mark.parametrize("case", CASES, ids=[f"case{i}" for i in range(len(CASES))])
def test_gpu_topk_matches_hand_worked_cases(case):
    import torch
    import paper_2606_06453_b200 as vx
    b, n, k, n_sink, n_local, scores, want = case
    P, pt_o = table_for(b, n, scores)
    dev = "cuda:0"
    ctx = vx.Context(dtype=torch.bfloat16, num_q_heads=8, num_kv_heads=1, qk_dim=128, v_dim=128, page_size=b,
                     sm_scale=1.0, n_sink=n_sink, n_local=n_local, max_batch=1, max_total_pages=P,
                     max_pages_per_req=P, max_budget=max(k, 1), device=dev)
    pt = vx.PageTable(torch.from_numpy(pt_o.page_indptr).to(dev), torch.from_numpy(pt_o.page_indices).to(dev),
                      torch.from_numpy(pt_o.seq_lens).to(dev), P, P)
    mb = max(k, 1)
    sl = torch.full((1, 1, mb), -7, dtype=torch.int32, device=dev)
    sp = torch.full_like(sl, -7)
    sc = torch.full((1, 1), -7, dtype=torch.int32, device=dev)
    ctx.topk_pages(torch.tensor([scores], dtype=torch.float32, device=dev), pt,
                   torch.tensor([k], dtype=torch.int32, device=dev), mb, sp, sl, sc)
    torch.cuda.synchronize()
    assert int(sc[0, 0]) == len(want)
    assert sl[0, 0, :len(want)].tolist() == want
    assert sp[0, 0, :len(want)].tolist() == [P + 2 - j for j in want]
    assert (sl[0, 0, len(want):] == -1).all() and (sp[0, 0, len(want):] == -1).all()
