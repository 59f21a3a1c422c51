"""Pins for oracle/vx_oracle_union.py (PAPER.md:538 `TopK, Union`): hand-worked cases and set identities."""
import numpy as np

from oracle import vx_oracle as vo
from oracle import vx_oracle_union as vu


def table(pages, b=16, seed=0):
    rng = np.random.default_rng(seed)
    indptr = np.concatenate([[0], np.cumsum(pages)]).astype(np.int32)
    T = int(indptr[-1])
    return indptr, rng.permutation(T + 5)[:T].astype(np.int32), np.array([p * b - 3 for p in pages], np.int32)


def test_hand_worked_case():
    indptr, idx, seq = table([10, 6])
    sel = np.full((2, 3, 4), -1, np.int32)
    cnt = np.zeros((2, 3), np.int32)
    sel[0, 0, :4] = [0, 3, 8, 9]; cnt[0, 0] = 4
    sel[0, 1, :4] = [0, 2, 3, 9]; cnt[0, 1] = 4
    sel[0, 2, :3] = [0, 7, 9];    cnt[0, 2] = 3
    sel[1, 0, :2] = [0, 5];       cnt[1, 0] = 2
    sel[1, 1, :2] = [0, 5];       cnt[1, 1] = 2
    sel[1, 2, :4] = [1, 5, 9, 0]; cnt[1, 2] = 2        # entries past the count (9, 0) must be ignored
    ul, up, uc = vu.union_pages(sel, cnt, indptr, idx, seq, 16, 8)
    assert uc.tolist() == [6, 3]
    assert ul[0].tolist() == [0, 2, 3, 7, 8, 9, -1, -1]
    assert ul[1].tolist() == [0, 1, 5, -1, -1, -1, -1, -1]
    assert up[0, :6].tolist() == [int(idx[j]) for j in [0, 2, 3, 7, 8, 9]]
    assert up[1, :3].tolist() == [int(idx[10 + j]) for j in [0, 1, 5]] and (up[1, 3:] == -1).all()


def test_set_identities_on_real_selections():
    rng = np.random.default_rng(1)
    pages, hkv, k = [300, 77, 1200], 4, 32
    indptr, idx, seq = table(pages, seed=2)
    T = int(indptr[-1])
    scores = rng.standard_normal((hkv, T))
    pt = vo.PageTable(indptr, idx, seq, 16)
    budget = np.full(3, k, np.int32)
    sl, sp, sc, _ = vo.topk_pages(scores, pt, budget, 1, 2, k)
    ul, up, uc = vu.union_pages(sl, sc, indptr, idx, seq, 16, hkv * k)
    for i, P in enumerate(pages):
        sets = [set(sl[i, h, :sc[i, h]].tolist()) for h in range(hkv)]
        got = ul[i, :uc[i]].tolist()
        assert got == sorted(set().union(*sets))                       # ascending, deduplicated
        assert max(len(s) for s in sets) <= uc[i] <= min(P, sum(len(s) for s in sets))
        assert {0, P - 2, P - 1} <= set(got)                           # PAPER.md:280 forced pages survive
        assert up[i, :uc[i]].tolist() == [int(idx[indptr[i] + j]) for j in got]
        assert (ul[i, uc[i]:] == -1).all() and (up[i, uc[i]:] == -1).all()
    # identical heads -> that head's set; idempotent; head / entry permutations change nothing
    same = np.repeat(sl[:, :1], hkv, axis=1)
    ul1, _, uc1 = vu.union_pages(same, np.repeat(sc[:, :1], hkv, axis=1), indptr, idx, seq, 16, hkv * k)
    assert np.array_equal(ul1[:, :k], sl[:, 0]) and (uc1 == sc[:, 0]).all()
    again = ul[:, None, :].copy()
    ul2, _, uc2 = vu.union_pages(again, uc[:, None], indptr, idx, seq, 16, hkv * k)
    assert np.array_equal(ul2, ul) and np.array_equal(uc2, uc)
    perm = sl[:, ::-1, ::-1].copy()                                     # heads reversed, entries reversed (pads first)
    for i in range(3):
        for h in range(hkv):
            row = perm[i, h]
            perm[i, h] = np.concatenate([row[row >= 0], row[row < 0]])
    ul3, _, uc3 = vu.union_pages(perm, sc[:, ::-1].copy(), indptr, idx, seq, 16, hkv * k)
    assert np.array_equal(ul3, ul) and np.array_equal(uc3, uc)


def test_disjoint_heads_concatenate_and_out_of_range_is_ignored():
    indptr, idx, seq = table([64])
    sel = np.full((1, 2, 8), -1, np.int32)
    sel[0, 0] = np.arange(0, 16, 2)
    sel[0, 1] = np.arange(1, 16, 2)
    cnt = np.array([[8, 8]], np.int32)
    ul, _, uc = vu.union_pages(sel, cnt, indptr, idx, seq, 16, 16)
    assert uc[0] == 16 and ul[0].tolist() == list(range(16))
    sel[0, 1, 0] = 64                                                   # P = 64: not a page of the request
    sel[0, 1, 1] = -1
    ul, _, uc = vu.union_pages(sel, cnt, indptr, idx, seq, 16, 16)
    assert uc[0] == 14 and 1 not in ul[0].tolist() and 3 not in ul[0].tolist()
