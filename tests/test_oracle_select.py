"""Pins for the oracle's summary, score and top-k.

PAPER.md:546 (key envelope), :552 (per-head envelope score), :92 (arg-top-k),
:280 (first + last blocks forced).  Brute force, invariants and special cases only.
"""
import itertools

import numpy as np
import pytest

from oracle import vx_oracle as vo
from tests.test_oracle_attention import make_pool, table


def gathered_keys(pool, pt, i, j, kvh):
    """valid keys of logical page j of request i, float64 [t, d] (plain numpy indexing)."""
    n = int(pt.seq_lens[i])
    phys = pt.page_indices[pt.page_indptr[i] + j]
    t_end = min(pt.page_size, n - j * pt.page_size)
    return pool.k[phys, kvh, :t_end].astype(np.float64)


# ------------------------------------------------------------------ summary
def test_summary_is_attained_envelope_and_ignores_stale_slots():
    rng = np.random.default_rng(0)
    hkv, b, d = 2, 4, 6
    pool = make_pool(rng, 12, hkv, b, d)
    pt = table(rng, [10, 7], b, 12)
    for i in range(2):                          # poison the invalid slots of each partial last page
        n = int(pt.seq_lens[i]); j = (n - 1) // b
        phys = pt.page_indices[pt.page_indptr[i] + j]
        pool.k[phys, :, n - j * b:, ::2] = 1e30
        pool.k[phys, :, n - j * b:, 1::2] = -1e30
    summ = vo.page_summary(pool, pt, hkv, d)
    used = set(pt.page_indices.tolist())
    for p in range(12):
        if p not in used:
            assert np.isnan(summ[p]).all()      # untouched
    for i in range(2):
        for j in range(pt.page_indptr[i + 1] - pt.page_indptr[i]):
            phys = pt.page_indices[pt.page_indptr[i] + j]
            for kvh in range(hkv):
                keys = gathered_keys(pool, pt, i, j, kvh)
                mn, mx = summ[phys, kvh, 0], summ[phys, kvh, 1]
                assert (mn <= keys).all() and (keys <= mx).all()
                assert ((keys == mn).any(0)).all() and ((keys == mx).any(0)).all()   # bounds attained
                assert np.abs(mx).max() < 1e29


def test_summary_append_by_append_equals_bulk():
    # grow a sequence token by token, rebuilding only the last page each time (G12)
    rng = np.random.default_rng(1)
    hkv, b, d = 1, 4, 5
    pool = make_pool(rng, 6, hkv, b, d)
    full = table(rng, [19], b, 6)
    summ = np.full((6, hkv, 2, d), np.nan)
    for n in range(1, 20):
        P = (n + b - 1) // b
        pt = vo.PageTable([0, P], full.page_indices[:P], [n], b)
        vo.page_summary(pool, pt, hkv, d, first_page=[(n - 1) // b], summary=summ)
    bulk = vo.page_summary(pool, full, hkv, d)
    assert np.array_equal(summ, bulk, equal_nan=True)


# ------------------------------------------------------------------ score
@pytest.mark.parametrize("agg", [vo.AGG_SUM, vo.AGG_MAX])
def test_score_upper_bounds_every_key_dot_product(agg):
    rng = np.random.default_rng(2)
    hq, hkv, b, d = 6, 2, 4, 8
    g = hq // hkv
    pool = make_pool(rng, 12, hkv, b, d)
    pt = table(rng, [18, 9], b, 12)
    q = rng.standard_normal((2, hq, d)).astype(np.float32)
    summ = vo.page_summary(pool, pt, hkv, d)
    u, s = vo.page_score(q, summ, pt, hq, hkv, agg)
    slack = []
    for i in range(2):
        for j in range(pt.page_indptr[i + 1] - pt.page_indptr[i]):
            col = pt.page_indptr[i] + j
            for kvh in range(hkv):
                keys = gathered_keys(pool, pt, i, j, kvh)
                dots = keys @ q[i, kvh * g:(kvh + 1) * g].astype(np.float64).T      # [t, g]
                assert (u[kvh * g:(kvh + 1) * g, col][None, :] >= dots - 1e-12).all()
                if agg == vo.AGG_SUM:
                    assert s[kvh, col] >= dots.sum(1).max() - 1e-12
                    assert abs(s[kvh, col] - u[kvh * g:(kvh + 1) * g, col].sum()) < 1e-12
                else:
                    assert s[kvh, col] >= dots.max() - 1e-12
                    assert s[kvh, col] == u[kvh * g:(kvh + 1) * g, col].max()
                slack.append(u[kvh * g:(kvh + 1) * g, col] - dots.max(0))
    assert np.min(slack) >= -1e-12 and np.max(slack) > 0.1     # a bound, and not vacuous equality


def test_score_is_tight_when_page_keys_are_identical_or_page_size_one():
    rng = np.random.default_rng(3)
    hq, hkv, d = 4, 2, 8
    q = rng.standard_normal((1, hq, d)).astype(np.float32)
    # (a) all keys of a page identical -> u = q . k exactly that dot product
    pool = make_pool(rng, 4, hkv, 4, d)
    pool.k[:] = pool.k[:, :, :1]
    pt = table(rng, [16], 4, 4)
    u, _ = vo.page_score(q, vo.page_summary(pool, pt, hkv, d), pt, hq, hkv)
    for j in range(4):
        for h in range(hq):
            k0 = pool.k[pt.page_indices[j], h // 2, 0].astype(np.float64)
            assert abs(u[h, j] - q[0, h].astype(np.float64) @ k0) < 1e-12
    # (b) page_size = 1 -> page score = token score, so selection = token-level top-k of sum_h q_h.k_t
    pool1 = make_pool(rng, 40, hkv, 1, d)
    pt1 = table(rng, [33], 1, 40)
    _, s1 = vo.page_score(q, vo.page_summary(pool1, pt1, hkv, d), pt1, hq, hkv)
    sl, _, sc, _ = vo.topk_pages(s1, pt1, [7], 0, 0, 7)
    for kvh in range(hkv):
        tok = pool1.k[pt1.page_indices, kvh, 0].astype(np.float64) @ q[0, kvh * 2:(kvh + 1) * 2].astype(np.float64).sum(0)
        np.testing.assert_allclose(s1[kvh], tok, atol=1e-12)
        assert set(sl[0, kvh, :7].tolist()) == set(np.argsort(-tok, kind="stable")[:7].tolist())


def test_sum_score_collapses_to_one_dot_product_per_page():
    # sum_h u[h,j] = Q+ . M_j + Q- . m_j   with Q+ = sum_h max(q_h,0), Q- = sum_h min(q_h,0)   (G2)
    rng = np.random.default_rng(4)
    hq, hkv, b, d = 8, 2, 4, 16
    pool = make_pool(rng, 10, hkv, b, d)
    pt = table(rng, [37], b, 10)
    q = rng.standard_normal((1, hq, d)).astype(np.float32)
    summ = vo.page_summary(pool, pt, hkv, d)
    _, s = vo.page_score(q, summ, pt, hq, hkv, vo.AGG_SUM)
    qd = q[0].astype(np.float64).reshape(hkv, hq // hkv, d)
    qp, qm = np.maximum(qd, 0).sum(1), np.minimum(qd, 0).sum(1)
    for j in range(10):
        phys = pt.page_indices[j]
        for kvh in range(hkv):
            assert abs(s[kvh, j] - (qp[kvh] @ summ[phys, kvh, 1] + qm[kvh] @ summ[phys, kvh, 0])) < 1e-12


def test_score_uses_the_right_request_query_and_is_unscaled():
    rng = np.random.default_rng(5)
    hq, hkv, b, d = 2, 1, 4, 8
    pool = make_pool(rng, 12, hkv, b, d)
    pt = table(rng, [12, 20], b, 12)
    q = rng.standard_normal((2, hq, d)).astype(np.float32)
    summ = vo.page_summary(pool, pt, hkv, d)
    _, s = vo.page_score(q, summ, pt, hq, hkv)
    _, s2 = vo.page_score((2 * q).astype(np.float32), summ, pt, hq, hkv)
    np.testing.assert_allclose(s2, 2 * s, rtol=1e-14)                    # positively homogeneous, no extra scale
    pt_b = vo.PageTable([0, 5], pt.page_indices[3:], [20], b)            # request 1 alone
    _, sb = vo.page_score(np.ascontiguousarray(q[1:]), summ, pt_b, hq, hkv)
    assert np.array_equal(sb[:, :], s[:, 3:])


# ------------------------------------------------------------------ top-k
def brute_select(scores, P, k, n_sink, n_local):
    """forced pages, then full sort of the rest by (score desc, index asc)."""
    if k >= P:
        return list(range(P))
    forced = sorted(set(range(min(n_sink, P))) | set(range(max(P - n_local, 0), P)))
    rest = [j for j in range(P) if j not in forced]
    rest.sort(key=lambda j: (-scores[j], j))
    return sorted(forced + rest[: max(k - len(forced), 0)])


def one_request_table(P, b=4, n=None):
    return vo.PageTable([0, P], np.arange(P)[::-1] + 3, [n if n else P * b], b)   # phys = reversed + 3


@pytest.mark.parametrize("n_sink,n_local", [(0, 0), (1, 1), (1, 2), (2, 3), (0, 4)])
def test_topk_grid_against_sort_and_forced_pages(n_sink, n_local):
    rng = np.random.default_rng(6)
    for P in [1, 2, 3, 5, 8, 13]:
        for k in range(max(1, n_sink + n_local), 16):
            pt = one_request_table(P)
            s = rng.standard_normal((2, P))
            s[1] = np.round(s[1] * 2) / 2                                 # many exact ties on head 1
            sl, sp, sc, _ = vo.topk_pages(s, pt, [k], n_sink, n_local, 16)
            for kvh in range(2):
                want = brute_select(s[kvh], P, k, n_sink, n_local)
                got = sl[0, kvh, : sc[0, kvh]].tolist()
                assert got == want, (P, k, kvh)
                assert sc[0, kvh] == min(k, P)
                assert (sl[0, kvh, sc[0, kvh]:] == -1).all() and (sp[0, kvh, sc[0, kvh]:] == -1).all()
                assert sp[0, kvh, : sc[0, kvh]].tolist() == [pt.page_indices[j] for j in want]
                for j in list(range(min(n_sink, P))) + list(range(max(P - n_local, 0), P)):
                    assert j in got                                       # sink / local always kept


def test_topk_is_the_max_sum_subset_by_enumeration():
    rng = np.random.default_rng(7)
    for P, k, ns, nl in [(9, 4, 1, 1), (12, 6, 1, 2), (10, 3, 0, 0), (11, 5, 2, 2)]:
        s = rng.standard_normal((1, P))
        sl, _, sc, _ = vo.topk_pages(s, one_request_table(P), [k], ns, nl, k)
        forced = set(range(ns)) | set(range(P - nl, P))
        free = [j for j in range(P) if j not in forced]
        best = max(itertools.combinations(free, k - len(forced)), key=lambda c: s[0, list(c)].sum())
        assert set(sl[0, 0, :k].tolist()) == forced | set(best)


def test_topk_tie_break_prefers_lower_logical_index_and_reports_threshold():
    s = np.array([[9.0, 1.0, 5.0, 5.0, 5.0, 5.0, 0.0, 7.0, 5.0, 9.0]])
    sl, _, sc, thr = vo.topk_pages(s, one_request_table(10), [5], 1, 1, 5)
    # forced {0, 9}; candidates by score: 7(7.0), then ties 2,3,4,5,8 at 5.0 -> take 2, 3
    assert sl[0, 0].tolist() == [0, 2, 3, 7, 9] and thr[0, 0] == 5.0
    sl, _, sc, thr = vo.topk_pages(s, one_request_table(10), [10], 1, 1, 10)
    assert sc[0, 0] == 10 and np.isnan(thr[0, 0])


def test_topk_ragged_batch_uses_each_requests_rows_and_budget():
    rng = np.random.default_rng(8)
    pt = vo.PageTable([0, 5, 5 + 9, 5 + 9 + 3], rng.permutation(40)[:17], [20, 33, 12], 4)
    s = rng.standard_normal((3, 17))
    budget = [4, 6, 8]
    sl, sp, sc, _ = vo.topk_pages(s, pt, budget, 1, 2, 8)
    for i, (o, P) in enumerate([(0, 5), (5, 9), (14, 3)]):
        for kvh in range(3):
            want = brute_select(s[kvh, o:o + P], P, budget[i], 1, 2)
            assert sl[i, kvh, : sc[i, kvh]].tolist() == want
            assert sp[i, kvh, : sc[i, kvh]].tolist() == pt.page_indices[o + np.array(want)].tolist()


def test_topk_rejects_more_forced_pages_than_budget():
    with pytest.raises(ValueError):
        vo.topk_pages(np.zeros((1, 10)), one_request_table(10), [3], 2, 2, 3)


def test_full_budget_step_equals_dense_attention():
    # whole pipeline: budget >= P  =>  every page selected  =>  dense attention, bit for bit
    import torch
    from paper_2606_06453_b200.workloads import SPECS, make_workload
    from dataclasses import replace
    from oracle.workload_io import oracle_step, to_oracle
    spec = replace(SPECS["C1"], budget=64)
    w = make_workload(spec)
    r = oracle_step(w)
    q, pool, pt = to_oracle(w)
    od, ld = vo.dense_attention(q, pool, pt, 4, 1, 64, 64, spec.sm_scale)
    assert (r["sel_count"] == 64).all()
    assert np.array_equal(r["out"], od) and np.array_equal(r["lse"], ld)
