"""Pins for the approximate radix top-k oracle (oracle/vx_oracle_approx.py).

The paper prints no worked example, so the pins are: tolerate_ratio 0 == the exact oracle (an independent
full-sort implementation in vx_oracle.c) and == brute force; the published SplitMix64 vector; the error bound
the method states (recall@k >= 1 - tolerate_ratio); structural invariants; the sampler's inclusion frequency.
"""
import os

import numpy as np
import pytest

from oracle import vx_oracle as vo
from oracle import vx_oracle_approx as va
from paper_2606_06453_b200.workloads import APPD_DISTRIBUTIONS, appd_scores

HERE = os.path.dirname(os.path.abspath(__file__))


def exact_sets(scores, P_list, budget, n_sink, n_local, max_budget, page_size=16):
    indptr = np.concatenate([[0], np.cumsum(P_list)]).astype(np.int32)
    pt = vo.PageTable(indptr, np.arange(indptr[-1], dtype=np.int32),
                      np.array([p * page_size for p in P_list], dtype=np.int32), page_size)
    sl, _, sc, _ = vo.topk_pages(scores.astype(np.float64), pt, budget, n_sink, n_local, max_budget)
    return indptr, pt, sl, sc


def test_splitmix64_published_vector():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "splitmix64.txt")) if not l.startswith("#")]
    assert len(rows) == 5
    for seed, idx, val in rows:
        assert va.splitmix64(int(seed), int(idx)) == int(val)


def test_keys_preserve_order_and_merge_zeros():
    x = np.array([-np.inf, -3.5, -1e-40, -0.0, 0.0, 1e-40, 2.0, 900.0, np.inf], dtype=np.float32)
    k = va.float_keys(x).astype(np.int64)
    assert (np.diff(k) >= 0).all() and k[3] == k[4] and (np.diff(k)[[0, 1, 2, 4, 5, 6, 7]] > 0).all()
    back = va.key_floats(va.float_keys(x))
    assert np.array_equal(back[[0, 1, 2, 5, 6, 7, 8]], x[[0, 1, 2, 5, 6, 7, 8]])


@pytest.mark.parametrize("dist", APPD_DISTRIBUTIONS)
def test_ratio_zero_is_the_exact_selection(dist):
    hkv, P_list, k = 2, [700, 2048, 300], 64
    T = sum(P_list)
    scores = appd_scores(dist, (hkv, T), seed=11).numpy()
    budget = np.full(len(P_list), k, dtype=np.int32)
    indptr, pt, sl_e, sc_e = exact_sets(scores, P_list, budget, 1, 2, k)
    sl, sp, sc, early = va.approx_topk_pages(scores, indptr, pt.page_indices, pt.seq_lens, 16, budget, 1, 2, k, 0.0, 5)
    assert not early.any()
    assert np.array_equal(sc, sc_e) and np.array_equal(sl, sl_e)


def test_ratio_zero_heavy_ties_and_sign_spanning_ranges():
    rng = np.random.default_rng(3)
    for trial in range(30):
        P = int(rng.integers(20, 900))
        k = int(rng.integers(4, min(P, 200)))
        kind = trial % 3
        if kind == 0:
            s = rng.integers(-3, 4, size=(1, P)).astype(np.float32)               # heavy ties, +-0
        elif kind == 1:
            s = (rng.standard_normal((1, P)) * 10.0 ** rng.integers(-20, 20)).astype(np.float32)
        else:
            s = np.round(rng.standard_normal((1, P)) * 4).astype(np.float32) / 4 + 1000.0
        budget = np.array([k], dtype=np.int32)
        indptr, pt, sl_e, sc_e = exact_sets(s, [P], budget, 1, 2, k)
        sl, _, sc, _ = va.approx_topk_pages(s, indptr, pt.page_indices, pt.seq_lens, 16, budget, 1, 2, k, 0.0, trial)
        assert np.array_equal(sl, sl_e), (trial, P, k)


def test_ratio_zero_ties_at_the_top_edge_of_a_float_bin():
    """Round-1 advisor finding: a heavy float-pass bin is handed over as the UNALIGNED key interval [bmin, bmax]; when
    its last integer sub-bin is heavy again the recursion window must end at bmax, or the first key of the next
    float bin is counted twice.  Scores {-1, 3, b + 1 ulp, b - 3000 ulp, 300 x b}, b = 1 - 2^-23 = the last fp32 value
    of float bin 1023 of the range [-1, 3].  Expected value: the exact C oracle (full sort)."""
    b = np.float32(1.0) - np.float32(2.0 ** -23)
    up = np.nextafter(b, np.float32(2.0))
    down = (b.view(np.uint32) - np.uint32(3000)).view(np.float32)
    s = np.array([-1.0, 3.0, up, down] + [b] * 300, dtype=np.float32)[None]
    for k in (3, 50, 102, 200, 302):
        budget = np.array([k], dtype=np.int32)
        indptr, pt, sl_e, sc_e = exact_sets(s, [s.shape[1]], budget, 0, 0, k)
        sel, info = va.select_one(s[0], k, 0, 0, 0.0, 0, 0)
        assert sel.shape[0] == k and len(set(sel.tolist())) == k
        assert sel.tolist() == sl_e[0, 0, :k].tolist(), k
        if 3 <= k <= 302:
            assert info["passes"] >= 3                                    # float pass -> integer pass -> recursion
    rng = np.random.default_rng(9)
    for trial in range(20):                                               # the same values in random order and counts
        n = int(rng.integers(300, 1500))
        row = rng.choice(np.array([-1.0, 3.0, up, down, b], np.float32), size=n, p=[0.05, 0.05, 0.1, 0.1, 0.7])
        k = int(rng.integers(3, n))
        budget = np.array([k], dtype=np.int32)
        indptr, pt, sl_e, _ = exact_sets(row[None], [n], budget, 1, 2, k)
        sel, _ = va.select_one(row, k, 1, 2, 0.0, 0, 0)
        assert sel.tolist() == sl_e[0, 0, :k].tolist(), (trial, n, k)


def test_ratio_zero_brute_force_tiny():
    rng = np.random.default_rng(4)
    for trial in range(200):
        P = int(rng.integers(1, 13))
        n_sink, n_local = int(rng.integers(0, 3)), int(rng.integers(0, 3))
        k = int(rng.integers(n_sink + n_local, max(n_sink + n_local + 1, P + 3)))
        if k == 0:
            continue
        s = rng.integers(0, 5, size=P).astype(np.float32) if trial % 2 else rng.standard_normal(P).astype(np.float32)
        forced = [j for j in range(P) if j < n_sink or j >= P - n_local]
        rest = sorted((j for j in range(P) if j not in forced), key=lambda j: (-float(s[j]), j))
        want = sorted(set(forced) | set(rest[:max(0, k - len(forced))])) if k < P else list(range(P))
        got, _ = va.select_one(s, k, n_sink, n_local, 0.0, 0, 0)
        assert got.tolist() == want, (trial, P, k, n_sink, n_local)


@pytest.mark.parametrize("dist", APPD_DISTRIBUTIONS)
@pytest.mark.parametrize("tau", [0.05, 0.25, 1.0])
def test_invariants_and_error_bound(dist, tau):
    P, k, n_sink, n_local = 4096, 128, 1, 2
    scores = appd_scores(dist, (4, P), seed=21).numpy()
    any_early = False
    for h in range(4):
        s = scores[h]
        exact, _ = va.select_one(s, k, n_sink, n_local, 0.0, 0, h)
        indptr, pt, sl_e, _ = exact_sets(s[None], [P], np.array([k], np.int32), n_sink, n_local, k)
        assert exact.tolist() == sl_e[0, 0].tolist()
        sel, info = va.select_one(s, k, n_sink, n_local, tau, 99, h)
        any_early |= info["early"]
        assert sel.shape[0] == k and len(set(sel.tolist())) == k and (np.diff(sel) > 0).all()
        assert {0, P - 2, P - 1} <= set(sel.tolist())                       # PAPER.md:280 forced pages
        ex = set(exact.tolist())
        assert set(info["sure"].tolist()) <= ex                             # high-confidence candidates are exact
        wrong = [j for j in sel.tolist() if j not in ex]
        assert len(wrong) <= int(np.floor(np.float32(tau) * np.float32(k)))  # the method's error bound
        assert va.recall_at_k(sel, exact) >= 1.0 - tau - 1e-12
        if info["early"]:
            assert set(wrong) <= set(info["members"].tolist())
            if info["passes"] == 1:                                         # wrong picks: within one bin of the threshold
                thr = min(float(s[j]) for j in ex if j not in (0, P - 2, P - 1))
                w = info["bin_width"] * (1 + 1e-5) + 1e-30
                assert all(abs(float(s[j]) - thr) <= w for j in wrong)
        else:
            assert sel.tolist() == exact.tolist()
    if tau == 1.0:
        assert any_early                                                    # ratio 1 stops after the first pass


def test_sampler_inclusion_frequency_is_need_over_cnt():
    P, k = 600, 40
    s = np.zeros(P, dtype=np.float32)
    s[:] = 5.0                                                              # one huge tie ... but not a single key:
    s += (np.arange(P) % 7).astype(np.float32) * 1e-4                       # seven close values in one float bin
    s[100] = 50.0                                                           # widen the range: all others share a bin
    hits = np.zeros(P)
    n = 400
    for seed in range(n):
        sel, info = va.select_one(s, k, 1, 2, 1.0, seed, 0)
        assert info["early"] and 100 in sel.tolist()
        hits[sel] += 1
    members = info["members"]
    need = info["need"]
    freq = hits[members] / n
    assert abs(freq.mean() - need / len(members)) < 1e-9                    # exactly need picks per draw
    assert freq.max() < 3 * need / len(members) and freq.min() > 0          # no member favoured or starved


# ---- the offline-profiled monotone remap (App. D.2; reading G29) ---------------------------------

def _knot_tables(rng):
    """identity, two extreme shapes, a flat table (every page in bin 0) and random monotone tables"""
    yield np.array([0.0, 1.0], dtype=np.float32)
    yield np.linspace(0, 1, 65, dtype=np.float32) ** 3
    yield np.sqrt(np.linspace(0, 1, 17, dtype=np.float32))
    yield np.zeros(9, dtype=np.float32)
    yield np.array([0.0, 0.0, 1.0, 1.0, 1.0], dtype=np.float32)
    for n in (2, 3, 33, 65):
        u = np.sort(rng.random(n)).astype(np.float32)
        yield u


def test_remap_bins_never_decrease_with_the_score():
    """the one property the selection needs of f (reading G29): the first-pass bin is non-decreasing in the score,
    across knots and whatever the fp32 rounding -- checked on every fp32 value of a dense score range"""
    rng = np.random.default_rng(7)
    lo = np.float32(0.37)
    dense = np.arange(np.float32(lo).view(np.uint32), np.float32(lo).view(np.uint32) + 300000, dtype=np.uint32).view(np.float32)
    wide = np.sort(np.concatenate([-np.geomspace(1e-6, 50, 4000), np.geomspace(1e-7, 900, 6000)]).astype(np.float32))
    for knots in _knot_tables(rng):
        for sc in (dense, wide):
            b = va.remap_bins(sc, sc[0], sc[-1], knots)
            assert (np.diff(b) >= 0).all() and b.min() >= 0 and b.max() <= va.K_BINS - 1


@pytest.mark.parametrize("dist", APPD_DISTRIBUTIONS)
def test_ratio_zero_with_any_remap_is_the_exact_selection(dist):
    """a monotone f only reshapes the first pass's bins: with tolerate_ratio 0 the selection is still the exact one"""
    rng = np.random.default_rng(21)
    hkv, P_list, k = 2, [700, 2048, 300], 64
    scores = appd_scores(dist, (hkv, sum(P_list)), seed=13).numpy()
    budget = np.full(len(P_list), k, dtype=np.int32)
    indptr, pt, sl_e, sc_e = exact_sets(scores, P_list, budget, 1, 2, k)
    for knots in _knot_tables(rng):
        sl, sp, sc, early = va.approx_topk_pages(scores, indptr, pt.page_indices, pt.seq_lens, 16, budget, 1, 2, k, 0.0, 5,
                                                 remap=knots)
        assert not early.any() and np.array_equal(sc, sc_e) and np.array_equal(sl, sl_e)


def test_ratio_zero_with_remap_on_ties_and_sign_spanning_ranges():
    rng = np.random.default_rng(5)
    tables = list(_knot_tables(rng))
    for trial in range(24):
        P = int(rng.integers(20, 900))
        k = int(rng.integers(4, min(P, 200)))
        kind = trial % 3
        if kind == 0:
            s = rng.integers(0, 4, size=P).astype(np.float32)                       # heavy ties
        elif kind == 1:
            s = (rng.standard_normal(P) * 10 ** rng.uniform(-20, 20, size=P)).astype(np.float32)   # 40 decades, both signs
        else:
            s = rng.standard_normal(P).astype(np.float32)
        budget = np.array([k], dtype=np.int32)
        indptr, pt, sl_e, sc_e = exact_sets(s[None, :], [P], budget, 1, 1, k)
        sl, _, sc, early = va.approx_topk_pages(s[None, :], indptr, pt.page_indices, pt.seq_lens, 16, budget, 1, 1, k, 0.0, 9,
                                                remap=tables[trial % len(tables)])
        assert not early.any() and np.array_equal(sc, sc_e) and np.array_equal(sl, sl_e), (trial, kind)


@pytest.mark.parametrize("dist", APPD_DISTRIBUTIONS)
@pytest.mark.parametrize("ratio", [0.1, 0.5])
def test_remap_keeps_the_recall_bound_and_the_sure_picks(dist, ratio):
    from paper_2606_06453_b200.remap_profile import profile_knots
    hkv, P_list, k = 1, [4096, 1500], 128
    scores = appd_scores(dist, (hkv, sum(P_list)), seed=17).numpy()
    knots = profile_knots(appd_scores(dist, (8, 4096), seed=99).numpy(), 33)       # profiled on OTHER draws of the distribution
    budget = np.full(len(P_list), k, dtype=np.int32)
    indptr, pt, sl_e, sc_e = exact_sets(scores, P_list, budget, 1, 2, k)
    for seed in range(4):
        sl, sp, sc, early = va.approx_topk_pages(scores, indptr, pt.page_indices, pt.seq_lens, 16, budget, 1, 2, k, ratio, seed,
                                                 remap=knots)
        assert np.array_equal(sc, sc_e)
        for i, P in enumerate(P_list):
            got, exact = sl[i, 0, :sc[i, 0]], sl_e[i, 0, :sc_e[i, 0]]
            assert (np.diff(got) > 0).all() and got[0] == 0 and set(range(P - 2, P)) <= set(got.tolist())
            assert va.recall_at_k(got, exact) >= 1.0 - ratio - 1e-9
            row = scores[0, indptr[i]:indptr[i] + P]
            _, info = va.select_one(row, k, 1, 2, ratio, seed, i, knots)
            assert set(info["sure"].tolist()) <= set(exact.tolist())


def test_profiled_remap_spreads_the_first_pass():
    """what the offline profile is for ("improves bin separation"): under the table fitted to a distribution the
    fullest first-pass bin holds far fewer pages than under the linear map; the table is a valid knot table"""
    from paper_2606_06453_b200.remap_profile import profile_knots
    for dist in ("lognormal", "bimodal"):
        knots = va.check_knots(profile_knots(appd_scores(dist, (16, 8192), seed=3).numpy(), 65))
        assert knots[0] == 0.0 and knots[-1] == 1.0
        s = np.sort(appd_scores(dist, (1, 8192), seed=4).numpy()[0])
        lin = np.minimum(va.K_BINS - 1, ((s - s[0]) * (np.float32(va.K_BINS) / (s[-1] - s[0]))).astype(np.int64))
        rem = va.remap_bins(s, s[0], s[-1], knots)
        assert np.bincount(rem).max() * 3 <= np.bincount(lin).max()
