"""Pins for the oracle's block top-k flow (section 3.1: centroid = mean of the block's keys,
score = mean over the head group of q . centroid, arg-top-k).  Closed forms, hand-worked roundings, invariants
and the b = 1 special case (which reduces to exact token-level top-k) -- none of them re-uses the oracle's code."""
import numpy as np

from oracle import vx_oracle as vo
from tests.test_oracle_attention import make_pool, table
from tests.test_oracle_select import gathered_keys


def bf16_bits(x):
    """float (exactly representable in bf16) -> uint16 bit pattern."""
    a = np.ascontiguousarray(x, dtype=np.float32)
    bits = a.view(np.uint32)
    assert ((bits & 0xFFFF) == 0).all(), "test value must be exact in bf16"
    return (bits >> 16).astype(np.uint16)


def one_page_pool_bf16(values):
    """pool of one page, one head, one channel per column of `values` [tokens, channels]."""
    v = np.ascontiguousarray(values, dtype=np.float32)
    t, d = v.shape
    k = bf16_bits(v).reshape(1, 1, t, d)
    pool = vo.Pool(k=k, v=k, stride_page=t * d, stride_token=d, stride_head=t * d, num_pool_pages=1)
    pt = vo.PageTable([0, 1], [0], [t], t)
    return pool, pt


def test_centroid_closed_forms_partial_pages_and_stale_slots():
    rng = np.random.default_rng(0)
    hkv, b, d = 2, 4, 6
    pool = make_pool(rng, 12, hkv, b, d)            # fp32 pool: the mean is rounded once, to fp32
    pt = table(rng, [10, 7], b, 12)
    for i in range(2):                              # poison the invalid slots of each partial last page
        n = int(pt.seq_lens[i]); j = (n - 1) // b
        phys = pt.page_indices[pt.page_indptr[i] + j]
        pool.k[phys, :, n - j * b:, :] = 1e30
    cen = vo.page_centroid(pool, pt, hkv, d)
    used = set(pt.page_indices.tolist())
    for p in range(12):
        if p not in used:
            assert np.isnan(cen[p]).all()           # untouched
    for i in range(2):
        for j in range(pt.page_indptr[i + 1] - pt.page_indptr[i]):
            phys = pt.page_indices[pt.page_indptr[i] + j]
            for kvh in range(hkv):
                keys = gathered_keys(pool, pt, i, j, kvh)          # float64 [valid tokens, d]
                want = (keys.sum(0) / keys.shape[0]).astype(np.float32).astype(np.float64)
                assert np.array_equal(cen[phys, kvh], want)
                assert (keys.min(0) - 1e-6 <= cen[phys, kvh]).all() and (cen[phys, kvh] <= keys.max(0) + 1e-6).all()
    # identical keys -> the centroid is that key, exactly
    pool.k[:, :, :, :] = pool.k[:, :, :1, :]
    cen = vo.page_centroid(pool, pt, hkv, d)
    for p in used:
        assert np.array_equal(cen[p], pool.k[p, :, 0, :].astype(np.float64))


def test_centroid_rounds_the_exact_mean_to_bf16_nearest_even():
    # hand-worked: bf16 has 8 significand bits, its spacing in [1, 2) is 2^-7
    u = 2.0 ** -7
    cols = np.array([
        [1.0, 1.0 + u],            # mean 1 + u/2: tie between 1 and 1+u        -> even significand: 1.0
        [1.0 + u, 1.0 + 2 * u],    # mean 1 + 1.5u: tie between 1+u and 1+2u    -> even: 1 + 2u
        [1.0, 1.0 + 2 * u],        # mean 1 + u: representable                   -> 1 + u
        [-3.0, 5.0],               # mean 1.0
        [0.5, -0.5],               # mean 0
    ], dtype=np.float32).T         # [2 tokens, 5 channels]
    pool, pt = one_page_pool_bf16(cols)
    cen = vo.page_centroid(pool, pt, 1, cols.shape[1])
    assert cen[0, 0].tolist() == [1.0, 1.0 + 2 * u, 1.0 + u, 1.0, 0.0]
    # three tokens: mean of (1, 1, 1+u) = 1 + u/3 -> below the midpoint -> 1.0; (1, 1+u, 1+u) -> 1 + 2u/3 -> 1 + u
    pool, pt = one_page_pool_bf16(np.array([[1.0, 1.0], [1.0, 1.0 + u], [1.0 + u, 1.0 + u]], dtype=np.float32))
    cen = vo.page_centroid(pool, pt, 1, 2)
    assert cen[0, 0].tolist() == [1.0, 1.0 + u]


def test_centroid_append_by_append_equals_bulk():
    rng = np.random.default_rng(1)
    hkv, b, d = 1, 4, 5
    pool = make_pool(rng, 6, hkv, b, d)
    full = table(rng, [19], b, 6)
    cen = np.full((6, hkv, d), np.nan)
    for n in range(1, 20):
        P = (n + b - 1) // b
        pt = vo.PageTable([0, P], full.page_indices[:P], [n], b)
        vo.page_centroid(pool, pt, hkv, d, first_page=[(n - 1) // b], centroid=cen)
    assert np.array_equal(cen, vo.page_centroid(pool, full, hkv, d), equal_nan=True)


def test_centroid_score_is_group_sum_of_q_dot_centroid_with_the_right_query():
    rng = np.random.default_rng(2)
    hq, hkv, b, d = 6, 2, 4, 8
    pool = make_pool(rng, 16, hkv, b, d)
    pt = table(rng, [9, 13], b, 16)
    q = rng.standard_normal((2, hq, d)).astype(np.float32)
    cen = vo.page_centroid(pool, pt, hkv, d)
    u, s = vo.centroid_score(q, cen, pt, hq, hkv)
    g = hq // hkv
    for i in range(2):
        for j in range(pt.page_indptr[i + 1] - pt.page_indptr[i]):
            col = pt.page_indptr[i] + j
            phys = pt.page_indices[col]
            for h in range(hq):
                want = float(q[i, h].astype(np.float64) @ cen[phys, h // g])        # numpy matmul, not the oracle
                assert abs(u[h, col] - want) <= 1e-12 * max(1.0, abs(want))
            for kvh in range(hkv):
                qsum = q[i, kvh * g:(kvh + 1) * g].astype(np.float64).sum(0)
                assert abs(s[kvh, col] - qsum @ cen[phys, kvh]) <= 1e-12 * max(1.0, abs(s[kvh, col]))
    # unscaled (Eq.2 carries no softmax scale) and linear in q
    _, s2 = vo.centroid_score(2 * q, cen, pt, hq, hkv)
    assert np.allclose(s2, 2 * s, rtol=1e-13, atol=0)
    # for fp32 data the centroid score is the mean of the per-token dot products (up to the fp32 rounding of the mean)
    i, j, kvh = 1, 2, 1
    keys = gathered_keys(pool, pt, i, j, kvh)
    qsum = q[i, kvh * g:(kvh + 1) * g].astype(np.float64).sum(0)
    assert abs(s[kvh, pt.page_indptr[i] + j] - (keys @ qsum).mean()) <= 1e-5


def test_page_size_one_block_topk_is_exact_token_topk():
    # b = 1: the centroid of a block is its only key, so block top-k = token-level top-k of sum_h q_h . K_t
    rng = np.random.default_rng(3)
    hq, hkv, d, n, k = 4, 2, 8, 40, 9
    pool = make_pool(rng, 64, hkv, 1, d)
    pt = table(rng, [n], 1, 64)
    q = rng.standard_normal((1, hq, d)).astype(np.float32)
    ref = vo.decode_step(q, pool, pt, [k], k, hq, hkv, d, d, d ** -0.5, n_sink=1, n_local=2, kind="centroid")
    g = hq // hkv
    for kvh in range(hkv):
        keys = np.stack([pool.k[pt.page_indices[t], kvh, 0].astype(np.float64) for t in range(n)])
        dots = keys @ q[0, kvh * g:(kvh + 1) * g].astype(np.float64).sum(0)
        forced = {0, n - 2, n - 1}
        rest = sorted((t for t in range(n) if t not in forced), key=lambda t: (-dots[t], t))[: k - 3]
        assert ref["sel_logical"][0, kvh, :k].tolist() == sorted(forced | set(rest))
