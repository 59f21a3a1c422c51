"""Pins for the oracle's attention / combine (SURVEY.md 8(c) "What pins the oracle").

None of these re-type the oracle's formula: they are closed forms, invariants and
limit cases that a dropped term, wrong sign, transposed operand or wrong index breaks.
PAPER.md:92 Eq. 4 (softmax attention over selected tokens), :75 (Flash-Decoding split).
"""
import math

import numpy as np
import pytest

from oracle import vx_oracle as vo


def make_pool(rng, n_pool, hkv, b, d, dv=None, dtype=np.float32, shared=False):
    k = rng.standard_normal((n_pool, hkv, b, d)).astype(dtype)
    v = None if shared else rng.standard_normal((n_pool, hkv, b, dv or d)).astype(dtype)
    return vo.Pool(k=k, v=v, stride_page=hkv * b * d, stride_token=d, stride_head=b * d,
                   num_pool_pages=n_pool)


def table(rng, seq_lens, b, n_pool):
    pages = [(n + b - 1) // b for n in seq_lens]
    indptr = np.concatenate([[0], np.cumsum(pages)]).astype(np.int32)
    perm = rng.permutation(n_pool)[: indptr[-1]].astype(np.int32)
    return vo.PageTable(indptr, perm, np.array(seq_lens, np.int32), b)


def all_pages_sel(pt, hkv):
    P = np.diff(pt.page_indptr)
    mb = int(P.max())
    sl = np.full((pt.batch, hkv, mb), -1, np.int32)
    for i in range(pt.batch):
        sl[i, :, : P[i]] = np.arange(P[i])
    return sl, np.repeat(P[:, None], hkv, 1).astype(np.int32)


def test_equal_keys_give_mean_of_values_and_log_n():
    # all keys identical => uniform softmax: o = mean(V), lse = x + ln n   (closed form)
    rng = np.random.default_rng(0)
    hq, hkv, b, d, n = 4, 2, 4, 8, 13          # 13 tokens: last page has 1 valid token
    pool = make_pool(rng, 8, hkv, b, d)
    key = rng.standard_normal((hkv, d)).astype(np.float32)
    pool.k[:] = key[None, :, None, :]
    pt = table(rng, [n], b, 8)
    q = rng.standard_normal((1, hq, d)).astype(np.float32)
    scale = 0.37
    out, lse = vo.dense_attention(q, pool, pt, hq, hkv, d, d, scale)
    phys = pt.page_indices
    for h in range(hq):
        kvh = h // (hq // hkv)
        vals = np.concatenate([pool.v[p, kvh] for p in phys])[:n].astype(np.float64)
        x = scale * float(q[0, h].astype(np.float64) @ key[kvh].astype(np.float64))
        np.testing.assert_allclose(out[0, h], vals.mean(0), rtol=0, atol=1e-13)
        assert abs(lse[0, h] - (x + math.log(n))) < 1e-12


def test_stale_slots_of_partial_page_are_ignored():
    # tokens at positions >= n must not contribute even if they hold huge keys
    rng = np.random.default_rng(1)
    pool = make_pool(rng, 4, 1, 4, 8)
    pt = table(rng, [6], 4, 4)                  # page 1 has 2 valid + 2 stale slots
    q = rng.standard_normal((1, 2, 8)).astype(np.float32)
    out0, lse0 = vo.dense_attention(q, pool, pt, 2, 1, 8, 8, 0.5)
    last = pt.page_indices[1]
    pool.k[last, 0, 2:] = 1e30
    pool.v[last, 0, 2:] = -1e30
    out1, lse1 = vo.dense_attention(q, pool, pt, 2, 1, 8, 8, 0.5)
    assert np.array_equal(out0, out1) and np.array_equal(lse0, lse1)


def test_one_dominant_key_selects_its_value():
    rng = np.random.default_rng(2)
    d = 8
    pool = make_pool(rng, 6, 1, 4, d)
    pool.k *= 0.01
    pt = table(rng, [20], 4, 6)
    q = np.zeros((1, 1, d), np.float32)
    q[0, 0, 3] = 1.0
    p, t = pt.page_indices[2], 1                # token 9
    pool.k[p, 0, t, 3] = 50.0                   # logit +50 above the rest
    out, lse = vo.dense_attention(q, pool, pt, 1, 1, d, d, 1.0)
    np.testing.assert_allclose(out[0, 0], pool.v[p, 0, t].astype(np.float64), atol=1e-18 + 20 * math.exp(-49) * 5)
    assert abs(lse[0, 0] - 50.0) < 1e-15 + 20 * math.exp(-49)


def test_constant_logit_shift_leaves_output_and_shifts_lse():
    # append one channel: q_extra = 1, k_extra = const for every token => logits + scale*const
    rng = np.random.default_rng(3)
    d, b, n = 8, 4, 19
    base = make_pool(rng, 8, 1, b, d)
    pt = table(rng, [n], b, 8)
    q = rng.standard_normal((1, 2, d)).astype(np.float32)
    k2 = np.concatenate([base.k, np.full(base.k.shape[:-1] + (1,), 3.0, np.float32)], -1)
    q2 = np.concatenate([q, np.ones((1, 2, 1), np.float32)], -1)
    pool2 = vo.Pool(k=np.ascontiguousarray(k2), v=base.v, stride_page=b * (d + 1), stride_token=d + 1,
                    stride_head=b * (d + 1), num_pool_pages=8)
    # V keeps its own (d-wide) strides only if strides match; use v with d+1 layout too
    v2 = np.concatenate([base.v, np.zeros(base.v.shape[:-1] + (1,), np.float32)], -1)
    pool2.v = np.ascontiguousarray(v2)
    vpad = vo.Pool(k=base.k, v=base.v, stride_page=b * d, stride_token=d, stride_head=b * d, num_pool_pages=8)
    o1, l1 = vo.dense_attention(q, vpad, pt, 2, 1, d, d, 0.7)
    o2, l2 = vo.dense_attention(q2, pool2, pt, 2, 1, d + 1, d, 0.7)
    np.testing.assert_allclose(o2, o1, rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(l2, l1 + 0.7 * 3.0, rtol=0, atol=1e-12)


def test_two_token_closed_form_checks_operand_roles():
    # n = 2, d = 1, dv = 2: o = sigmoid weights of exp(s*q*k0), exp(s*q*k1) applied to V rows
    pool = vo.Pool(k=np.array([[[[2.0], [-1.0]]]], np.float32), v=np.array([[[[1.0, 10.0], [3.0, -4.0]]]], np.float32),
                   stride_page=2, stride_token=1, stride_head=2, num_pool_pages=1)
    # V strides differ from K's here, so give V the K strides by padding: use d=1,dv=1 twice instead
    pool.v = np.array([[[[5.0], [-7.0]]]], np.float32)
    pt = vo.PageTable([0, 1], [0], [2], 2)
    q = np.array([[[1.5]]], np.float32)
    out, lse = vo.dense_attention(q, pool, pt, 1, 1, 1, 1, 0.5)
    e0, e1 = math.exp(0.5 * 1.5 * 2.0), math.exp(0.5 * 1.5 * -1.0)
    assert abs(out[0, 0, 0] - (e0 * 5.0 + e1 * -7.0) / (e0 + e1)) < 1e-14
    assert abs(lse[0, 0] - math.log(e0 + e1)) < 1e-14


def test_gqa_head_to_kv_head_mapping():
    # q head h must read KV head h // g: make KV heads differ grossly and compare per-head single-head runs
    rng = np.random.default_rng(4)
    hq, hkv, b, d = 6, 3, 4, 8
    pool = make_pool(rng, 8, hkv, b, d)
    pt = table(rng, [14], b, 8)
    q = rng.standard_normal((1, hq, d)).astype(np.float32)
    out, lse = vo.dense_attention(q, pool, pt, hq, hkv, d, d, 0.3)
    for h in range(hq):
        kvh = h // 2
        single = vo.Pool(k=np.ascontiguousarray(pool.k[:, kvh:kvh + 1]), v=np.ascontiguousarray(pool.v[:, kvh:kvh + 1]),
                         stride_page=b * d, stride_token=d, stride_head=b * d, num_pool_pages=8)
        o1, l1 = vo.dense_attention(np.ascontiguousarray(q[:, h:h + 1]), single, pt, 1, 1, d, d, 0.3)
        assert np.array_equal(o1[0, 0], out[0, h]) and l1[0, 0] == lse[0, h]


@pytest.mark.parametrize("shared", [False, True])
def test_pool_permutation_invariance(shared):
    # relabelling physical pages (pool rows + page table together) changes nothing
    rng = np.random.default_rng(5)
    hq, hkv, b, d = 4, (1 if shared else 2), 4, 12
    dv = 8 if shared else d                      # one stride set serves K and V (header: vx_kv_pool)
    pool = make_pool(rng, 10, hkv, b, d, dv, shared=shared)
    pt = table(rng, [9, 17], b, 10)
    q = rng.standard_normal((2, hq, d)).astype(np.float32)
    o1, l1 = vo.dense_attention(q, pool, pt, hq, hkv, d, dv, 0.25)
    perm = rng.permutation(10)
    inv = np.argsort(perm)
    pool2 = vo.Pool(k=np.ascontiguousarray(pool.k[perm]), v=None if shared else np.ascontiguousarray(pool.v[perm]),
                    stride_page=pool.stride_page, stride_token=pool.stride_token,
                    stride_head=pool.stride_head, num_pool_pages=10)
    pt2 = vo.PageTable(pt.page_indptr, inv[pt.page_indices].astype(np.int32), pt.seq_lens, b)
    o2, l2 = vo.dense_attention(q, pool2, pt2, hq, hkv, d, dv, 0.25)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


def test_mla_value_is_first_channels_of_latent():
    # kv_shared: same result as an explicit V pool holding K[..., :dv]   (G8)
    rng = np.random.default_rng(6)
    b, d, dv = 4, 12, 8
    pool = make_pool(rng, 6, 1, b, d, shared=True)
    pt = table(rng, [21], b, 6)
    q = rng.standard_normal((1, 3, d)).astype(np.float32)
    o1, l1 = vo.dense_attention(q, pool, pt, 3, 1, d, dv, 0.2)
    vfull = np.ascontiguousarray(pool.k.copy())
    vfull[..., dv:] = 777.0                      # must never be read
    o2, l2 = vo.dense_attention(q, vo.Pool(pool.k, vfull, pool.stride_page, pool.stride_token, pool.stride_head, 6),
                                pt, 3, 1, d, dv, 0.2)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


def test_sparse_on_all_pages_equals_dense_bitwise():
    rng = np.random.default_rng(7)
    hq, hkv, b, d = 4, 2, 4, 8
    pool = make_pool(rng, 16, hkv, b, d)
    pt = table(rng, [13, 30], b, 16)
    q = rng.standard_normal((2, hq, d)).astype(np.float32)
    sl, sc = all_pages_sel(pt, hkv)
    o1, l1 = vo.sparse_attention(q, pool, pt, sl, sc, hq, hkv, d, d, 0.4)
    o2, l2 = vo.dense_attention(q, pool, pt, hq, hkv, d, d, 0.4)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


@pytest.mark.parametrize("S", [2, 3, 5])
def test_split_and_lse_combine_equals_unsplit(S):
    rng = np.random.default_rng(8 + S)
    hq, hkv, b, d = 4, 2, 4, 8
    pool = make_pool(rng, 16, hkv, b, d)
    pt = table(rng, [45], b, 16)
    q = (3 * rng.standard_normal((1, hq, d))).astype(np.float32)
    sel = np.sort(rng.permutation(12)[:9]).astype(np.int32)
    sl = np.tile(sel, (1, hkv, 1))
    o_ref, l_ref = vo.sparse_attention(q, pool, pt, sl, np.full((1, hkv), 9, np.int32), hq, hkv, d, d, 0.5)
    cuts = np.sort(rng.permutation(np.arange(1, 9))[: S - 1])
    parts = np.split(sel, cuts) + [np.zeros(0, np.int32)]      # plus one EMPTY part (lse = -inf)
    o_parts, l_parts = [], []
    for part in parts:
        slp = np.full((1, hkv, 9), -1, np.int32)
        slp[:, :, : len(part)] = part
        o, l = vo.sparse_attention(q, pool, pt, slp, np.full((1, hkv), len(part), np.int32), hq, hkv, d, d, 0.5)
        o_parts.append(o[0]); l_parts.append(l[0])
    o_c, l_c = vo.combine(np.stack(o_parts, 1), np.stack(l_parts, 1))
    np.testing.assert_allclose(o_c, o_ref[0], rtol=0, atol=1e-12)
    np.testing.assert_allclose(l_c, l_ref[0], rtol=0, atol=1e-12)


def test_bf16_inputs_are_widened_exactly():
    # bf16 bit patterns and the same values in fp32 give identical results
    rng = np.random.default_rng(9)
    b, d = 4, 8
    kf = rng.standard_normal((6, 1, b, d)).astype(np.float32)
    vf = rng.standard_normal((6, 1, b, d)).astype(np.float32)
    qf = rng.standard_normal((1, 2, d)).astype(np.float32)
    trunc = lambda a: (a.view(np.uint32) & 0xFFFF0000).view(np.float32)
    bits = lambda a: (a.view(np.uint32) >> 16).astype(np.uint16)
    kf, vf, qf = trunc(kf), trunc(vf), trunc(qf)
    pt = table(rng, [22], b, 6)
    mk = lambda k, v: vo.Pool(k, v, b * d, d, b * d, 6)
    o1, l1 = vo.dense_attention(qf, mk(kf, vf), pt, 2, 1, d, d, 0.3)
    o2, l2 = vo.dense_attention(bits(qf), mk(bits(kf), bits(vf)), pt, 2, 1, d, d, 0.3)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)
