"""Pins of the fp8 KV-cache oracle (-m "not gpu"): oracle/vx_oracle_fp8.py and the VXO_F64 element path of vx_oracle.c.

What fixes the decode (reading G25): the hand-written landmark codes of tests/golden/fp8_landmarks.txt (from the format
definitions), the structure of the formats (sign symmetry, monotone in the code, spacing = 2^(e - bias - mbits), counts
of finite / NaN / inf patterns), and torch's own float8 dtypes on all 256 codes (a library routine, not our code).
What fixes the use (G26, G27): scale * decode is exact; an fp8 pool run through the oracle equals the SAME values stored
as fp32 run through the untouched fp32 path bit for bit; a power-of-two scale commutes with everything; the selection
does not depend on k_scale; bf16-representable pools stored as fp8 losslessly reproduce the bf16 oracle's outputs."""
import os
from dataclasses import replace

import numpy as np
import pytest
import torch

from oracle import vx_oracle as vo
from oracle.vx_oracle_fp8 import FORMATS, dequantize, pool_fp8, widen_fp8
from oracle.workload_io import oracle_step, to_oracle
from paper_2606_06453_b200.workloads import SPECS, make_workload, with_fp8

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "fp8_landmarks.txt")
ALL = np.arange(256, dtype=np.uint8)


def test_landmark_codes():
    n = 0
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        fmt, code, val = line.split()
        got = float(widen_fp8(np.array([int(code, 16)], dtype=np.uint8), fmt)[0])
        want = float(val)
        if np.isnan(want):
            assert np.isnan(got), line
        else:
            assert got == want and np.signbit(got) == np.signbit(want), line
        n += 1
    assert n == 32


@pytest.mark.parametrize("fmt", FORMATS)
def test_structure_of_the_format(fmt):
    v = widen_fp8(ALL, fmt)
    pos, neg = v[:128], v[128:]
    assert np.array_equal(np.isnan(pos), np.isnan(neg))
    ok = ~np.isnan(pos)
    assert np.array_equal(neg[ok], -pos[ok]), "sign bit only flips the sign"
    fin = pos[np.isfinite(pos)]
    assert (np.diff(fin) > 0).all(), "positive codes are ordered like their values"
    mbits, bias = (3, 7) if fmt == "e4m3" else (2, 15)
    assert int(np.isnan(pos).sum()) == (1 if fmt == "e4m3" else 3) and int(np.isinf(pos).sum()) == (0 if fmt == "e4m3" else 1)
    step = np.diff(fin)                                   # spacing inside binade e is 2^(e - bias - mbits), subnormals as e = 1
    for c in range(len(fin) - 1):
        e = max(c >> mbits, 1)
        assert step[c] == 2.0 ** (e - bias - mbits), (fmt, c)
    assert fin[-1] == (448.0 if fmt == "e4m3" else 57344.0)


@pytest.mark.parametrize("fmt,tdt", [("e4m3", torch.float8_e4m3fn), ("e5m2", torch.float8_e5m2)])
def test_against_the_library_dtype_on_all_codes(fmt, tdt):
    ref = torch.from_numpy(ALL.copy()).view(tdt).to(torch.float64).numpy()
    got = widen_fp8(ALL, fmt)
    assert np.array_equal(np.isnan(got), np.isnan(ref))
    assert np.array_equal(got[~np.isnan(ref)], ref[~np.isnan(ref)])


def test_scale_is_applied_once_and_exactly():
    codes = ALL[np.isfinite(widen_fp8(ALL, "e4m3"))]
    s = np.float32(0.0892857164144516)
    got = dequantize(codes, "e4m3", s)
    assert np.array_equal(got, widen_fp8(codes, "e4m3") * float(s))
    assert (np.abs(got) <= 448.0 * float(s)).all() and got[np.argmax(np.abs(got))] in (448.0 * float(s), -448.0 * float(s))
    assert dequantize(np.array([0x38], np.uint8), "e4m3", 3.0)[0] == 3.0      # code of 1.0


def _fp32_twin(w):
    """the same workload with the values its fp8 codes stand for stored as fp32 (exact when the scale is a power of two)"""
    k = torch.from_numpy(dequantize(vo.as_np(w.k_pool), w.spec.kv_dtype, w.k_scale).astype(np.float32))
    v = None if w.v_pool is None else torch.from_numpy(dequantize(vo.as_np(w.v_pool), w.spec.kv_dtype, w.v_scale).astype(np.float32))
    return replace(w, spec=replace(w.spec, kv_dtype="", dtype="f32"), k_pool=k, v_pool=v, q=w.q.float(), k_scale=1.0, v_scale=1.0)


@pytest.mark.parametrize("name,fmt", [("C2-small", "e4m3"), ("C4-small", "e5m2")])
def test_fp8_pool_equals_the_same_values_through_the_fp32_path(name, fmt):
    w = make_workload(replace(with_fp8(name, fmt), batch=2))
    w = replace(w, k_scale=0.125, v_scale=0.03125)        # powers of two: scale * decode(code) is exact in fp32 too
    if w.v_pool is None:
        w = replace(w, v_scale=w.k_scale)
    a = oracle_step(w)                                    # VXO_F64 element path
    tw = _fp32_twin(w)
    tw = replace(tw, q=w.q)                               # (the same bf16 queries)
    b = oracle_step(tw)                                   # the untouched fp32 element path
    for key in ("scores", "sel_logical", "sel_count", "out", "lse", "summary"):
        assert np.array_equal(a[key], b[key], equal_nan=True), key


def test_selection_does_not_depend_on_k_scale_and_scores_scale_linearly():
    w = make_workload(replace(with_fp8("C5-small"), batch=3))
    a = oracle_step(replace(w, k_scale=1.0))
    b = oracle_step(replace(w, k_scale=0.25))             # G27: a positive common factor changes no selection
    assert np.array_equal(a["sel_logical"], b["sel_logical"])
    assert np.array_equal(a["scores"] * 0.25, b["scores"])
    c = oracle_step(replace(w, v_scale=2.0 * w.v_scale))  # v_scale is linear in the output, absent from lse
    d = oracle_step(w)
    np.testing.assert_allclose(c["out"], 2.0 * d["out"], rtol=1e-13)
    assert np.array_equal(c["lse"], d["lse"])


def test_lossless_fp8_storage_reproduces_the_bf16_oracle():
    """keys / values drawn ON the e4m3 grid: bf16 storage and fp8 storage hold the same numbers -> identical results"""
    spec = replace(SPECS["C2-small"], batch=2, outlier_channels=0)
    w = make_workload(spec)
    grid = lambda t: t.float().to(torch.float8_e4m3fn).float().to(torch.bfloat16)       # exact in bf16
    wb = replace(w, k_pool=grid(w.k_pool), v_pool=grid(w.v_pool))
    w8 = replace(wb, spec=with_fp8(spec), k_pool=wb.k_pool.float().to(torch.float8_e4m3fn).view(torch.uint8),
                 v_pool=wb.v_pool.float().to(torch.float8_e4m3fn).view(torch.uint8), k_scale=1.0, v_scale=1.0)
    a, b = oracle_step(wb), oracle_step(w8)
    for key in ("scores", "sel_logical", "out", "lse"):
        assert np.array_equal(a[key], b[key]), key
