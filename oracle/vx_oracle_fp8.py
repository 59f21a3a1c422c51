"""fp8 KV cache for the oracle (test infrastructure only, like everything under oracle/).

PAPER.md:200 (section 5.3: the decode backends' "precision support, such as fp8 KV cache", is inherited), :520 / :525
(Listing 2: kv_cache_dtype "fp8_e4m3"; "supports bfloat16, fp8_e4m3 and fp8_e5m2").  The paper gives neither the bit
layouts nor a scale convention; DESIGN.md readings:
  G25  fp8_e4m3 is the OCP 8-bit "E4M3" finite-only format (1 sign, 4 exponent bits of bias 7, 3 mantissa bits; no
       infinities, S.1111.111 is NaN, largest value 448); fp8_e5m2 is the OCP "E5M2" format (5 exponent bits of bias 15,
       2 mantissa bits, IEEE-like: exponent 31 holds the infinities and NaNs, largest finite value 57,344).
  G26  a stored code c stands for the value  scale * decode(c)  with one fp32 scale per pool tensor (k_scale for K,
       v_scale for V; the MLA latent pool has one scale, used for both roles): the per-layer convention of the serving
       systems the paper plugs into.  q, out and lse keep the query dtype.
  G27  page summaries of an fp8 pool are fp8 codes too (the min / max of representable values is representable), and
       page scores are computed on the decoded codes WITHOUT k_scale: a positive factor common to every page of the
       layer changes no selection.  Attention uses the scaled values.

This file is the plain definition: decode(c) written out from the two bit layouts, in float64 (every fp8 value and its
product with an fp32 scale is exact in double).  No code shared with csrc/.
"""
import numpy as np

from oracle import vx_oracle as vo

FORMATS = ("e4m3", "e5m2")


def widen_fp8(codes, fmt: str) -> np.ndarray:
    """uint8 codes -> float64 values, from the format definition (G25)."""
    c = np.asarray(codes, dtype=np.uint8).astype(np.int64)
    sign = np.where(c >> 7, -1.0, 1.0)
    if fmt == "e4m3":
        e, m, mbits, bias = (c >> 3) & 15, c & 7, 3, 7
        nan = (e == 15) & (m == 7)                         # the only NaN pattern; there are no infinities
        inf = np.zeros_like(nan)
    elif fmt == "e5m2":
        e, m, mbits, bias = (c >> 2) & 31, c & 3, 2, 15
        nan = (e == 31) & (m != 0)
        inf = (e == 31) & (m == 0)
    else:
        raise ValueError(fmt)
    frac = m.astype(np.float64) / (1 << mbits)
    normal = (1.0 + frac) * np.exp2((e - bias).astype(np.float64))
    subnormal = frac * np.exp2(float(1 - bias))
    v = np.where(e == 0, subnormal, normal)
    v = np.where(inf, np.inf, v)
    v = np.where(nan, np.nan, v)
    return sign * v


def dequantize(codes, fmt: str, scale=1.0) -> np.ndarray:
    """the values an fp8 pool stands for: float64(scale as fp32) * decode(code)   (G26); exact in double"""
    return widen_fp8(codes, fmt) * float(np.float32(scale))


def pool_fp8(k_codes, v_codes, fmt, k_scale, v_scale, stride_page, stride_token, stride_head, num_pool_pages) -> vo.Pool:
    """an oracle Pool of doubles for fp8 code tensors (v_codes None: kv_shared, V = K[..., :v_dim] with k_scale)"""
    k = np.ascontiguousarray(dequantize(k_codes, fmt, k_scale))
    v = None if v_codes is None else np.ascontiguousarray(dequantize(v_codes, fmt, v_scale))
    return vo.Pool(k=k, v=v, stride_page=stride_page, stride_token=stride_token, stride_head=stride_head,
                   num_pool_pages=num_pool_pages)
