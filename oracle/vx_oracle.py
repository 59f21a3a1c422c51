"""ctypes loader for oracle/vx_oracle.c -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It does not import paper_2606_06453_b200 and shares
no code with the CUDA path.  All arithmetic lives in vx_oracle.c (plain fp64 C,
written from PAPER.md); this file only marshals numpy arrays.

Arrays: bf16 data is passed as numpy uint16 (raw bits), fp32 as float32.  Use
``as_np`` to turn a CPU torch tensor into the right view.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vx_oracle.c")
_LIB = os.path.join(_HERE, "libvx_oracle.so")

BF16, F32, F64 = 0, 1, 2   # F64: values that are already doubles (fp8 pools widened by vx_oracle_fp8.py)
AGG_SUM, AGG_MAX = 0, 1


def build(force: bool = False) -> str:
    """Compile vx_oracle.c with gcc (-O2 -fopenmp); returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.vxo_num_threads.restype = C.c_int
        _lib.vxo_topk_pages.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().vxo_num_threads())


def as_np(t):
    """CPU torch tensor (bf16 / fp32 / int32) or ndarray -> contiguous ndarray (bf16 -> uint16 bits)."""
    if isinstance(t, np.ndarray):
        return np.ascontiguousarray(t)
    import torch  # only for the dtype switch; no torch arithmetic is used

    t = t.detach().cpu().contiguous()
    if t.dtype == torch.bfloat16:
        return t.view(torch.int16).numpy().view(np.uint16)
    return t.numpy()


def _dt(a: np.ndarray) -> int:
    if a.dtype == np.uint16:
        return BF16
    if a.dtype == np.float32:
        return F32
    if a.dtype == np.float64:
        return F64
    raise TypeError(f"oracle takes bf16 bits (uint16), float32 or float64, got {a.dtype}")


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _i32(a):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.int32))
    return a


@dataclass
class PageTable:
    """The paper's C = (b, p, I)."""

    page_indptr: np.ndarray   # [batch+1] int32
    page_indices: np.ndarray  # [total_pages] int32 physical ids in logical order
    seq_lens: np.ndarray      # [batch] int32 tokens, including the one just appended
    page_size: int

    def __post_init__(self):
        self.page_indptr = _i32(self.page_indptr)
        self.page_indices = _i32(self.page_indices)
        self.seq_lens = _i32(self.seq_lens)

    @property
    def batch(self) -> int:
        return len(self.seq_lens)

    @property
    def total_pages(self) -> int:
        return int(self.page_indptr[-1])


@dataclass
class Pool:
    """K (and V) pool with element strides; kv_shared pools pass v=None (V = K[..., :v_dim])."""

    k: np.ndarray
    v: np.ndarray | None
    stride_page: int
    stride_token: int
    stride_head: int
    num_pool_pages: int


def page_summary(pool: Pool, pt: PageTable, num_kv_heads: int, qk_dim: int, first_page=None,
                 summary: np.ndarray | None = None) -> np.ndarray:
    """float64 [num_pool_pages, Hkv, 2, d]; [...,0,:]=min, [...,1,:]=max.  Untouched pages stay NaN."""
    if summary is None:
        summary = np.full((pool.num_pool_pages, num_kv_heads, 2, qk_dim), np.nan, dtype=np.float64)
    fp = _i32(first_page) if first_page is not None else None
    lib().vxo_page_summary(_p(pool.k), _dt(pool.k), C.c_int64(pool.stride_page),
                           C.c_int64(pool.stride_token), C.c_int64(pool.stride_head),
                           num_kv_heads, qk_dim, pt.page_size, pt.batch, _p(pt.page_indptr),
                           _p(pt.page_indices), _p(pt.seq_lens), _p(fp), _p(summary))
    return summary


def page_score(q: np.ndarray, summary: np.ndarray, pt: PageTable, num_q_heads: int,
               num_kv_heads: int, agg: int = AGG_SUM):
    """returns (u [Hq, T] per-head envelope scores, S [Hkv, T] group-aggregated), float64."""
    d = summary.shape[-1]
    T = pt.total_pages
    u = np.zeros((num_q_heads, T), dtype=np.float64)
    s = np.zeros((num_kv_heads, T), dtype=np.float64)
    summary = np.ascontiguousarray(summary, dtype=np.float64)
    lib().vxo_page_score(_p(q), _dt(q), _p(summary), num_q_heads, num_kv_heads, d, pt.batch,
                         _p(pt.page_indptr), _p(pt.page_indices), _p(pt.seq_lens), pt.page_size,
                         agg, _p(u), _p(s))
    return u, s


def page_centroid(pool: Pool, pt: PageTable, num_kv_heads: int, qk_dim: int, first_page=None,
                  centroid: np.ndarray | None = None) -> np.ndarray:
    """Block top-k summaries (Eq.1): float64 [num_pool_pages, Hkv, d], the mean over the valid
    tokens rounded to the KV dtype (bf16 / fp32).  Untouched pages stay NaN."""
    if centroid is None:
        centroid = np.full((pool.num_pool_pages, num_kv_heads, qk_dim), np.nan, dtype=np.float64)
    fp = _i32(first_page) if first_page is not None else None
    lib().vxo_page_centroid(_p(pool.k), _dt(pool.k), C.c_int64(pool.stride_page),
                            C.c_int64(pool.stride_token), C.c_int64(pool.stride_head),
                            num_kv_heads, qk_dim, pt.page_size, pt.batch, _p(pt.page_indptr),
                            _p(pt.page_indices), _p(pt.seq_lens), _p(fp), _p(centroid))
    return centroid


def centroid_score(q: np.ndarray, centroid: np.ndarray, pt: PageTable, num_q_heads: int,
                   num_kv_heads: int):
    """returns (u [Hq, T] per-head q_h . centroid, S [Hkv, T] group sums; Eq.2), float64."""
    d = centroid.shape[-1]
    T = pt.total_pages
    u = np.zeros((num_q_heads, T), dtype=np.float64)
    s = np.zeros((num_kv_heads, T), dtype=np.float64)
    centroid = np.ascontiguousarray(centroid, dtype=np.float64)
    lib().vxo_centroid_score(_p(q), _dt(q), _p(centroid), num_q_heads, num_kv_heads, d, pt.batch,
                             _p(pt.page_indptr), _p(pt.page_indices), _p(pt.seq_lens), pt.page_size,
                             _p(u), _p(s))
    return u, s


def topk_pages(scores: np.ndarray, pt: PageTable, budget, n_sink: int, n_local: int,
               max_budget: int):
    """returns (sel_logical, sel_phys [B,Hkv,max_budget] pad -1, sel_count [B,Hkv], thr [B,Hkv])."""
    scores = np.ascontiguousarray(scores, dtype=np.float64)
    hkv = scores.shape[0]
    budget = _i32(budget)
    sl = np.full((pt.batch, hkv, max_budget), -1, dtype=np.int32)
    sp = np.full((pt.batch, hkv, max_budget), -1, dtype=np.int32)
    sc = np.zeros((pt.batch, hkv), dtype=np.int32)
    thr = np.full((pt.batch, hkv), np.nan, dtype=np.float64)
    bad = lib().vxo_topk_pages(_p(scores), hkv, pt.batch, _p(pt.page_indptr), _p(pt.page_indices),
                               _p(pt.seq_lens), pt.page_size, _p(budget), n_sink, n_local,
                               max_budget, _p(sl), _p(sp), _p(sc), _p(thr))
    if bad:
        raise ValueError("precondition n_sink + n_local <= budget <= max_budget violated (G6)")
    return sl, sp, sc, thr


def _attn_common(q, pool: Pool, num_q_heads, num_kv_heads, qk_dim, v_dim):
    v = pool.v if pool.v is not None else pool.k
    assert _dt(v) == _dt(pool.k)
    return v


def sparse_attention(q: np.ndarray, pool: Pool, pt: PageTable, sel_logical, sel_count,
                     num_q_heads: int, num_kv_heads: int, qk_dim: int, v_dim: int, sm_scale: float):
    """softmax attention over the selected pages; returns (out [B,Hq,dv], lse [B,Hq]) float64."""
    v = _attn_common(q, pool, num_q_heads, num_kv_heads, qk_dim, v_dim)
    sel_logical = _i32(sel_logical)
    sel_count = _i32(sel_count)
    max_budget = sel_logical.shape[-1]
    out = np.zeros((pt.batch, num_q_heads, v_dim), dtype=np.float64)
    lse = np.zeros((pt.batch, num_q_heads), dtype=np.float64)
    lib().vxo_sparse_attention(_p(q), _dt(q), _p(pool.k), _p(v), _dt(pool.k),
                               C.c_int64(pool.stride_page), C.c_int64(pool.stride_token),
                               C.c_int64(pool.stride_head), num_q_heads, num_kv_heads, qk_dim,
                               v_dim, pt.page_size, pt.batch, _p(pt.page_indptr),
                               _p(pt.page_indices), _p(pt.seq_lens), _p(sel_logical),
                               _p(sel_count), max_budget, C.c_double(sm_scale), _p(out), _p(lse))
    return out, lse


def dense_attention(q: np.ndarray, pool: Pool, pt: PageTable, num_q_heads: int, num_kv_heads: int,
                    qk_dim: int, v_dim: int, sm_scale: float):
    v = _attn_common(q, pool, num_q_heads, num_kv_heads, qk_dim, v_dim)
    out = np.zeros((pt.batch, num_q_heads, v_dim), dtype=np.float64)
    lse = np.zeros((pt.batch, num_q_heads), dtype=np.float64)
    lib().vxo_dense_attention(_p(q), _dt(q), _p(pool.k), _p(v), _dt(pool.k),
                              C.c_int64(pool.stride_page), C.c_int64(pool.stride_token),
                              C.c_int64(pool.stride_head), num_q_heads, num_kv_heads, qk_dim,
                              v_dim, pt.page_size, pt.batch, _p(pt.page_indptr),
                              _p(pt.page_indices), _p(pt.seq_lens), C.c_double(sm_scale),
                              _p(out), _p(lse))
    return out, lse


def combine(o_part: np.ndarray, lse_part: np.ndarray):
    """o_part [rows, S, dv], lse_part [rows, S] -> (out [rows, dv], lse [rows])."""
    o_part = np.ascontiguousarray(o_part, dtype=np.float64)
    lse_part = np.ascontiguousarray(lse_part, dtype=np.float64)
    rows, S, dv = o_part.shape
    out = np.zeros((rows, dv), dtype=np.float64)
    lse = np.zeros((rows,), dtype=np.float64)
    lib().vxo_combine(_p(o_part), _p(lse_part), C.c_int64(rows), S, dv, _p(out), _p(lse))
    return out, lse


def decode_step(q, pool: Pool, pt: PageTable, budget, max_budget: int, num_q_heads: int,
                num_kv_heads: int, qk_dim: int, v_dim: int, sm_scale: float, n_sink: int,
                n_local: int, agg: int = AGG_SUM, summary: np.ndarray | None = None,
                kind: str = "envelope"):
    """the whole step in the paper's order: summary -> score -> top-k -> attention.
    kind = "envelope" (Quest) or "centroid" (block top-k, Eq.1-2)."""
    if kind == "centroid":
        if summary is None:
            summary = page_centroid(pool, pt, num_kv_heads, qk_dim)
        u, s = centroid_score(q, summary, pt, num_q_heads, num_kv_heads)
    else:
        if summary is None:
            summary = page_summary(pool, pt, num_kv_heads, qk_dim)
        u, s = page_score(q, summary, pt, num_q_heads, num_kv_heads, agg)
    sl, sp, sc, thr = topk_pages(s, pt, budget, n_sink, n_local, max_budget)
    out, lse = sparse_attention(q, pool, pt, sl, sc, num_q_heads, num_kv_heads, qk_dim, v_dim, sm_scale)
    return dict(summary=summary, u=u, scores=s, sel_logical=sl, sel_phys=sp, sel_count=sc,
                thr=thr, out=out, lse=lse)
