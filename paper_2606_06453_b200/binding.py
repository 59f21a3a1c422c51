"""Thin ctypes binding over libvortex_b200.so (include/vortex_b200.h).

Argument marshalling only: every step of the path runs in the CUDA kernels behind the C
ABI.  torch is used for device memory and streams.  There is no CPU fallback -- if the
library is missing or the device is not a B200, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libvortex_b200.so")

VX_OK, VX_ERR_INVALID_ARG, VX_ERR_UNSUPPORTED, VX_ERR_WORKSPACE, VX_ERR_CUDA = range(5)
VX_DT_BF16, VX_DT_F32 = 0, 1
VX_AGG_SUM, VX_AGG_MAX = 0, 1
VX_SUMMARY_ENVELOPE, VX_SUMMARY_CENTROID = 0, 1
VX_STEP_UPDATE_SUMMARY = 1
VX_STEP_APPROX_TOPK = 2
VX_TRACE_SCORE, VX_TRACE_TOPK, VX_TRACE_DECODE = 1, 2, 4
VX_KV_SAME, VX_KV_FP8_E4M3, VX_KV_FP8_E5M2 = 0, 1, 2
VX_OPT_MLA_STEP, VX_OPT_MLA_FLAT_SPLITS, VX_OPT_MLA_FLAT_WAVES = 1, 2, 3
VX_MLA_STEP_AUTO, VX_MLA_STEP_FUSED, VX_MLA_STEP_CHAINED, VX_MLA_STEP_FLAT = 0, 1, 2, 3

EXPORTS = ["vx_workspace_bytes", "vx_create", "vx_destroy", "vx_last_error", "vx_last_launch_count",
           "vx_page_summary_update", "vx_page_score", "vx_topk_pages", "vx_sparse_paged_decode",
           "vx_sparse_decode_step", "vx_sparse_decode_step_host", "vx_trace_attach",
           "vx_topk_pages_approx", "vx_set_topk_approx", "vx_set_topk_remap", "vx_union_pages", "vx_set_option",
           "vx_sparse_paged_decode_static", "vx_static_scratch_bytes", "vx_static_last_error"]


class VxGeom(C.Structure):
    _fields_ = [("dtype", C.c_int32), ("num_q_heads", C.c_int32), ("num_kv_heads", C.c_int32),
                ("qk_dim", C.c_int32), ("v_dim", C.c_int32), ("page_size", C.c_int32),
                ("kv_shared", C.c_int32), ("sm_scale", C.c_float), ("n_sink", C.c_int32),
                ("n_local", C.c_int32), ("agg", C.c_int32), ("summary_kind", C.c_int32), ("kv_format", C.c_int32), ("block_size", C.c_int32)]


class VxPageTable(C.Structure):
    _fields_ = [("batch", C.c_int32), ("page_indptr", C.c_void_p), ("page_indices", C.c_void_p),
                ("seq_lens", C.c_void_p), ("total_pages", C.c_int32), ("max_pages_per_req", C.c_int32)]


class VxKvPool(C.Structure):
    _fields_ = [("k", C.c_void_p), ("v", C.c_void_p), ("stride_page", C.c_int64),
                ("stride_token", C.c_int64), ("stride_head", C.c_int64), ("num_pool_pages", C.c_int32),
                ("k_scale", C.c_float), ("v_scale", C.c_float)]


class VortexError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"vortex_b200 status {status}: {msg}")
        self.status = status


_lib = None


def load_library():
    """dlopen the in-tree library (build it with `python -m paper_2606_06453_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    # VX_B200_LIBRARY: another build of the same library (trace.py points it at libvortex_b200_trace.so)
    path = os.environ.get("VX_B200_LIBRARY") or LIB_PATH
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -m paper_2606_06453_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(path)
    P, I32, U32, SZ = C.c_void_p, C.c_int32, C.c_uint32, C.c_size_t
    G, T, K = C.POINTER(VxGeom), C.POINTER(VxPageTable), C.POINTER(VxKvPool)
    sig = {
        "vx_workspace_bytes": (SZ, [G, I32, I32, I32, I32]),
        "vx_create": (I32, [C.POINTER(P), G, C.c_int, P, SZ, I32, I32, I32, I32]),
        "vx_destroy": (None, [P]),
        "vx_last_error": (C.c_char_p, [P]),
        "vx_last_launch_count": (I32, [P]),
        "vx_trace_attach": (I32, [P, P, I32, I32]),
        "vx_page_summary_update": (I32, [P, K, T, P, P, P]),
        "vx_page_score": (I32, [P, P, P, T, P, P]),
        "vx_topk_pages": (I32, [P, P, T, P, I32, P, P, P, P]),
        "vx_topk_pages_approx": (I32, [P, P, T, P, I32, C.c_float, C.c_uint64, P, P, P, P]),
        "vx_set_topk_approx": (I32, [P, C.c_float, C.c_uint64]),
        "vx_set_topk_remap": (I32, [P, P, I32]),
        "vx_set_option": (I32, [P, I32, I32]),
        "vx_sparse_paged_decode_static": (I32, [G, P, K, T, P, P, P, I32, P, P, P]),
        "vx_static_scratch_bytes": (C.c_size_t, []),
        "vx_static_last_error": (C.c_char_p, []),
        "vx_union_pages": (I32, [P, T, P, P, I32, I32, P, P, P, P]),
        "vx_sparse_paged_decode": (I32, [P, P, K, T, P, P, P, I32, P, P, P]),
        "vx_sparse_decode_step": (I32, [P, P, K, P, T, P, I32, U32, P, P, P, P, P, P]),
        "vx_sparse_decode_step_host": (I32, [P, P, K, P, I32, P, P, P, P, I32, U32, P, P, P]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


class PageTable:
    """Device page table C = (b, p, I) plus the host scalars that size grids."""

    def __init__(self, page_indptr, page_indices, seq_lens, total_pages: int, max_pages_per_req: int):
        for t in (page_indptr, page_indices, seq_lens):
            assert t.dtype == torch.int32 and t.is_contiguous()
        self.tensors = (page_indptr, page_indices, seq_lens)
        self.c = VxPageTable(seq_lens.numel(), page_indptr.data_ptr(), page_indices.data_ptr(),
                             seq_lens.data_ptr(), int(total_pages), int(max_pages_per_req))

    @property
    def batch(self):
        return self.c.batch


class KvPool:
    """K/V pools [N_pool, Hkv, page, d] (or any layout expressed by element strides)."""

    def __init__(self, k, v, stride_page: int, stride_token: int, stride_head: int, k_scale: float = 1.0,
                 v_scale: float = 1.0):
        self.tensors = (k, v)
        self.c = VxKvPool(k.data_ptr(), 0 if v is None else v.data_ptr(), stride_page, stride_token,
                          stride_head, k.shape[0], float(k_scale), float(v_scale))


class Context:
    """One geometry on one device; owns its workspace tensor."""

    def __init__(self, *, dtype, num_q_heads, num_kv_heads, qk_dim, v_dim, page_size, sm_scale,
                 n_sink, n_local, kv_shared=False, agg=VX_AGG_SUM, summary_kind=VX_SUMMARY_ENVELOPE, kv_format=0, block_size=0, max_batch,
                 max_total_pages,
                 max_pages_per_req, max_budget, device="cuda:0"):
        self.lib = load_library()
        self.torch_dtype = dtype
        dt = {torch.bfloat16: VX_DT_BF16, torch.float32: VX_DT_F32}[dtype]
        self.geom = VxGeom(dt, num_q_heads, num_kv_heads, qk_dim, v_dim, page_size, int(kv_shared),
                           float(sm_scale), n_sink, n_local, agg, summary_kind, int(kv_format), int(block_size))
        self.device = torch.device(device)
        self.max = (int(max_batch), int(max_total_pages), int(max_pages_per_req), int(max_budget))
        need = self.lib.vx_workspace_bytes(C.byref(self.geom), *self.max)
        if need == 0:
            raise VortexError(VX_ERR_UNSUPPORTED, "geometry rejected by vx_workspace_bytes")
        if self.device.type != "cuda":
            raise VortexError(VX_ERR_CUDA, "vortex_b200 needs a CUDA device; there is no CPU path")
        self.workspace = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self._h = C.c_void_p()
        st = self.lib.vx_create(C.byref(self._h), C.byref(self.geom), self.device.index or 0,
                                C.c_void_p(base), need, *self.max)
        if st != VX_OK:
            raise VortexError(st, self.lib.vx_last_error(None).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self.lib.vx_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def _check(self, st):
        if st != VX_OK:
            raise VortexError(st, self.lib.vx_last_error(self._h).decode())

    @property
    def last_launch_count(self) -> int:
        return int(self.lib.vx_last_launch_count(self._h))

    # ---- the calls of include/vortex_b200.h, same names ---------------------------------
    def page_summary_update(self, pool: KvPool, pt: PageTable, summary, first_new_pos=None, stream=None):
        self._check(self.lib.vx_page_summary_update(self._h, C.byref(pool.c), C.byref(pt.c),
                                                    _ptr(first_new_pos), _ptr(summary), _stream(stream)))

    def page_score(self, q, summary, pt: PageTable, scores, stream=None):
        self._check(self.lib.vx_page_score(self._h, _ptr(q), _ptr(summary), C.byref(pt.c), _ptr(scores),
                                           _stream(stream)))

    def trace_attach(self, buffer, kernels):
        """buffer: int64 CUDA tensor [max_ctas, 16], zeroed by the caller (None detaches); trace builds only."""
        n = 0 if buffer is None else buffer.shape[0]
        self._check(self.lib.vx_trace_attach(self._h, _ptr(buffer), n, kernels))

    def topk_pages(self, scores, pt: PageTable, budget, max_budget, sel_phys, sel_logical, sel_count,
                   stream=None):
        self._check(self.lib.vx_topk_pages(self._h, _ptr(scores), C.byref(pt.c), _ptr(budget), max_budget,
                                           _ptr(sel_phys), _ptr(sel_logical), _ptr(sel_count),
                                           _stream(stream)))

    def topk_pages_approx(self, scores, pt: PageTable, budget, max_budget, tolerate_ratio, seed, sel_phys,
                          sel_logical, sel_count, stream=None):
        self._check(self.lib.vx_topk_pages_approx(self._h, _ptr(scores), C.byref(pt.c), _ptr(budget), max_budget,
                                                  float(tolerate_ratio), int(seed), _ptr(sel_phys),
                                                  _ptr(sel_logical), _ptr(sel_count), _stream(stream)))

    def union_pages(self, pt: PageTable, sel_logical, sel_count, max_budget, max_union, union_phys, union_logical,
                    union_count, stream=None):
        self._check(self.lib.vx_union_pages(self._h, C.byref(pt.c), _ptr(sel_logical), _ptr(sel_count), max_budget,
                                            max_union, _ptr(union_phys), _ptr(union_logical), _ptr(union_count),
                                            _stream(stream)))

    def set_option(self, option, value):
        self._check(self.lib.vx_set_option(self._h, int(option), int(value)))

    def set_topk_approx(self, tolerate_ratio, seed):
        self._check(self.lib.vx_set_topk_approx(self._h, float(tolerate_ratio), int(seed)))

    def set_topk_remap(self, knots):
        """knots: sequence of 2..65 floats in [0, 1], non-decreasing (remap_profile.profile_knots), or None to clear"""
        if knots is None or len(knots) == 0:
            self._check(self.lib.vx_set_topk_remap(self._h, None, 0))
            return
        arr = (C.c_float * len(knots))(*[float(v) for v in knots])
        self._check(self.lib.vx_set_topk_remap(self._h, C.cast(arr, C.c_void_p), len(knots)))

    def sparse_paged_decode(self, q, pool: KvPool, pt: PageTable, sel_phys, sel_logical, sel_count,
                            max_budget, out, lse=None, stream=None):
        self._check(self.lib.vx_sparse_paged_decode(self._h, _ptr(q), C.byref(pool.c), C.byref(pt.c),
                                                    _ptr(sel_phys), _ptr(sel_logical), _ptr(sel_count),
                                                    max_budget, _ptr(out), _ptr(lse), _stream(stream)))

    def sparse_decode_step(self, q, pool: KvPool, summary, pt: PageTable, budget, max_budget, out,
                           lse=None, sel_phys=None, sel_logical=None, sel_count=None, flags=0,
                           stream=None):
        self._check(self.lib.vx_sparse_decode_step(self._h, _ptr(q), C.byref(pool.c), _ptr(summary),
                                                   C.byref(pt.c), _ptr(budget), max_budget, flags,
                                                   _ptr(out), _ptr(lse), _ptr(sel_phys),
                                                   _ptr(sel_logical), _ptr(sel_count), _stream(stream)))

    def sparse_decode_step_host(self, h_q, pool: KvPool, summary, h_page_indptr, h_page_indices,
                                h_seq_lens, h_budget, max_budget, h_out, h_lse=None, flags=0,
                                stream=None):
        """Host (CPU, ideally pinned) tensors in, host tensors out; synchronous."""
        for t in (h_q, h_page_indptr, h_page_indices, h_seq_lens, h_budget, h_out):
            assert t.device.type == "cpu" and t.is_contiguous()
        self._check(self.lib.vx_sparse_decode_step_host(
            self._h, _ptr(h_q), C.byref(pool.c), _ptr(summary), h_seq_lens.numel(), _ptr(h_page_indptr),
            _ptr(h_page_indices), _ptr(h_seq_lens), _ptr(h_budget), max_budget, flags, _ptr(h_out),
            _ptr(h_lse), _stream(stream)))


def sparse_paged_decode_static(geom: VxGeom, q, pool: KvPool, pt: PageTable, sel_phys, sel_logical, sel_count, max_budget,
                               out, lse=None, stream=None):
    """vx_sparse_paged_decode_static: no context, no workspace, no allocation (scratch in a static device array)."""
    lib = load_library()
    st = lib.vx_sparse_paged_decode_static(C.byref(geom), _ptr(q), C.byref(pool.c), C.byref(pt.c), _ptr(sel_phys),
                                           _ptr(sel_logical), _ptr(sel_count), max_budget, _ptr(out), _ptr(lse),
                                           _stream(stream))
    if st != VX_OK:
        raise VortexError(st, lib.vx_static_last_error().decode())


# ---- conveniences used by tests / bench (allocation + marshalling only) -----------------------
def context_for(w, device=None, **over) -> Context:
    """Context sized for a workloads.Workload."""
    s = w.spec
    kw = dict(dtype={"bf16": torch.bfloat16, "f32": torch.float32}[s.dtype], num_q_heads=s.num_q_heads,
              num_kv_heads=s.num_kv_heads, qk_dim=s.qk_dim, v_dim=s.v_dim, page_size=s.page_size,
              sm_scale=s.sm_scale, n_sink=s.n_sink, n_local=s.n_local, kv_shared=s.kv_shared,
              max_batch=s.batch, max_total_pages=w.total_pages, max_pages_per_req=w.max_pages_per_req,
              max_budget=w.max_budget, device=device or w.q.device,
              block_size=getattr(s, "block_size", 0),
              kv_format={"": VX_KV_SAME, "e4m3": VX_KV_FP8_E4M3, "e5m2": VX_KV_FP8_E5M2}[getattr(s, "kv_dtype", "")])
    kw.update(over)
    return Context(**kw)


def tables_for(w):
    sp, st, sh = w.strides
    pool = KvPool(w.k_pool, w.v_pool, sp, st, sh, getattr(w, "k_scale", 1.0), getattr(w, "v_scale", 1.0))
    pt = PageTable(w.page_indptr, w.page_indices, w.seq_lens, w.total_pages, w.max_pages_per_req)
    return pool, pt


def alloc_summary(w, summary_kind=VX_SUMMARY_ENVELOPE):
    s = w.spec
    bs = getattr(s, "block_size", 0)
    n = w.num_pool_pages * (s.page_size // bs if bs else 1)       # one summary per selection block (= page unless finer)
    shape = (n, s.num_kv_heads, s.qk_dim) if summary_kind == VX_SUMMARY_CENTROID else (n, s.num_kv_heads, 2, s.qk_dim)
    return torch.zeros(shape, dtype=w.k_pool.dtype, device=w.k_pool.device)
