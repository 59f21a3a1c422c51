"""Parity comparators (BASELINE.json north_star criteria).

selection : sets per (request, KV head) must match the oracle exactly, except pages whose ORACLE
            score is within 1e-3 relative of the oracle's threshold (k-th) score.
attention : compared with the oracle evaluated on the GPU's own selected set:
            bf16: out max-abs <= 2e-2 and row-relative (inf-norm) <= 1e-2, LSE abs <= 1e-3
            fp32: out max-abs <= 1e-4, row-relative <= 1e-4, LSE abs <= 1e-5   (G17)
"""
import numpy as np

from oracle import vx_oracle as vo
from oracle.workload_io import to_oracle

TOL = {"bf16": dict(abs=2e-2, rel=1e-2, lse=1e-3), "f32": dict(abs=1e-4, rel=1e-4, lse=1e-5)}


NEAR_TIE = 1e-3          # north star: a differing page must score within this (relative) of the oracle's k-th score
FP32_BAND = 1e-4         # worst-case fp32 rounding of a 1,152-term score sum (n * 2^-24), rounded up
PARITY_LOG = []          # one record per check_selection call; conftest.py prints the totals and writes gpurun_out/parity_counts.json


class SelectionStats(dict):
    """problems, excepted (problems that needed the near-tie rule), swapped_pages (pages in the symmetric difference),
    fp32_band_pages (oracle pages within FP32_BAND of the threshold: the ceiling for swapped_pages), max_rel."""

    def __int__(self):
        return self["excepted"]

    def __radd__(self, other):
        return other + self["excepted"]

    def __add__(self, other):
        return self["excepted"] + int(other)


def check_selection(w, gpu_logical, gpu_phys, gpu_count, ref, label=None):
    """Selection parity per (request, KV head); returns SelectionStats (int(stats) = problems that needed the near-tie rule).
    The stated rule: a page in the symmetric difference must score within 1e-3 relative of the oracle's threshold.  On top
    of it the exception is BOUNDED: a problem may not swap more pages than the oracle itself finds inside the fp32 rounding
    band (FP32_BAND) around its threshold -- a kernel that mis-ranks pages 5e-4 apart passes the rule but not the ceiling."""
    sl, sp, sc = (np.asarray(t) for t in (gpu_logical, gpu_phys, gpu_count))
    from oracle.workload_io import block_table
    indptr, indices = block_table(w)                     # pages, or blocks finer than the page (physical block ids)
    assert np.array_equal(sc, ref["sel_count"]), "sel_count differs"
    st = SelectionStats(problems=0, excepted=0, swapped_pages=0, fp32_band_pages=0, max_rel=0.0)
    for i in range(sc.shape[0]):
        for h in range(sc.shape[1]):
            n = sc[i, h]
            got = sl[i, h, :n]
            st["problems"] += 1
            assert (sl[i, h, n:] == -1).all() and (sp[i, h, n:] == -1).all(), "padding must be -1"
            assert (np.diff(got) > 0).all(), "logical ids must be strictly ascending (no duplicates)"
            assert np.array_equal(sp[i, h, :n], indices[indptr[i] + got]), "physical ids do not match the page table"
            want = ref["sel_logical"][i, h, :n]
            thr = ref["thr"][i, h]
            if np.isfinite(thr):
                allp = ref["scores"][h, indptr[i]:indptr[i + 1]]
                band = int((np.abs(allp - thr) / np.maximum(np.abs(allp), np.abs(thr)) < FP32_BAND).sum())
            else:
                band = 0
            st["fp32_band_pages"] += band
            if np.array_equal(got, want):
                continue
            diff = np.setxor1d(got, want)
            s = ref["scores"][h, indptr[i] + diff]
            rel = np.abs(s - thr) / np.maximum(np.abs(s), np.abs(thr))
            assert np.isfinite(thr) and (rel < NEAR_TIE).all(), \
                f"selection differs beyond the 1e-3 near-tie rule at request {i} head {h}: pages {diff}, rel {rel}"
            assert len(diff) <= band, \
                f"request {i} head {h}: {len(diff)} pages swapped but only {band} oracle scores lie within {FP32_BAND} of the threshold"
            st["excepted"] += 1
            st["swapped_pages"] += len(diff)
            st["max_rel"] = max(st["max_rel"], float(rel.max()))
    PARITY_LOG.append(dict(st, label=label or getattr(w.spec, "name", "?")))
    return st


def oracle_attention_on(w, sel_logical, sel_count):
    q, pool, pt = to_oracle(w)
    s = w.spec
    return vo.sparse_attention(q, pool, pt, np.asarray(sel_logical), np.asarray(sel_count), s.num_q_heads,
                               s.num_kv_heads, s.qk_dim, s.v_dim, s.sm_scale)


def check_attention(dtype, out, lse, o_ref, l_ref):
    tol = TOL[dtype]
    out = np.asarray(out, dtype=np.float64)
    err = np.abs(out - o_ref)
    row_rel = err.max(-1) / np.maximum(np.abs(o_ref).max(-1), 1e-30)
    assert err.max() <= tol["abs"], f"out max-abs {err.max():.3e} > {tol['abs']}"
    assert row_rel.max() <= tol["rel"], f"out row-rel {row_rel.max():.3e} > {tol['rel']}"
    if lse is not None:
        lerr = np.abs(np.asarray(lse, dtype=np.float64) - l_ref).max()
        assert lerr <= tol["lse"], f"lse err {lerr:.3e} > {tol['lse']}"
    return float(err.max()), float(row_rel.max())
