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


def check_selection(w, gpu_logical, gpu_phys, gpu_count, ref):
    """returns the number of (request, head) problems that needed the near-tie exception."""
    sl, sp, sc = (np.asarray(t) for t in (gpu_logical, gpu_phys, gpu_count))
    indptr = np.asarray(w.page_indptr.cpu())
    indices = np.asarray(w.page_indices.cpu())
    assert np.array_equal(sc, ref["sel_count"]), "sel_count differs"
    excepted = 0
    for i in range(sc.shape[0]):
        for h in range(sc.shape[1]):
            n = sc[i, h]
            got = sl[i, h, :n]
            assert (sl[i, h, n:] == -1).all() and (sp[i, h, n:] == -1).all(), "padding must be -1"
            assert (np.diff(got) > 0).all(), "logical ids must be strictly ascending (no duplicates)"
            assert np.array_equal(sp[i, h, :n], indices[indptr[i] + got]), "physical ids do not match the page table"
            want = ref["sel_logical"][i, h, :n]
            if np.array_equal(got, want):
                continue
            diff = np.setxor1d(got, want)
            thr = ref["thr"][i, h]
            s = ref["scores"][h, indptr[i] + diff]
            rel = np.abs(s - thr) / np.maximum(np.abs(s), np.abs(thr))
            assert np.isfinite(thr) and (rel < 1e-3).all(), \
                f"selection differs beyond the 1e-3 near-tie rule at request {i} head {h}: pages {diff}, rel {rel}"
            excepted += 1
    return excepted


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
