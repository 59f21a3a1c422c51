"""Oracle-side glue (test infrastructure, like everything under oracle/): hand a workloads.Workload (torch tensors) to
oracle/vx_oracle.py (numpy).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import it."""
import numpy as np

from oracle import vx_oracle as vo


def to_oracle(w):
    """Workload (any device) -> (q, Pool, PageTable) numpy views on CPU copies.  With selection blocks finer than the page
    (spec.block_size) the pool and the table are the BLOCK-level ones of oracle/vx_oracle_blocks.py (page_size = block size)."""
    q, pool, pt = _to_oracle_pages(w)
    bs = getattr(w.spec, "block_size", 0)
    if bs and bs != w.spec.page_size:
        from oracle.vx_oracle_blocks import block_problem
        pool, pt = block_problem(pool, pt, bs, w.spec.num_kv_heads, w.spec.qk_dim, w.spec.v_dim)
    return q, pool, pt


def block_table(w):
    """(indptr, indices) of the selection units of a workload: the page table, or its expansion into blocks (G28)"""
    indptr, indices = vo.as_np(w.page_indptr).astype(np.int64), vo.as_np(w.page_indices).astype(np.int64)
    bs = getattr(w.spec, "block_size", 0)
    if bs and bs != w.spec.page_size:
        bpp = w.spec.page_size // bs
        return indptr * bpp, (indices[:, None] * bpp + np.arange(bpp)[None, :]).reshape(-1)
    return indptr, indices


def _to_oracle_pages(w):
    sp, st, sh = w.strides
    if getattr(w.spec, "kv_dtype", ""):                  # fp8 KV cache: the doubles scale * decode(code) (vx_oracle_fp8.py)
        from oracle.vx_oracle_fp8 import pool_fp8
        pool = pool_fp8(vo.as_np(w.k_pool), None if w.v_pool is None else vo.as_np(w.v_pool), w.spec.kv_dtype,
                        w.k_scale, w.v_scale, sp, st, sh, w.num_pool_pages)
        pt = vo.PageTable(vo.as_np(w.page_indptr), vo.as_np(w.page_indices), vo.as_np(w.seq_lens), w.spec.page_size)
        return vo.as_np(w.q), pool, pt
    pool = vo.Pool(k=vo.as_np(w.k_pool), v=None if w.v_pool is None else vo.as_np(w.v_pool),
                   stride_page=sp, stride_token=st, stride_head=sh, num_pool_pages=w.num_pool_pages)
    pt = vo.PageTable(vo.as_np(w.page_indptr), vo.as_np(w.page_indices), vo.as_np(w.seq_lens),
                      w.spec.page_size)
    return vo.as_np(w.q), pool, pt


def oracle_step(w, agg=vo.AGG_SUM):
    q, pool, pt = to_oracle(w)
    s = w.spec
    return vo.decode_step(q, pool, pt, vo.as_np(w.budget), w.max_budget, s.num_q_heads,
                          s.num_kv_heads, s.qk_dim, s.v_dim, s.sm_scale, s.n_sink, s.n_local, agg)


def bf16_bits_to_f64(a):
    if a.dtype == np.uint16:
        return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return a.astype(np.float64)


def parity_sample(w, requests, sel_logical, sel_count, out, lse):
    """Counts for bench.py's "parity" object: the GPU's step outputs for the sampled `requests` of workload `w` against the
    oracle (selection sets by the 1e-3 near-tie rule, attention on the GPU's own selected set).  No assertion here -- the
    asserting comparators are tests/parity.py; this reports what they would see."""
    from paper_2606_06453_b200.workloads import subproblem
    s = w.spec
    st = dict(requests=list(requests), problems=0, excepted=0, swapped_pages=0, beyond_rule=0, out_max_abs=0.0,
              out_row_rel=0.0, lse_max_abs=0.0)
    sl_all, sc_all = vo.as_np(sel_logical), vo.as_np(sel_count)
    o_all, l_all = vo.as_np(out.float()), vo.as_np(lse)
    for r in requests:
        sub = subproblem(w, [r])
        ref = oracle_step(sub)
        sl, sc = sl_all[r:r + 1], sc_all[r:r + 1]
        indptr = vo.as_np(sub.page_indptr)
        for h in range(sc.shape[1]):
            n = int(sc[0, h])
            st["problems"] += 1
            got, want = sl[0, h, :n], ref["sel_logical"][0, h, :n]
            if n != int(ref["sel_count"][0, h]):
                st["beyond_rule"] += 1
                continue
            if np.array_equal(got, want):
                continue
            diff = np.setxor1d(got, want)
            thr = ref["thr"][0, h]
            sco = ref["scores"][h, indptr[0] + diff]
            rel = np.abs(sco - thr) / np.maximum(np.abs(sco), np.abs(thr))
            st["excepted"] += 1
            st["swapped_pages"] += int(len(diff))
            st["beyond_rule"] += int((rel >= 1e-3).sum())
        q, opool, opt = to_oracle(sub)
        o_ref, l_ref = vo.sparse_attention(q, opool, opt, sl, sc, s.num_q_heads, s.num_kv_heads, s.qk_dim, s.v_dim, s.sm_scale)
        err = np.abs(o_all[r:r + 1].astype(np.float64) - o_ref)
        st["out_max_abs"] = max(st["out_max_abs"], float(err.max()))
        st["out_row_rel"] = max(st["out_row_rel"], float((err.max(-1) / np.maximum(np.abs(o_ref).max(-1), 1e-30)).max()))
        st["lse_max_abs"] = max(st["lse_max_abs"], float(np.abs(l_all[r:r + 1].astype(np.float64) - l_ref).max()))
    return st
