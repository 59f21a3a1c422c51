"""Oracle-side glue (test infrastructure, like everything under oracle/): hand a workloads.Workload (torch tensors) to
oracle/vx_oracle.py (numpy).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import it."""
import numpy as np

from oracle import vx_oracle as vo


def to_oracle(w):
    """Workload (any device) -> (q, Pool, PageTable) numpy views on CPU copies."""
    sp, st, sh = w.strides
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
