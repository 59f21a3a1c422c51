"""vx_sparse_paged_decode_static (-m gpu; collected last on purpose): the decode entry point that allocates nothing --
no context, no workspace, split partials in a file-scope device array -- against the existing vx_sparse_paged_decode
on the same selection, within the tolerances the parity tests use, on two calls in a row (the array keeps the first
call's contents).  Also: the torch allocator sees no allocation during the calls, and a problem beyond the array is refused."""
import ctypes as C

import pytest
import torch

from tests.parity import TOL, check_attention, oracle_attention_on

pytestmark = pytest.mark.gpu


def _setup(name):
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload
    w = make_workload(name, device="cuda:0")
    s = w.spec
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    dev = w.q.device
    out = torch.empty(s.batch, s.num_q_heads, s.v_dim, dtype=w.q.dtype, device=dev)
    lse = torch.empty(s.batch, s.num_q_heads, dtype=torch.float32, device=dev)
    sp = torch.empty(s.batch, s.num_kv_heads, w.max_budget, dtype=torch.int32, device=dev)
    sl, sc = torch.empty_like(sp), torch.empty(s.batch, s.num_kv_heads, dtype=torch.int32, device=dev)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc)
    ctx.sparse_paged_decode(w.q, pool, pt, sp, sl, sc, w.max_budget, out, lse)      # the existing path, same selection
    torch.cuda.synchronize()
    return vx, w, ctx, pool, pt, sp, sl, sc, out, lse


@pytest.mark.parametrize("name", ["C1", "C2-small", "C4-small", "C5-small"])
def test_static_decode_matches_the_existing_path_twice_in_a_row(name):
    vx, w, ctx, pool, pt, sp, sl, sc, out, lse = _setup(name)
    from paper_2606_06453_b200.binding import sparse_paged_decode_static
    s = w.spec
    o_ref, l_ref = oracle_attention_on(w, sl.cpu().numpy(), sc.cpu().numpy())
    tol = TOL[s.dtype]
    assert vx.load_library().vx_static_scratch_bytes() == 8 << 20
    for call in range(2):
        out2 = torch.full_like(out, float("nan"))
        lse2 = torch.full_like(lse, float("nan"))
        torch.cuda.synchronize()
        before = torch.cuda.memory_stats()["allocation.all.allocated"]
        sparse_paged_decode_static(ctx.geom, w.q, pool, pt, sp, sl, sc, w.max_budget, out2, lse2)
        torch.cuda.synchronize()
        assert torch.cuda.memory_stats()["allocation.all.allocated"] == before
        # against the existing path (both within the oracle tolerance of the truth, so twice that of each other) ...
        d = (out2.float() - out.float()).abs()
        assert float(d.max()) <= 2 * tol["abs"], (call, float(d.max()))
        assert float((lse2 - lse).abs().max()) <= 2 * tol["lse"], call
        # ... and against the oracle on the same selected set, by the parity comparator itself
        check_attention(s.dtype, out2.float().cpu().numpy(), lse2.cpu().numpy(), o_ref, l_ref)
        if call == 0:                                   # a different problem in between: the array holds ITS partials now
            q2 = torch.randn_like(w.q.float()).to(w.q.dtype)
            sparse_paged_decode_static(ctx.geom, q2, pool, pt, sp, sl, sc, w.max_budget, torch.empty_like(out), None)
    ctx.close()


def test_static_decode_refuses_what_does_not_fit():
    vx, w, ctx, pool, pt, sp, sl, sc, out, lse = _setup("C2-small")
    from paper_2606_06453_b200.binding import VxPageTable, sparse_paged_decode_static
    lib = vx.load_library()
    big = VxPageTable(100000, pt.c.page_indptr, pt.c.page_indices, pt.c.seq_lens, pt.c.total_pages, pt.c.max_pages_per_req)
    st = lib.vx_sparse_paged_decode_static(C.byref(ctx.geom), C.c_void_p(w.q.data_ptr()), C.byref(pool.c), C.byref(big),
                                           C.c_void_p(sp.data_ptr()), C.c_void_p(sl.data_ptr()), C.c_void_p(sc.data_ptr()),
                                           w.max_budget, C.c_void_p(out.data_ptr()), None, None)
    assert st == 3 and b"static" in lib.vx_static_last_error()          # VX_ERR_WORKSPACE, nothing launched
    with pytest.raises(vx.VortexError):
        sparse_paged_decode_static(ctx.geom, None, pool, pt, sp, sl, sc, w.max_budget, out, lse)
    torch.cuda.synchronize()
    ctx.close()
