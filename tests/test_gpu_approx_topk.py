"""vx_topk_pages_approx (-m gpu).

THE PARITY GATE is `check_against_exact`: every case's GPU output is held against the EXACT C oracle
(oracle/vx_oracle.c, a full sort -- code that shares nothing with the kernel) by the properties the paper fixes for a
lossy selection: recall@k >= 1 - tolerate_ratio (|exact minus gpu| <= floor(tolerate_ratio * k), :196, :538), forced pages
present (:280), sel_count = min(k, P), strictly ascending in-range ids, physical ids through the page table, the same
seed gives the same set, and tolerate_ratio = 0 gives the exact set.

The bit-equality with oracle/vx_oracle_approx.py that the tests also assert is a REGRESSION check only: that file
follows the kernel's encoding (bin count, remap, sampler; readings G20-G23), so agreeing with it shows that the
encoding did not drift, not that it is right."""
import numpy as np
import pytest
import torch

from oracle import vx_oracle as vo
from oracle import vx_oracle_approx as va
from paper_2606_06453_b200.workloads import APPD_DISTRIBUTIONS, appd_scores
from tests.test_gpu_topk_fuzz import KINDS, draw_scores

pytestmark = pytest.mark.gpu


def check_against_exact(scores, pages, seq, indices, budget, n_sink, n_local, tau, gpu, b=16):
    """the structure-independent gate: GPU output vs the exact C oracle (see the module docstring)"""
    sl, sp, sc = gpu
    indptr = np.concatenate([[0], np.cumsum(pages)]).astype(np.int64)
    pt_o = vo.PageTable(indptr.astype(np.int32), indices, np.array(seq, np.int32), b)
    mb = int(budget.max())
    sl_e, _, sc_e, _ = vo.topk_pages(scores.astype(np.float64), pt_o, budget, n_sink, n_local, mb)
    assert np.array_equal(sc, sc_e), "sel_count != min(k, P)"
    worst = 1.0
    for i, P in enumerate(pages):
        k = min(int(budget[i]), mb)
        for h in range(scores.shape[0]):
            n = int(sc_e[i, h])
            assert n == min(k, P)
            got = sl[i, h, :n]
            assert (sl[i, h, n:] == -1).all() and (sp[i, h, n:] == -1).all(), "padding"
            assert got.min(initial=0) >= 0 and got.max(initial=0) < P and (np.diff(got) > 0).all(), "ascending in-range ids"
            assert np.array_equal(sp[i, h, :n], indices[indptr[i] + got]), "physical ids follow the page table"
            forced = [j for j in range(P) if j < n_sink or j >= P - n_local]
            if k >= len(forced):
                assert set(forced) <= set(got.tolist()), "forced pages (PAPER.md:280)"
            missed = len(set(sl_e[i, h, :n].tolist()) - set(got.tolist()))
            allowed = int(np.floor(np.float32(tau) * np.float32(k)))
            assert missed <= allowed, f"request {i} head {h}: {missed} exact pages missed, {allowed} allowed at ratio {tau}"
            if n:
                worst = min(worst, 1.0 - missed / n)
            if tau == 0.0:
                assert np.array_equal(got, sl_e[i, h, :n]), "ratio 0 is the exact selection"
    return worst


def run_both(scores, pages, seq, indices, budget, n_sink, n_local, tau, seed, b=16, remap=None):
    import paper_2606_06453_b200 as vx
    hkv = scores.shape[0]
    indptr = np.concatenate([[0], np.cumsum(pages)]).astype(np.int32)
    T = int(indptr[-1])
    mb = int(budget.max())
    ref = va.approx_topk_pages(scores, indptr, indices, np.array(seq, np.int32), b, budget, n_sink, n_local, mb, tau, seed,
                               remap=remap)
    dev = "cuda:0"
    ctx = vx.Context(dtype=torch.bfloat16, num_q_heads=4 * hkv, num_kv_heads=hkv, qk_dim=128, v_dim=128, page_size=b,
                     sm_scale=1.0, n_sink=n_sink, n_local=n_local, max_batch=len(pages), max_total_pages=T,
                     max_pages_per_req=max(pages), max_budget=mb, device=dev)
    pt = vx.PageTable(torch.from_numpy(indptr).to(dev), torch.from_numpy(indices).to(dev),
                      torch.tensor(seq, dtype=torch.int32, device=dev), T, max(pages))
    if remap is not None:
        ctx.set_topk_remap(remap)
    sl = torch.full((len(pages), hkv, mb), -7, dtype=torch.int32, device=dev)
    sp = torch.full_like(sl, -7)
    sc = torch.full((len(pages), hkv), -7, dtype=torch.int32, device=dev)
    ctx.topk_pages_approx(torch.from_numpy(scores).to(dev), pt, torch.from_numpy(budget).to(dev), mb, tau, seed,
                          sp, sl, sc)
    torch.cuda.synchronize()
    gpu = (sl.cpu().numpy(), sp.cpu().numpy(), sc.cpu().numpy())
    sl2, sp2 = torch.full_like(sl, -7), torch.full_like(sl, -7)         # the same seed reproduces the selection
    ctx.topk_pages_approx(torch.from_numpy(scores).to(dev), pt, torch.from_numpy(budget).to(dev), mb, tau, seed,
                          sp2, sl2, sc)
    torch.cuda.synchronize()
    assert torch.equal(sl2, sl) and torch.equal(sp2, sp)
    ctx.close()
    check_against_exact(scores, pages, seq, indices, budget, n_sink, n_local, tau, gpu, b)     # the parity gate
    return ref, gpu


@pytest.mark.parametrize("dist", APPD_DISTRIBUTIONS)
@pytest.mark.parametrize("tau", [0.0, 0.05, 0.25, 1.0])
def test_appd_distributions(dist, tau):
    rng = np.random.default_rng(5)
    pages = [2048, 777, 8192, 40, 4100]
    hkv = 2
    T = sum(pages)
    seq = [p * 16 - int(rng.integers(0, 16)) for p in pages]
    indices = rng.permutation(T + 9)[:T].astype(np.int32)
    budget = np.array([128, 64, 256, 64, 200], np.int32)
    scores = appd_scores(dist, (hkv, T), seed=31).numpy()
    (sl_r, sp_r, sc_r, early), (sl, sp, sc) = run_both(scores, pages, seq, indices, budget, 1, 2, tau, 2024)
    assert np.array_equal(sc, sc_r)
    assert np.array_equal(sl, sl_r), (dist, tau)
    assert np.array_equal(sp, sp_r), (dist, tau)
    if tau == 1.0:
        assert early[[0, 1, 2, 4]].all()          # budget < pages: one pass, then the sampler (request 3: k >= P)
    if tau == 0.0:                                # ratio 0 is the exact selection (the C oracle's full sort)
        indptr = np.concatenate([[0], np.cumsum(pages)]).astype(np.int32)
        pt_o = vo.PageTable(indptr, indices, np.array(seq, np.int32), 16)
        sl_e, _, _, _ = vo.topk_pages(scores.astype(np.float64), pt_o, budget, 1, 2, int(budget.max()))
        assert np.array_equal(sl, sl_e)


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("tau", [0.1, 0.5])
def test_fuzz_kinds(kind, tau):
    rng = np.random.default_rng(77 + KINDS.index(kind))
    n_sink, n_local = int(rng.integers(0, 3)), int(rng.integers(0, 4))
    pages = [int(x) for x in rng.choice([1, 3, 40, 300, 1025, 2048, 5000, 8192], size=5)]
    seq = [p * 16 - int(rng.integers(0, 16)) for p in pages]
    T = sum(pages)
    indices = rng.permutation(T + 17)[:T].astype(np.int32)
    budget = np.array([max(n_sink + n_local, int(rng.integers(1, max(2, min(p + 3, 600))))) for p in pages], np.int32)
    scores = np.stack([draw_scores(rng, kind, T) for _ in range(2)])
    (sl_r, sp_r, sc_r, _), (sl, sp, sc) = run_both(scores, pages, seq, indices, budget, n_sink, n_local, tau, 9)
    assert np.array_equal(sc, sc_r)
    assert np.array_equal(sl, sl_r), kind
    assert np.array_equal(sp, sp_r), kind


@pytest.mark.parametrize("dist", APPD_DISTRIBUTIONS)
@pytest.mark.parametrize("tau", [0.05, 0.25])
def test_seed_changes_only_the_sampled_members_and_recall_holds(dist, tau):
    pages, k = [4096], 128
    scores = appd_scores(dist, (8, 4096), seed=41).numpy()
    indices = np.arange(4096, dtype=np.int32)
    budget = np.array([k], np.int32)
    exact = run_both(scores, pages, [4096 * 16], indices, budget, 1, 2, 0.0, 0)[1][0]
    (_, _, _, early), (a, _, _) = run_both(scores, pages, [4096 * 16], indices, budget, 1, 2, tau, 1)
    b = run_both(scores, pages, [4096 * 16], indices, budget, 1, 2, tau, 2)[1][0]
    if early.any():
        assert not np.array_equal(a, b)
    for h in range(8):                                  # (run_both has already held a and b against the exact oracle)
        assert va.recall_at_k(a[0, h], exact[0, h]) >= 1 - tau
        assert va.recall_at_k(b[0, h], exact[0, h]) >= 1 - tau
        if not early[0, h]:
            assert np.array_equal(a[0, h], exact[0, h])


@pytest.mark.parametrize("dist", APPD_DISTRIBUTIONS)
@pytest.mark.parametrize("tau", [0.05, 0.25, 1.0])
def test_long_requests_beyond_the_register_kernel(dist, tau):
    """requests of more than 8,192 pages: the lossy selection in the shared-memory-key kernel (cta_select_pages<.., kApprox>)"""
    rng = np.random.default_rng(11)
    pages = [9000, 20000, 300, 33001]
    hkv = 2
    T = sum(pages)
    seq = [p * 16 - int(rng.integers(0, 16)) for p in pages]
    indices = rng.permutation(T + 5)[:T].astype(np.int32)
    budget = np.array([256, 1500, 64, 400], np.int32)
    scores = appd_scores(dist, (hkv, T), seed=57).numpy()
    (sl_r, sp_r, sc_r, early), (sl, sp, sc) = run_both(scores, pages, seq, indices, budget, 1, 2, tau, 77)
    assert np.array_equal(sc, sc_r) and np.array_equal(sl, sl_r) and np.array_equal(sp, sp_r), (dist, tau)
    if tau == 1.0:
        assert early.all()


@pytest.mark.parametrize("kind", KINDS)
def test_long_requests_fuzz_kinds(kind):
    rng = np.random.default_rng(177 + KINDS.index(kind))
    n_sink, n_local = int(rng.integers(0, 3)), int(rng.integers(0, 4))
    pages = [int(x) for x in rng.choice([8193, 10000, 16384, 25000], size=3)]
    seq = [p * 16 - int(rng.integers(0, 16)) for p in pages]
    T = sum(pages)
    indices = rng.permutation(T + 3)[:T].astype(np.int32)
    budget = np.array([int(rng.integers(n_sink + n_local + 1, 900)) for _ in pages], np.int32)
    scores = np.stack([draw_scores(rng, kind, T) for _ in range(2)])
    (sl_r, sp_r, sc_r, _), (sl, sp, sc) = run_both(scores, pages, seq, indices, budget, n_sink, n_local, 0.25, 5)
    assert np.array_equal(sc, sc_r) and np.array_equal(sl, sl_r) and np.array_equal(sp, sp_r), kind


def test_argument_checks():
    import paper_2606_06453_b200 as vx
    dev = "cuda:0"
    P = 50000                                      # beyond the 49,152 keys the shared-memory-key kernel caches
    ctx = vx.Context(dtype=torch.bfloat16, num_q_heads=8, num_kv_heads=2, qk_dim=128, v_dim=128, page_size=16,
                     sm_scale=1.0, n_sink=1, n_local=2, max_batch=1, max_total_pages=P, max_pages_per_req=P,
                     max_budget=64, device=dev)
    pt = vx.PageTable(torch.tensor([0, P], dtype=torch.int32, device=dev), torch.arange(P, dtype=torch.int32, device=dev),
                      torch.tensor([P * 16], dtype=torch.int32, device=dev), P, P)
    scores = torch.randn(2, P, device=dev)
    budget = torch.tensor([64], dtype=torch.int32, device=dev)
    sl = torch.empty(1, 2, 64, dtype=torch.int32, device=dev)
    sp, sc = torch.empty_like(sl), torch.empty(1, 2, dtype=torch.int32, device=dev)
    with pytest.raises(vx.VortexError):           # more pages per request than either lossy kernel holds
        ctx.topk_pages_approx(scores, pt, budget, 64, 0.25, 1, sp, sl, sc)
    with pytest.raises(vx.VortexError):
        ctx.topk_pages_approx(scores, pt, budget, 64, 1.5, 1, sp, sl, sc)
    with pytest.raises(vx.VortexError):
        ctx.set_topk_approx(-0.1, 1)
    ctx.topk_pages_approx(scores, pt, budget, 64, 0.0, 1, sp, sl, sc)     # ratio 0: the exact kernel, any size
    torch.cuda.synchronize()
    ctx.close()


@pytest.mark.parametrize("name", ["C2-small", "C4-small", "C5-small"])
def test_fused_step_with_approximate_selection(name):
    """VX_STEP_APPROX_TOPK: the fused step selects with the approximate kernel (vx_set_topk_approx's ratio and seed):
    its selection equals the approximate oracle's on the GPU's own fp32 scores bit for bit, and its attention output
    matches the fp64 oracle evaluated on that selection within the bf16 tolerances."""
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload
    from tests.parity import check_attention, oracle_attention_on
    w = make_workload(name, device="cuda:0")
    s = w.spec
    dev = "cuda:0"
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    scores = torch.empty(s.num_kv_heads, w.total_pages, dtype=torch.float32, device=dev)
    ctx.page_score(w.q, summary, pt, scores)
    tau, seed = 0.25, 123
    ctx.set_topk_approx(tau, seed)
    out = torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev)
    lse = torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    sl = torch.full((s.batch, s.num_kv_heads, w.max_budget), -7, dtype=torch.int32, device=dev)
    sp, sc = torch.full_like(sl, -7), torch.full((s.batch, s.num_kv_heads), -7, dtype=torch.int32, device=dev)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc,
                           flags=vx.VX_STEP_UPDATE_SUMMARY | vx.VX_STEP_APPROX_TOPK)
    torch.cuda.synchronize()
    sl_r, sp_r, sc_r, early = va.approx_topk_pages(scores.cpu().numpy(), w.page_indptr.cpu().numpy(),
                                                   w.page_indices.cpu().numpy(), w.seq_lens.cpu().numpy(), s.page_size,
                                                   w.budget.cpu().numpy(), s.n_sink, s.n_local, w.max_budget, tau, seed)
    assert early.any()                                                  # the lossy path was actually taken
    pages = [int(x) for x in np.diff(w.page_indptr.cpu().numpy())]
    check_against_exact(scores.cpu().numpy(), pages, w.seq_lens.cpu().numpy().tolist(), w.page_indices.cpu().numpy(),
                        w.budget.cpu().numpy(), s.n_sink, s.n_local, tau,
                        (sl.cpu().numpy(), sp.cpu().numpy(), sc.cpu().numpy()), b=s.page_size)   # the parity gate
    assert np.array_equal(sc.cpu().numpy(), sc_r)
    assert np.array_equal(sl.cpu().numpy(), sl_r) and np.array_equal(sp.cpu().numpy(), sp_r)
    o_ref, l_ref = oracle_attention_on(w, sl.cpu().numpy(), sc.cpu().numpy())
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)
    ctx.close()


# ---- the offline-profiled remap of the first pass (App. D.2; reading G29; vx_set_topk_remap) --------

def _random_knots(rng, n):
    return np.sort(rng.random(n)).astype(np.float32)


@pytest.mark.parametrize("dist", APPD_DISTRIBUTIONS)
@pytest.mark.parametrize("tau", [0.0, 0.1, 0.5])
def test_remap_profiled_on_the_distribution(dist, tau):
    """the table fitted offline to OTHER draws of the distribution; ratio 0 must stay the exact selection (run_both's gate)"""
    from paper_2606_06453_b200.remap_profile import profile_knots
    rng = np.random.default_rng(15)
    pages = [2048, 777, 8192, 40, 4100]
    T = sum(pages)
    seq = [p * 16 - int(rng.integers(0, 16)) for p in pages]
    indices = rng.permutation(T + 9)[:T].astype(np.int32)
    budget = np.array([128, 64, 256, 64, 200], np.int32)
    scores = appd_scores(dist, (2, T), seed=131).numpy()
    knots = profile_knots(appd_scores(dist, (8, 4096), seed=977).numpy(), 33)
    (sl_r, sp_r, sc_r, early), (sl, sp, sc) = run_both(scores, pages, seq, indices, budget, 1, 2, tau, 4, remap=knots)
    assert np.array_equal(sc, sc_r) and np.array_equal(sl, sl_r) and np.array_equal(sp, sp_r), (dist, tau)
    if tau == 0.0:
        assert not early.any()


@pytest.mark.parametrize("kind", KINDS)
def test_remap_random_tables_on_the_fuzz_kinds_stay_exact(kind):
    """any monotone table, nasty score sets (ties, signed zeros, denormals, 40 decades), short and long requests:
    at ratio 0 the selection is the exact one (held against the C oracle inside run_both) and equals the mirror oracle"""
    rng = np.random.default_rng(277 + KINDS.index(kind))
    n_sink, n_local = int(rng.integers(0, 3)), int(rng.integers(0, 4))
    pages = [int(x) for x in rng.choice([3, 40, 300, 1025, 2048, 5000, 8192, 9000, 16384], size=4)]
    seq = [p * 16 - int(rng.integers(0, 16)) for p in pages]
    T = sum(pages)
    indices = rng.permutation(T + 17)[:T].astype(np.int32)
    budget = np.array([max(n_sink + n_local, int(rng.integers(1, max(2, min(p + 3, 600))))) for p in pages], np.int32)
    scores = np.stack([draw_scores(rng, kind, T) for _ in range(2)])
    knots = [np.zeros(5, np.float32), np.array([0, 1], np.float32), _random_knots(rng, 65), _random_knots(rng, 3)][KINDS.index(kind) % 4]
    for tau in (0.0, 0.25):
        (sl_r, sp_r, sc_r, _), (sl, sp, sc) = run_both(scores, pages, seq, indices, budget, n_sink, n_local, tau, 9, remap=knots)
        assert np.array_equal(sc, sc_r) and np.array_equal(sl, sl_r) and np.array_equal(sp, sp_r), (kind, tau)


def test_remap_in_the_fused_step_and_argument_checks():
    """VX_STEP_APPROX_TOPK with a table and ratio 0: the step's selections and outputs are those of the exact step"""
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200 import binding
    from paper_2606_06453_b200.remap_profile import profile_knots
    from paper_2606_06453_b200.workloads import make_workload
    w = make_workload("C2-small", device="cuda:0")
    s = w.spec
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    outs = []
    for flags, knots in ((0, None), (binding.VX_STEP_APPROX_TOPK, profile_knots(np.random.default_rng(1).standard_normal((4, 500)), 17))):
        if knots is not None:
            ctx.set_topk_remap(knots)
            ctx.set_topk_approx(0.0, 3)
        out = torch.empty(s.batch, s.num_q_heads, s.v_dim, dtype=w.q.dtype, device="cuda:0")
        sp = torch.full((s.batch, s.num_kv_heads, w.max_budget), -7, dtype=torch.int32, device="cuda:0")
        sl, sc = torch.full_like(sp, -7), torch.full((s.batch, s.num_kv_heads), -7, dtype=torch.int32, device="cuda:0")
        ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, None, sp, sl, sc, flags=flags)
        torch.cuda.synchronize()
        outs.append((out, sp, sl, sc))
    for a, b in zip(outs[0], outs[1]):
        assert torch.equal(a, b)
    for bad in ([0.5], [0.2, 0.1], [0.0, 1.5], [float("nan"), 1.0], list(np.linspace(0, 1, 66))):
        with pytest.raises(vx.VortexError):
            ctx.set_topk_remap(bad)
    ctx.set_topk_remap(None)                      # cleared: back to the linear map
    ctx.close()
