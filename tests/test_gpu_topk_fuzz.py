"""Bit-exact fuzz of vx_topk_pages against the oracle (-m gpu): every path of the radix select -- direct ranking
of a small threshold bin, recursion into a heavy bin (more than 256 tied or near-tied keys), the float-domain
first pass for ranges that span the sign change or many exponents and its hand-over to integer keys, single-value
ranges, +-0, denormals -- on ragged batches with random budgets and forced-page settings.  Both sides decide on
the same fp32 values, so the comparison is exact (ids, order, counts, padding)."""
import numpy as np
import pytest
import torch

from oracle import vx_oracle as vo

pytestmark = pytest.mark.gpu


def draw_scores(rng, kind, n):
    if kind == "few_values":                    # heavy ties: >> 256 members in the threshold bin
        return rng.choice(np.array([-3.5, -1.0, 0.0, 0.25, 2.0], np.float32), size=n)
    if kind == "constant":
        return np.full(n, 7.125, np.float32)
    if kind == "signed_zero":
        return rng.choice(np.array([0.0, -0.0, 1e-30, -1e-30], np.float32), size=n)
    if kind == "bimodal_sign":                  # float first pass, light bins
        pick = rng.random(n) < 0.2
        return np.where(pick, rng.normal(40, 2, n), rng.normal(-10, 2, n)).astype(np.float32)
    if kind == "wide_then_ties":                # float first pass whose threshold bin is heavy -> integer hand-over
        base = rng.choice(np.array([-1000.0, 5.0, 5.0 + 2 ** -20, 5.0 + 2 ** -19, 6000.0], np.float32), size=n,
                          p=[0.2, 0.3, 0.2, 0.2, 0.1])
        return base
    if kind == "narrow":                        # same exponent, tiny spread: integer first pass, shift 0 quickly
        return (np.float32(900.0) + rng.integers(0, 12, n).astype(np.float32) * np.float32(2 ** -13))
    if kind == "lognormal":
        return np.exp(rng.normal(0, 2.0, n)).astype(np.float32)
    if kind == "denormal":
        return (rng.integers(-50, 50, n).astype(np.float32) * np.float32(1e-42)).astype(np.float32)
    if kind == "edge_ties":
        # > 256 ties at the TOP edge of a float-pass bin, a neighbour 1 ulp above (next float bin) and a member 3000 ulp
        # below: the heavy float bin is handed over as the unaligned key interval [b - 3000 ulp, b], its last 2-key
        # sub-bin is heavy again, and the recursion window must stop at b (round-1 advisor finding: it ran one key past
        # it and counted the neighbour twice).  With min -1 and max 3 the float bins are 2^-9 wide and
        # fl(s + 1) * 512 < 1024  <=>  s <= 1 - 2^-23, so b = 1 - 2^-23 is the last fp32 value of bin 1023.
        b = np.float32(1.0) - np.float32(2.0 ** -23)
        up = np.nextafter(b, np.float32(2.0))
        down = (b.view(np.uint32) - np.uint32(3000)).view(np.float32)
        return rng.choice(np.array([-1.0, 3.0, up, down, b], np.float32), size=n, p=[0.05, 0.05, 0.1, 0.1, 0.7])
    raise ValueError(kind)


KINDS = ["few_values", "constant", "signed_zero", "bimodal_sign", "wide_then_ties", "narrow", "lognormal", "denormal",
         "edge_ties"]


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("seed", [0, 1])
def test_topk_fuzz_is_bit_exact(kind, seed):
    import paper_2606_06453_b200 as vx
    rng = np.random.default_rng(1000 * seed + KINDS.index(kind))
    b = 16
    n_sink, n_local = int(rng.integers(0, 3)), int(rng.integers(0, 4))
    pages = [int(x) for x in rng.choice([1, 3, 40, 300, 1025, 2048, 5000, 9000, 20000], size=5)]
    hkv = 2
    seq = [p * b - int(rng.integers(0, b)) for p in pages]
    indptr = np.concatenate([[0], np.cumsum(pages)]).astype(np.int32)
    T = int(indptr[-1])
    indices = rng.permutation(T + 17)[:T].astype(np.int32)
    budget = np.array([max(n_sink + n_local, int(rng.integers(1, max(2, min(p + 3, 600))))) for p in pages], np.int32)
    mb = int(budget.max())
    scores = np.stack([draw_scores(rng, kind, T) for _ in range(hkv)])
    pt_o = vo.PageTable(indptr, indices, np.array(seq, np.int32), b)
    sl_r, sp_r, sc_r, _ = vo.topk_pages(scores.astype(np.float64), pt_o, budget, n_sink, n_local, mb)
    dev = "cuda:0"
    ctx = vx.Context(dtype=torch.bfloat16, num_q_heads=8, num_kv_heads=hkv, qk_dim=128, v_dim=128, page_size=b,
                     sm_scale=1.0, n_sink=n_sink, n_local=n_local, max_batch=len(pages), max_total_pages=T,
                     max_pages_per_req=max(pages), max_budget=mb, device=dev)
    pt = vx.PageTable(torch.from_numpy(indptr).to(dev), torch.from_numpy(indices).to(dev),
                      torch.tensor(seq, dtype=torch.int32, device=dev), T, max(pages))
    sl = torch.full((len(pages), hkv, mb), -7, dtype=torch.int32, device=dev)
    sp = torch.full_like(sl, -7)
    sc = torch.full((len(pages), hkv), -7, dtype=torch.int32, device=dev)
    ctx.topk_pages(torch.from_numpy(scores).to(dev), pt, torch.from_numpy(budget).to(dev), mb, sp, sl, sc)
    torch.cuda.synchronize()
    assert np.array_equal(sc.cpu().numpy(), sc_r)
    got = sl.cpu().numpy()
    for i in range(len(pages)):                 # exactly n_sel distinct in-range ids, whatever the oracle says
        for h in range(hkv):
            n = int(sc_r[i, h])
            assert len(set(got[i, h, :n].tolist())) == n and got[i, h, :n].min() >= 0 and got[i, h, :n].max() < pages[i]
    assert np.array_equal(got, sl_r), kind
    assert np.array_equal(sp.cpu().numpy(), sp_r), kind


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("big", [2049, 4096, 4097, 8192])
def test_topk_pair_kernel_fuzz_is_bit_exact(kind, big):
    """Few problems of 2,049..8,192 pages run on clusters of two CTAs (vx_topk_pair.cu): same bit-exact contract."""
    import paper_2606_06453_b200 as vx
    rng = np.random.default_rng(7000 + 10 * KINDS.index(kind) + big)
    b = 16
    n_sink, n_local = int(rng.integers(0, 3)), int(rng.integers(0, 4))
    pages = [big] + [int(x) for x in rng.choice([1, 3, 40, 300, 1025, 2048, 2100, big - 1, big], size=4)]
    hkv = 2
    seq = [p * b - int(rng.integers(0, b)) for p in pages]
    indptr = np.concatenate([[0], np.cumsum(pages)]).astype(np.int32)
    T = int(indptr[-1])
    indices = rng.permutation(T + 17)[:T].astype(np.int32)
    budget = np.array([max(n_sink + n_local, int(rng.integers(1, max(2, min(p + 3, 3000))))) for p in pages], np.int32)
    mb = int(budget.max())
    scores = np.stack([draw_scores(rng, kind, T) for _ in range(hkv)])
    pt_o = vo.PageTable(indptr, indices, np.array(seq, np.int32), b)
    sl_r, sp_r, sc_r, _ = vo.topk_pages(scores.astype(np.float64), pt_o, budget, n_sink, n_local, mb)
    dev = "cuda:0"
    ctx = vx.Context(dtype=torch.bfloat16, num_q_heads=8, num_kv_heads=hkv, qk_dim=128, v_dim=128, page_size=b,
                     sm_scale=1.0, n_sink=n_sink, n_local=n_local, max_batch=len(pages), max_total_pages=T,
                     max_pages_per_req=max(pages), max_budget=mb, device=dev)
    pt = vx.PageTable(torch.from_numpy(indptr).to(dev), torch.from_numpy(indices).to(dev),
                      torch.tensor(seq, dtype=torch.int32, device=dev), T, max(pages))
    for with_logical in (True, False):
        sl = torch.full((len(pages), hkv, mb), -7, dtype=torch.int32, device=dev)
        sp = torch.full_like(sl, -7)
        sc = torch.full((len(pages), hkv), -7, dtype=torch.int32, device=dev)
        ctx.topk_pages(torch.from_numpy(scores).to(dev), pt, torch.from_numpy(budget).to(dev), mb, sp,
                       sl if with_logical else None, sc)
        torch.cuda.synchronize()
        assert np.array_equal(sc.cpu().numpy(), sc_r)
        assert np.array_equal(sp.cpu().numpy(), sp_r), kind
        if with_logical:
            assert np.array_equal(sl.cpu().numpy(), sl_r), kind
    ctx.close()
