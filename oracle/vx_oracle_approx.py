"""Approximate radix top-k page selection (stochastic early termination) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It does not import paper_2606_06453_b200 and shares no code with the CUDA path.

What the paper fixes (PAPER.md:194-196 section 5.2, :538 Table 1 `approxTopK`, :495-509 App. D.2/D.3):
a radix top-k "iteratively partitions values into bins based on their radix digits"; the lossy variant
"terminates early once enough high-confidence candidates have been collected and then randomly samples
the remaining elements from the threshold bin", with `tolerate_ratio in [0, 1]` trading exactness for
speed, judged by recall@k.  The paper prints no pseudo-code, bin count, termination test or sampler, so
this is an ENCODING whose free choices are the readings G20-G23 of DESIGN.md section 12; the oracle
follows them step by step, in this order, with plain numpy (uint32 / float32 scalars and arrays):

  per (request i, KV head h), P pages, budget k (forced pages included, G4), forced set F (G6):
  0. k >= P: every page.  Otherwise candidates = pages not in F, need = k - |F| of them are to be taken.
  1. key(j) = order-preserving uint32 of the fp32 score (-0.0 and +0.0 share a key).  [lo, lo+width) is the
     live key range, first the candidates' [kmin, kmax].
  2. one radix pass = a 2,048-bin histogram of the candidates inside the live range.  Bin of a key:
     (key - lo) >> shift with shift = max(0, bitlen(width - 1) - 11); on the FIRST pass only, when the range
     spans at least 2^25 key steps, the monotone remap  bin = min(2047, int((score - smin) * (2048 /
     (smax - smin))))  in fp32 ("monotonic transformation ... fused into the histogram pass").
  3. threshold bin t = the highest bin with  #(keys in bins > t) < need <= #(keys in bins >= t).  The keys in
     bins > t are the pass's high-confidence candidates: all are taken; need -= their number.
  4. the bin is a single key value (integer pass with shift == 0): take the `need` lowest-index members. Done.
  5. EARLY TERMINATION (G21): if need <= floor(tolerate_ratio * k) (fp32 product), take `need` of the bin's cnt
     members as a random cyclic window (G22): members ranked r = 0..cnt-1 by logical page index, start
     s = splitmix64(seed, problem = i * Hkv + h) >> 32 mod cnt, taken iff (r - s) mod cnt < need.  Done.
  6. cnt <= 256: the bin is resolved exactly (the `need` best members, ties to the lower index).  Done (G23).
  7. otherwise the live range becomes the bin's (float pass: [min, max] key of its members; integer pass: the
     bin's key interval) and the algorithm continues at 2.
  Emission: forced pages, every candidate above the final threshold bin, the chosen members; ascending
  logical order; physical ids through the page table; count = min(k, P).

REMAP (App. D.2 "we apply a monotonic transformation x' = f(x) that preserves ordering while reshaping the
value distribution ... selected offline through profiling and fused into the histogram pass"; reading G29): an
optional table of n knot values 0 <= u_0 <= ... <= u_{n-1} <= 1 (2 <= n <= 65) is f on the normalised score, piecewise
linear between the knots at t = 0, 1/(n-1), ..., 1.  With a table installed the FIRST pass always bins through it (whatever
the key range), every operation rounded to fp32 in this order:
     x = (score - smin) * ((n-1) / (smax - smin));   i = min(n-2, int(x));   fr = x - i;
     u = min(u_{i+1}, fr * (u_{i+1} - u_i) + u_i);   bin = min(2047, int(u * 2048))
(the min with u_{i+1} keeps the bin non-decreasing in the score across a knot whatever the rounding, which is all the
selection needs: the members of a bin are then a contiguous key interval, and steps 3-7 are unchanged).  The table is an
INPUT here; how it is profiled is the product's business (paper_2606_06453_b200/remap_profile.py).

tolerate_ratio = 0 never terminates early and is the exact selection (with or without a remap).  At most floor(tolerate_ratio * k)
selected pages differ from the exact set, so recall@k >= 1 - tolerate_ratio.

Pins (tests/test_oracle_approx_topk.py): tolerate_ratio 0 == the exact oracle (vx_oracle.c, a full sort) and
== brute force on tiny inputs; splitmix64 against its published test vector; count / forced / order
invariants; every page taken above the threshold bin is in the exact top-k; the recall bound; wrongly taken
pages lie within one bin width of the exact threshold; inclusion frequency need / cnt over seeds.
"""
from __future__ import annotations

import numpy as np

K_BINS = 2048
K_BIN_BITS = 11
K_LIST = 256
_M64 = (1 << 64) - 1


def splitmix64(seed: int, index: int) -> int:
    """The (index+1)-th output of the SplitMix64 generator started at `seed` (Steele, Lea, Flood 2014):
    counter-based, so a problem's draw needs no shared state."""
    z = (seed + 0x9E3779B97F4A7C15 * (index + 1)) & _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def float_keys(scores_f32: np.ndarray) -> np.ndarray:
    """Order-preserving uint32 key of each fp32 score (larger score <=> larger key; -0.0 == +0.0)."""
    u = np.ascontiguousarray(scores_f32, dtype=np.float32).view(np.uint32).copy()
    u[u == np.uint32(0x80000000)] = np.uint32(0)
    neg = (u & np.uint32(0x80000000)) != 0
    return np.where(neg, ~u, u | np.uint32(0x80000000)).astype(np.uint32)


def key_floats(keys: np.ndarray) -> np.ndarray:
    k = np.asarray(keys, dtype=np.uint32)
    pos = (k & np.uint32(0x80000000)) != 0
    return np.where(pos, k & np.uint32(0x7FFFFFFF), ~k).astype(np.uint32).view(np.float32)


def _bitlen(x: int) -> int:
    return int(x).bit_length()


def remap_bins(sc32: np.ndarray, smin, smax, knots: np.ndarray) -> np.ndarray:
    """The first-pass bin of each fp32 score under the knot table (reading G29), fp32 operation by operation."""
    u_k = np.ascontiguousarray(knots, dtype=np.float32)
    n = int(u_k.shape[0])
    with np.errstate(divide="ignore", invalid="ignore", over="ignore"):
        tscale = np.float32(n - 1) / np.float32(smax - smin)
        x = ((sc32 - np.float32(smin)).astype(np.float32) * tscale).astype(np.float32)
    i = np.minimum(n - 2, x.astype(np.int64))
    fr = (x - i.astype(np.float32)).astype(np.float32)
    d = (u_k[i + 1] - u_k[i]).astype(np.float32)
    u = np.minimum(u_k[i + 1], ((fr * d).astype(np.float32) + u_k[i]).astype(np.float32))
    return np.minimum(K_BINS - 1, (u * np.float32(K_BINS)).astype(np.float32).astype(np.int64))


def check_knots(knots) -> np.ndarray:
    u_k = np.ascontiguousarray(knots, dtype=np.float32)
    assert u_k.ndim == 1 and 2 <= u_k.shape[0] <= 65, "2..65 knots"
    assert np.all(np.isfinite(u_k)) and u_k.min() >= 0.0 and u_k.max() <= 1.0 and np.all(np.diff(u_k) >= 0), \
        "knots: finite, in [0, 1], non-decreasing"
    return u_k


def select_one(scores_f32: np.ndarray, k: int, n_sink: int, n_local: int, tolerate_ratio: float,
               seed: int, problem: int, remap=None):
    """One (request, KV head): scores of its P logical pages -> (sorted selected logical ids, info).
    remap: None, or the knot table of reading G29."""
    knots = None if remap is None else check_knots(remap)
    P = int(scores_f32.shape[0])
    info = {"passes": 0, "early": False, "sure": np.zeros(0, np.int64), "members": np.zeros(0, np.int64),
            "need": 0, "bin_width": 0.0}
    if k >= P:
        return np.arange(P, dtype=np.int64), info
    j = np.arange(P)
    forced = (j < n_sink) | (j >= P - n_local)
    n_forced = min(P, min(n_sink, P) + min(n_local, P))
    assert n_forced <= k, "precondition n_sink + n_local <= budget (G6)"
    need = k - n_forced
    if need <= 0:
        return j[forced].astype(np.int64), info
    cand = j[~forced]
    key = float_keys(scores_f32)[cand].astype(np.uint64)          # uint64 holds every intermediate exactly
    sc32 = key_floats(key.astype(np.uint32))                      # the score each key stands for (fp32)
    tol = int(np.floor(np.float32(tolerate_ratio) * np.float32(k)))
    kmin, kmax = int(key.min()), int(key.max())
    lo, width = kmin, kmax - kmin + 1
    shift = max(0, _bitlen(kmax - kmin) - K_BIN_BITS)
    smin = key_floats(np.array([kmin], np.uint32))[0]
    smax = key_floats(np.array([kmax], np.uint32))[0]
    with np.errstate(divide="ignore", invalid="ignore", over="ignore"):
        fscale = np.float32(K_BINS) / np.float32(smax - smin)
    fpass = ((kmax - kmin) >= (1 << 25) or knots is not None) and bool(np.isfinite(fscale)) and bool(fscale > 0)
    taken_above = np.zeros(cand.shape[0], dtype=bool)
    while True:
        info["passes"] += 1
        live = (key >= lo) & (key - np.uint64(lo) < np.uint64(width))
        if fpass and knots is not None:
            b = remap_bins(sc32, smin, smax, knots)
        elif fpass:
            b = np.minimum(K_BINS - 1, ((sc32 - smin).astype(np.float32) * fscale).astype(np.float32).astype(np.int64))
        else:
            b = ((key - np.uint64(lo)) >> np.uint64(shift)).astype(np.int64)
        b = np.where(live, b, -1)
        hist = np.bincount(b[live], minlength=K_BINS)
        above_of = np.concatenate([np.cumsum(hist[::-1])[::-1][1:], [0]])        # keys in bins > t
        t = max(tt for tt in range(K_BINS) if above_of[tt] < need <= above_of[tt] + hist[tt])
        taken_above |= live & (b > t)
        need -= int(above_of[t])
        members = live & (b == t)
        cnt = int(hist[t])
        m_idx = np.nonzero(members)[0]                            # ascending logical order (cand is ascending)
        info.update(need=need, members=cand[m_idx].astype(np.int64))
        if fpass and knots is not None:
            ms = sc32[m_idx]
            info["bin_width"] = float(ms.max()) - float(ms.min())    # (the spread of the bin's members: f has no closed inverse)
        elif fpass:
            info["bin_width"] = float(smax - smin) / K_BINS
        else:
            blo = lo + (t << shift)
            bhi = min(blo + (1 << shift) - 1, lo + width - 1, 0xFFFFFFFF)
            info["bin_width"] = float(key_floats(np.array([bhi], np.uint32))[0]) - \
                float(key_floats(np.array([blo], np.uint32))[0])
        if not fpass and shift == 0:                              # step 4: one key value
            chosen = m_idx[:need]
            break
        if need <= tol:                                           # step 5: stochastic early termination
            s = (splitmix64(seed, problem) >> 32) % cnt
            r = np.arange(cnt)
            chosen = m_idx[((r - s) % cnt) < need]
            info["early"] = True
            break
        if cnt <= K_LIST:                                         # step 6: exact among the members
            order = sorted(m_idx.tolist(), key=lambda c: (-int(key[c]), c))
            chosen = np.array(sorted(order[:need]), dtype=np.int64)
            break
        if fpass:                                                 # step 7: continue inside the bin
            mk = key[m_idx]
            lo, width = int(mk.min()), int(mk.max()) - int(mk.min()) + 1
            shift = max(0, _bitlen(width - 1) - K_BIN_BITS)
            fpass = False
        else:
            blo = lo + (t << shift)
            lo, width = blo, min(1 << shift, lo + width - blo)    # the window never leaves [lo, lo + width)
            shift = max(0, shift - K_BIN_BITS)
    info["sure"] = cand[taken_above].astype(np.int64)
    sel = np.concatenate([j[forced], cand[taken_above], cand[chosen]]).astype(np.int64)
    sel.sort()
    return sel, info


def approx_topk_pages(scores: np.ndarray, page_indptr, page_indices, seq_lens, page_size: int, budget,
                      n_sink: int, n_local: int, max_budget: int, tolerate_ratio: float, seed: int, remap=None):
    """scores fp32 [Hkv, T] ragged by page_indptr -> (sel_logical, sel_phys [B,Hkv,max_budget] pad -1,
    sel_count [B,Hkv], early [B,Hkv] bool)."""
    scores = np.ascontiguousarray(scores, dtype=np.float32)
    hkv = scores.shape[0]
    indptr = np.asarray(page_indptr, dtype=np.int64)
    indices = np.asarray(page_indices, dtype=np.int64)
    B = indptr.shape[0] - 1
    sl = np.full((B, hkv, max_budget), -1, dtype=np.int32)
    sp = np.full((B, hkv, max_budget), -1, dtype=np.int32)
    cnt = np.zeros((B, hkv), dtype=np.int32)
    early = np.zeros((B, hkv), dtype=bool)
    for i in range(B):
        P = (int(seq_lens[i]) + page_size - 1) // page_size
        k = min(int(budget[i]), max_budget)
        for h in range(hkv):
            row = scores[h, indptr[i]:indptr[i] + P]
            sel, info = select_one(row, k, n_sink, n_local, tolerate_ratio, seed, i * hkv + h, remap)
            n = sel.shape[0]
            assert n == min(k, P)
            sl[i, h, :n] = sel
            sp[i, h, :n] = indices[indptr[i] + sel]
            cnt[i, h] = n
            early[i, h] = info["early"]
    return sl, sp, cnt, early


def recall_at_k(sel_a: np.ndarray, sel_exact: np.ndarray) -> float:
    """recall@k: share of the exact top-k set that the approximate set holds."""
    a = set(int(x) for x in sel_a if x >= 0)
    e = set(int(x) for x in sel_exact if x >= 0)
    return len(a & e) / max(1, len(e))
