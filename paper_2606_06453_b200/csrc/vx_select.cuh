// vx_select.cuh -- (a3) exact top-k page selection of ONE (request, KV head) problem by one CTA, keys in shared memory.
// PAPER.md:92 Eq.3 (arg-top-k of the block scores), :194 (radix top-k), :280 (first block and last blocks always
// attended; readings G4-G6: the budget includes the forced pages, ties go to the lower logical page,
// k >= P selects everything).
//
// The device function below is the selection as the standalone kernel `topk_kernel` (vx_topk.cu) runs it for
// requests whose keys fit shared memory, and as the fused MLA step kernel (vx_decode_mla.cu) runs it on the scores
// it has just computed: a range-adaptive radix select (2,048 bins over the LIVE key range of the request's
// candidates, first pass in the float domain when the range spans the sign change or several exponents, the few
// members of the threshold bin ranked directly, heavy ties recursing 11 bits at a time), then an ordered emission
// that resolves ties to the lowest logical page and leaves the selected ids in ascending logical order.
#pragma once
#include "vx_common.cuh"

namespace vx {

constexpr int kBins = 2048;                     // 11 bits per pass
constexpr int kBinBits = 11;
constexpr int kList = 256;                      // threshold-bin members ranked directly
constexpr uint32_t kForcedKey = 0xFFFFFFFFu;    // not the key of any finite float

__device__ __forceinline__ bool page_forced(int j, int n_pages, int n_sink, int n_local) {
  return (j < n_sink) || (j >= n_pages - n_local);
}

struct SelectScratch {                          // ~10 KB of shared memory
  int hist[kBins];                              // a pass's histogram; on return the selected logical pages, ascending
  uint32_t list[kList];
  uint32_t wmin[32], wmax[32];
  int wsum[32];
  int2 wcnt[32];
  int bin, above, cnt, nlist, need_eq;
  uint32_t thr, bmin, bmax;
  float knot[65];                               // kApprox: the remap's knot table (vx_internal.h kTopkRemapMaxKnots)
};

// keys[0 .. n_pages): on entry the BIT PATTERNS of the fp32 scores of logical pages 0 .. n_pages-1, on return their
// order-preserving keys (forced pages: kForcedKey).  k = the budget including forced pages (>= 0).
// Returns n_sel = min(k, n_pages) and leaves the selected logical pages in sc.hist[0 .. n_sel), ascending.
// Requires n_sel <= kBins.  Every one of the THREADS threads of the selecting group calls it (it synchronises the group);
// the caller has synchronised after writing keys[].  The group is the whole CTA (BAR = 0: __syncthreads) or the THREADS
// consecutive threads starting at thread TID0, which synchronise on the named barrier BAR while the rest of the CTA does
// something else (the flat MLA step kernel selects on one warpgroup while the other warps stream summaries).
template <int THREADS, int BAR>
__device__ __forceinline__ void select_sync() {
  if constexpr (BAR == 0) __syncthreads();
  else asm volatile("bar.sync %0, %1;" ::"n"(BAR), "n"(THREADS) : "memory");
}
// kApprox (PAPER.md:196 stochastic early termination, readings G20-G23): after a pass, when the pages
// still to take from the threshold bin number at most floor(tolerate_ratio * k), they are drawn from the bin's members as
// the cyclic window of member ranks (page order) that starts at a SplitMix64 draw of (seed, problem) -- the same rule,
// constants and order of tests as topk_reg_kernel<.., true>, so both kernels and oracle/vx_oracle_approx.py agree bit for bit.
template <int THREADS, int BAR = 0, int TID0 = 0, bool kApprox = false>
__device__ int cta_select_pages(SelectScratch& sc, uint32_t* keys, int n_pages, int k, int n_sink, int n_local,
                                float tolerate_ratio = 0.f, uint64_t seed = 0, int problem = 0,
                                const float* remap = nullptr, int remap_n = 0) {
  constexpr int WARPS = THREADS / kWarp;
  constexpr int BPT = kBins / THREADS;          // bins per thread in the suffix scan
  static_assert(kBins % THREADS == 0 && WARPS <= 32, "shape");
  const int tid = (int)threadIdx.x - TID0, lane = tid % kWarp, warp = tid / kWarp;
  const int n_sel = min(k, n_pages);
  if (k >= n_pages) {                           // G6: the budget covers the request -> every page
    for (int r = tid; r < n_pages; r += THREADS) sc.hist[r] = r;
    select_sync<THREADS, BAR>();
    return n_sel;
  }

  const int rn = kApprox ? remap_n : 0;         // knots of the offline-profiled remap (reading G29); 0: none
  if constexpr (kApprox)
    for (int t = tid; t < rn; t += THREADS) sc.knot[t] = remap[t];      // (visible after the barrier below)
  // ---- keys, and the min / max key of the non-forced pages ------------------------------------
  uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
  for (int j = tid; j < n_pages; j += THREADS) {
    const bool forced = page_forced(j, n_pages, n_sink, n_local);
    const uint32_t key = forced ? kForcedKey : float_to_key(__uint_as_float(keys[j]));
    keys[j] = key;
    if (!forced) { kmin = min(kmin, key); kmax = max(kmax, key); }
  }
  kmin = __reduce_min_sync(0xffffffffu, kmin);
  kmax = __reduce_max_sync(0xffffffffu, kmax);
  if (lane == 0) { sc.wmin[warp] = kmin; sc.wmax[warp] = kmax; }
  select_sync<THREADS, BAR>();
#pragma unroll
  for (int w = 0; w < WARPS; ++w) { kmin = min(kmin, sc.wmin[w]); kmax = max(kmax, sc.wmax[w]); }

  const int sink = min(n_sink, n_pages), local = min(n_local, n_pages);
  const int n_forced = min(n_pages, sink + local);
  int need = k - n_forced;                      // non-forced pages still to take (precondition: >= 0)
  uint32_t thr = kForcedKey;                    // take keys > thr, and the first need_eq keys == thr
  int need_eq = 0;
  // early termination (kApprox): ties = the members of the threshold bin (key interval [m_lo, m_hi], or float bin t_bin),
  // taken as the cyclic window of need_eq member ranks that starts at rot
  [[maybe_unused]] bool early = false, fterm = false;
  [[maybe_unused]] uint32_t m_lo = 0u, m_hi = 0u;
  [[maybe_unused]] int t_bin = 0, rot = 0, wrap = 0;
  const float smin = key_to_float(kmin), smax = key_to_float(kmax);
  const float fscale = (float)kBins / (smax - smin);
  const float tscale = (float)(rn - 1) / (smax - smin);
  auto fbin = [&](uint32_t key) -> int {        // (the same arithmetic, operation by operation, as topk_reg_kernel's)
    const float d0 = key_to_float(key) - smin;
    if (kApprox && rn > 0) {
      const float x = __fmul_rn(d0, tscale);
      const int i0 = max(0, min(rn - 2, (int)x));      // (>= 0 for every candidate; the emission also asks for absent pages)
      const float k0 = sc.knot[i0], k1 = sc.knot[i0 + 1];
      const float u = fminf(k1, __fadd_rn(__fmul_rn(__fsub_rn(x, (float)i0), __fsub_rn(k1, k0)), k0));
      return min(kBins - 1, (int)__fmul_rn(u, (float)kBins));
    }
    return min(kBins - 1, (int)(d0 * fscale));
  };

  if (need > 0) {
    // ---- radix select over the live key range [lo, lo + width) ----------------------------------
    uint32_t lo = kmin;
    uint64_t width = (uint64_t)(kmax - kmin) + 1;
    int shift = max(0, (32 - __clz(kmax - kmin)) - kBinBits);     // ((kmax - kmin) >> shift) < kBins
    [[maybe_unused]] const int tol = kApprox ? (int)(tolerate_ratio * (float)k) : 0;   // floor: both factors >= 0
    // First pass in the FLOAT domain: bin = floor((score - min) * 2048 / (max - min)) is monotone in the score, and
    // unlike the integer key it is linear across the sign change and across exponents.  The members of one float bin
    // are a contiguous key interval, so deeper passes continue on integer keys.  Only when the key range spans the
    // sign change or several exponents (>= 2^25 key steps): a narrow range is linear enough in the integer key.
    bool fpass = (kmax - kmin >= (1u << 25) || rn > 0) && isfinite(fscale) && fscale > 0.f;
#pragma unroll 1
    while (true) {
      for (int b = tid; b < kBins; b += THREADS) sc.hist[b] = 0;
      select_sync<THREADS, BAR>();
      for (int j = tid; j < n_pages; j += THREADS) {
        const uint32_t key = keys[j];
        if (key != kForcedKey && key >= lo && (uint64_t)(key - lo) < width)
          atomicAdd(&sc.hist[fpass ? fbin(key) : (int)((key - lo) >> shift)], 1);
      }
      select_sync<THREADS, BAR>();
      // threshold bin: the highest b with  #keys in bins > b  <  need  <=  #keys in bins >= b
      int h[BPT], mine = 0;
#pragma unroll
      for (int e = 0; e < BPT; ++e) { h[e] = sc.hist[tid * BPT + e]; mine += h[e]; }
      int inc = mine;                           // inclusive suffix sum over threads (tid' >= tid)
#pragma unroll
      for (int o = 1; o < kWarp; o <<= 1) {
        const int a = __shfl_down_sync(0xffffffffu, inc, o);
        if (lane + o < kWarp) inc += a;
      }
      if (lane == 0) sc.wsum[warp] = inc;
      select_sync<THREADS, BAR>();
      int run = inc - mine;                     // keys in bins owned by higher threads
#pragma unroll
      for (int w = 0; w < WARPS; ++w) run += (w > warp) ? sc.wsum[w] : 0;
#pragma unroll
      for (int e = BPT - 1; e >= 0; --e) {
        if (run < need && run + h[e] >= need) { sc.bin = tid * BPT + e; sc.above = run; sc.cnt = h[e]; }
        run += h[e];
      }
      if (tid == 0) { sc.nlist = 0; sc.bmin = 0xFFFFFFFFu; sc.bmax = 0u; }
      select_sync<THREADS, BAR>();
      const int bin = sc.bin, cnt = sc.cnt;
      need -= sc.above;                         // still to take from the threshold bin
      const uint32_t bin_lo = lo + ((uint32_t)bin << shift);
      if (!fpass && shift == 0) {               // the bin is one key value: take the first `need` by index
        thr = bin_lo;
        need_eq = need;
        break;
      }
      // members of the threshold bin: rank them if they are few, else continue on their key interval
      const uint64_t bin_w = (uint64_t)1 << shift;
      if constexpr (kApprox) {
        if (need <= tol) {                      // enough high-confidence pages: sample the rest from the bin's members
          early = true;
          fterm = fpass;
          t_bin = bin;
          m_lo = bin_lo;
          m_hi = (uint32_t)min((uint64_t)bin_lo + bin_w - 1, (uint64_t)lo + width - 1);
          need_eq = need;
          uint64_t z = seed + 0x9E3779B97F4A7C15ull * (uint64_t)(problem + 1);   // SplitMix64 draw
          z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
          z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
          z ^= z >> 31;
          rot = (int)((uint32_t)(z >> 32) % (uint32_t)cnt);
          wrap = max(0, rot + need - cnt);      // member ranks [0, wrap) and [rot, rot + need - wrap) are taken
          break;
        }
      }
      for (int j = tid; j < n_pages; j += THREADS) {
        const uint32_t key = keys[j];
        const bool in_range = key != kForcedKey && key >= lo && (uint64_t)(key - lo) < width;
        const bool member = in_range && (fpass ? fbin(key) == bin : (key >= bin_lo && (uint64_t)(key - bin_lo) < bin_w));
        if (member) {
          if (cnt <= kList) sc.list[atomicAdd(&sc.nlist, 1)] = key;
          else if (fpass) { atomicMin(&sc.bmin, key); atomicMax(&sc.bmax, key); }
        }
      }
      select_sync<THREADS, BAR>();
      if (cnt <= kList) {
        for (int t = tid; t < cnt; t += THREADS) {
          const uint32_t mykey = sc.list[t];
          int gt = 0, ge = 0;
          for (int j = 0; j < cnt; ++j) {
            const uint32_t o = sc.list[j];
            gt += o > mykey;
            ge += o >= mykey;
          }
          if (gt < need && need <= ge) { sc.thr = mykey; sc.need_eq = need - gt; }   // same values from every tie
        }
        select_sync<THREADS, BAR>();
        thr = sc.thr;
        need_eq = sc.need_eq;
        break;
      }
      if (fpass) {                              // heavy float bin: its members are exactly the keys in [bmin, bmax]
        lo = sc.bmin;
        width = (uint64_t)(sc.bmax - sc.bmin) + 1;
        shift = max(0, (32 - __clz(sc.bmax - sc.bmin)) - kBinBits);
        fpass = false;
      } else {                                  // heavy ties: recurse into the bin, 11 more bits, never past the live window
        width = min(bin_w, (uint64_t)lo + width - bin_lo);
        lo = bin_lo;
        shift = max(0, shift - kBinBits);
      }
      select_sync<THREADS, BAR>();                          // bmin / bmax / bin are read before the next pass rewrites them
    }
  }

  // ---- ordered emission: warp w owns a contiguous run of pages, 32 at a time ------------------
  // class of a page: sure (forced or key > thr) / tie (key == thr, the first need_eq by index are taken)
  const int per_warp = ((n_pages + WARPS - 1) / WARPS + kWarp - 1) / kWarp * kWarp;
  const int j_begin = min(warp * per_warp, n_pages), j_end = min(j_begin + per_warp, n_pages);
  int n_sure = 0, n_tie = 0;                    // warp-uniform
  // class of a key: exact threshold key; (early stop) the key interval of the threshold bin; (early stop on the float pass) its float bin
  auto classify = [&](uint32_t key, bool exists, bool& sure, bool& tie) {
    const bool forced = key == kForcedKey;
    if (!kApprox || !early) {
      sure = exists && (forced || key > thr);
      tie = exists && !forced && key == thr;
    } else if (!fterm) {
      sure = exists && (forced || key > m_hi);
      tie = exists && !forced && key >= m_lo && key <= m_hi;
    } else {
      const int fb = forced ? kBins : fbin(key);
      sure = exists && fb > t_bin;
      tie = exists && fb == t_bin;
    }
  };
  for (int base = j_begin; base < j_end; base += kWarp) {
    const int j = base + lane;
    const uint32_t key = j < j_end ? keys[j] : 0u;
    bool sure, tie;
    classify(key, j < j_end, sure, tie);
    n_sure += __popc(__ballot_sync(0xffffffffu, sure));
    n_tie += __popc(__ballot_sync(0xffffffffu, tie));
  }
  if (lane == 0) sc.wcnt[warp] = make_int2(n_sure, n_tie);
  select_sync<THREADS, BAR>();
  int gt = 0, eq = 0;                           // sure / tie pages before this warp's run
#pragma unroll
  for (int w = 0; w < WARPS; ++w) {
    const int2 c = sc.wcnt[w];
    gt += (w < warp) ? c.x : 0;
    eq += (w < warp) ? c.y : 0;
  }
  const unsigned lt_mask = (1u << lane) - 1u;
  for (int base = j_begin; base < j_end; base += kWarp) {
    const int j = base + lane;
    const uint32_t key = j < j_end ? keys[j] : 0u;
    bool sure, tie;
    classify(key, j < j_end, sure, tie);
    const unsigned b_sure = __ballot_sync(0xffffffffu, sure), b_tie = __ballot_sync(0xffffffffu, tie);
    const int my_gt = gt + __popc(b_sure & lt_mask), my_eq = eq + __popc(b_tie & lt_mask);
    bool take;
    int pos;
    if (kApprox && early) {                       // ranks [0, wrap) and [rot, rot + need_eq - wrap)
      const int span = need_eq - wrap;
      take = sure || (tie && (my_eq < wrap || (my_eq >= rot && my_eq < rot + span)));
      pos = my_gt + min(my_eq, wrap) + min(max(my_eq - rot, 0), span);
    } else {
      take = sure || (tie && my_eq < need_eq);
      pos = my_gt + min(my_eq, need_eq);
    }
    if (take && pos < n_sel) sc.hist[pos] = j;    // (the histogram is free now)
    gt += __popc(b_sure);
    eq += __popc(b_tie);
  }
  select_sync<THREADS, BAR>();
  return n_sel;
}

}  // namespace vx
