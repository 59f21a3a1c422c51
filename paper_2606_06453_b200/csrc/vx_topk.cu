// vx_topk.cu -- (a3) exact top-k page selection per (request, KV head).
// PAPER.md:92 Eq.3 (arg-top-k of the block scores), :194 (radix top-k, "highly sensitive to the score
// distribution"), :280 (first block and last blocks always attended; readings G4-G6: the
// budget includes the forced pages, ties go to the lower logical page, k >= P selects everything).
//
// One CTA per (request, KV head).  Scores become order-preserving uint32 keys held in shared memory.
// The select is a radix select made insensitive to the score distribution: the block first reduces
// the min / max key of the non-forced pages and histograms (key - min) >> shift into 2048 bins that
// span exactly that range, so one pass resolves 11 bits of the LIVE range (page scores of one request
// cluster in a few exponent values; a fixed MSB-first digit would spend its first passes on bits that
// are identical for every page).  When the range spans the sign change or several exponents the first
// pass bins in the float domain instead (monotone in the score, linear across exponents), and deeper
// passes continue on the integer keys of the chosen bin.  The bin that holds the k-th key usually has a
// handful of members:
// they are ranked directly (all-pairs count in shared memory); only if it holds more than kList keys
// (heavy ties) the select recurses into that bin, 11 more bits per pass, down to single key values.
// The result is the exact threshold key and how many keys equal to it are taken; the ordered emission
// then resolves ties to the lowest logical index and writes ids in ascending logical order (so the
// partial last page comes last); the selected ids are staged in shared memory and the physical ids
// gathered from the page table in one parallel pass.
// Integer work on a few KB per problem -- latency-bound, not bandwidth-bound.
#include <type_traits>

#include "vx_common.cuh"
#include "vx_internal.h"
#include "vx_select.cuh"

namespace vx {

constexpr int kTopkSmemKeys = 48 * 1024;        // keys cached in shared memory (192 KB); more -> re-read scores

__device__ __forceinline__ uint32_t page_key(const float* __restrict__ sc, int j, int n_pages, int n_sink,
                                             int n_local) {
  return page_forced(j, n_pages, n_sink, n_local) ? kForcedKey : float_to_key(sc[j]);
}

template <int THREADS>
__global__ void __launch_bounds__(THREADS)
topk_kernel(const float* __restrict__ scores, int num_kv_heads, int total_pages,
            const int32_t* __restrict__ page_indptr, const int32_t* __restrict__ page_indices,
            const int32_t* __restrict__ seq_lens, int page_size, const int32_t* __restrict__ budget,
            int n_sink, int n_local, int max_budget, int smem_keys, int32_t* __restrict__ sel_phys,
            int32_t* __restrict__ sel_logical, int32_t* __restrict__ sel_count, int req0, const PrefetchPlan pf,
            const ApproxPlan ap) {
  constexpr int WARPS = THREADS / kWarp;
  constexpr int BPT = kBins / THREADS;          // bins per thread in the suffix scan
  static_assert(kBins % THREADS == 0 && THREADS >= kList, "shape");
  extern __shared__ uint32_t s_keys[];
  __shared__ int s_hist[kBins];
  __shared__ uint32_t s_list[kList];
  __shared__ uint32_t s_wmin[WARPS], s_wmax[WARPS];
  __shared__ int s_wsum[WARPS];
  __shared__ int2 s_wcnt[WARPS];
  __shared__ int s_bin, s_above, s_cnt, s_nlist, s_need_eq;
  __shared__ uint32_t s_thr, s_bmin, s_bmax;

  const int kvh = blockIdx.x, i = blockIdx.y + req0;
  const int tid = threadIdx.x, lane = tid % kWarp, warp = tid / kWarp;
  const int n_pages = (seq_lens[i] + page_size - 1) / page_size;
  const int k = max(0, min(budget[i], max_budget));   // a negative budget selects nothing (never indexes below the row)
  const int row0 = page_indptr[i];
  pdl_wait();                                   // the scores (and, in a step, nothing else) come from the predecessor
  const int64_t out0 = ((int64_t)i * num_kv_heads + kvh) * max_budget;
  const int n_sel = min(k, n_pages);
  if (tid == 0) sel_count[i * num_kv_heads + kvh] = n_sel;

  if (k >= n_pages) {                           // G6: budget covers the request -> every page
    for (int r = tid; r < max_budget; r += THREADS) {
      const bool ok = r < n_pages;
      sel_phys[out0 + r] = ok ? page_indices[row0 + r] : -1;
      if (sel_logical) sel_logical[out0 + r] = ok ? r : -1;
    }
    return;
  }

  const float* sc = scores + (int64_t)kvh * total_pages + row0;
  const bool cached = n_pages <= smem_keys;
  if (cached && n_sel <= kBins) {
    // the usual case: the request's keys fit shared memory -> the CTA-wide selection of vx_select.cuh (the same
    // device function the fused MLA step kernel runs), then the page-table gather as one parallel pass
    __shared__ SelectScratch scratch;
    for (int j0 = tid; j0 < n_pages; j0 += 8 * THREADS) {        // 8 independent loads in flight per thread
      float v[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) v[u] = j0 + u * THREADS < n_pages ? sc[j0 + u * THREADS] : 0.f;
#pragma unroll
      for (int u = 0; u < 8; ++u)
        if (j0 + u * THREADS < n_pages) s_keys[j0 + u * THREADS] = __float_as_uint(v[u]);
    }
    __syncthreads();
    if (ap.active())                            // (requests beyond the register kernel's 8,192 pages)
      cta_select_pages<THREADS, 0, 0, true>(scratch, s_keys, n_pages, k, n_sink, n_local, ap.tolerate_ratio, ap.seed, i * num_kv_heads + kvh,
                                            ap.remap, ap.remap_n);
    else
      cta_select_pages<THREADS>(scratch, s_keys, n_pages, k, n_sink, n_local);
    pdl_trigger();
    const int per_split = (n_sel + pf.splits - 1) / pf.splits;
    for (int r = tid; r < n_sel; r += THREADS) {
      const int j = scratch.hist[r];
      const int phys = page_indices[row0 + j];
      sel_phys[out0 + r] = phys;
      if (sel_logical) sel_logical[out0 + r] = j;
      // the decode kernel starts every split at its first pages: pull those into L2 while HBM is idle
      if (pf.k != nullptr && r % per_split < pf.pages_per_split) {
        const int64_t off = (int64_t)phys * pf.page_bytes + (int64_t)kvh * pf.head_bytes;
        l2_prefetch(static_cast<const uint8_t*>(pf.k) + off, pf.chunk_bytes);
        if (pf.v != nullptr) l2_prefetch(static_cast<const uint8_t*>(pf.v) + off, pf.chunk_bytes);
      }
    }
    for (int r = n_sel + tid; r < max_budget; r += THREADS) {
      sel_phys[out0 + r] = -1;
      if (sel_logical) sel_logical[out0 + r] = -1;
    }
    return;
  }
  // ---- requests beyond the shared-memory key cache, or budgets beyond the staging area: the general form -------
  // keys, and the min / max key of the non-forced pages
  uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
  for (int j0 = tid; j0 < n_pages; j0 += 8 * THREADS) {          // 8 independent loads in flight per thread
    float v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = j0 + u * THREADS < n_pages ? sc[j0 + u * THREADS] : 0.f;
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int j = j0 + u * THREADS;
      if (j < n_pages) {
        const uint32_t key = page_forced(j, n_pages, n_sink, n_local) ? kForcedKey : float_to_key(v[u]);
        if (cached) s_keys[j] = key;
        if (key != kForcedKey) { kmin = min(kmin, key); kmax = max(kmax, key); }
      }
    }
  }
  kmin = __reduce_min_sync(0xffffffffu, kmin);
  kmax = __reduce_max_sync(0xffffffffu, kmax);
  if (lane == 0) { s_wmin[warp] = kmin; s_wmax[warp] = kmax; }
  __syncthreads();
#pragma unroll
  for (int w = 0; w < WARPS; ++w) { kmin = min(kmin, s_wmin[w]); kmax = max(kmax, s_wmax[w]); }
  auto key_at = [&](int j) -> uint32_t {
    return cached ? s_keys[j] : page_key(sc, j, n_pages, n_sink, n_local);
  };

  const int sink = min(n_sink, n_pages), local = min(n_local, n_pages);
  const int n_forced = min(n_pages, sink + local);
  int need = k - n_forced;                      // non-forced pages still to take (precondition: >= 0)
  uint32_t thr = kForcedKey;                    // take keys > thr, and the first need_eq keys == thr
  int need_eq = 0;

  if (need > 0) {
    // ---- radix select over the live key range [lo, lo + width) ----------------------------------
    uint32_t lo = kmin;
    uint64_t width = (uint64_t)(kmax - kmin) + 1;
    int shift = max(0, (32 - __clz(kmax - kmin)) - kBinBits);     // ((kmax - kmin) >> shift) < kBins
    // First pass in the FLOAT domain: bin = floor((score - min) * 2048 / (max - min)) is monotone in the score, and
    // unlike the integer key it is linear across the sign change and across exponents -- a request whose scores
    // straddle zero (centroid scores, bimodal distributions) would otherwise spend its first pass on a few coarse
    // bins.  The members of one float bin are a contiguous key interval, so deeper passes continue on integer keys.
    const float smin = key_to_float(kmin), smax = key_to_float(kmax);
    const float fscale = (float)kBins / (smax - smin);
    // (only when the key range spans the sign change or several exponents -- >= 2^25 key steps; a narrow range is
    //  already linear enough in the integer key and its pass is ~1 us cheaper)
    bool fpass = kmax - kmin >= (1u << 25) && isfinite(fscale) && fscale > 0.f;
    auto fbin = [&](uint32_t key) -> int { return min(kBins - 1, (int)((key_to_float(key) - smin) * fscale)); };
#pragma unroll 1
    while (true) {
      for (int b = tid; b < kBins; b += THREADS) s_hist[b] = 0;
      __syncthreads();
      for (int j = tid; j < n_pages; j += THREADS) {
        const uint32_t key = key_at(j);
        if (key != kForcedKey && key >= lo && (uint64_t)(key - lo) < width) atomicAdd(&s_hist[fpass ? fbin(key) : (int)((key - lo) >> shift)], 1);
      }
      __syncthreads();
      // threshold bin: the highest b with  #keys in bins > b  <  need  <=  #keys in bins >= b
      int h[BPT], mine = 0;
#pragma unroll
      for (int e = 0; e < BPT; ++e) { h[e] = s_hist[tid * BPT + e]; mine += h[e]; }
      int inc = mine;                           // inclusive suffix sum over threads (tid' >= tid)
#pragma unroll
      for (int o = 1; o < kWarp; o <<= 1) {
        const int a = __shfl_down_sync(0xffffffffu, inc, o);
        if (lane + o < kWarp) inc += a;
      }
      if (lane == 0) s_wsum[warp] = inc;
      __syncthreads();
      int run = inc - mine;                     // keys in bins owned by higher threads
#pragma unroll
      for (int w = 0; w < WARPS; ++w) run += (w > warp) ? s_wsum[w] : 0;
#pragma unroll
      for (int e = BPT - 1; e >= 0; --e) {
        if (run < need && run + h[e] >= need) { s_bin = tid * BPT + e; s_above = run; s_cnt = h[e]; }
        run += h[e];
      }
      if (tid == 0) s_nlist = 0;
      __syncthreads();
      const int bin = s_bin, cnt = s_cnt;
      need -= s_above;                          // still to take from the threshold bin
      if (fpass) {                              // float pass: rank the bin's members, or continue on its key interval
        if (tid == 0) { s_bmin = 0xFFFFFFFFu; s_bmax = 0u; }
        __syncthreads();
        for (int j = tid; j < n_pages; j += THREADS) {
          const uint32_t key = key_at(j);
          if (key != kForcedKey && fbin(key) == bin) {
            if (cnt <= kList) s_list[atomicAdd(&s_nlist, 1)] = key;
            else { atomicMin(&s_bmin, key); atomicMax(&s_bmax, key); }
          }
        }
        __syncthreads();
        if (cnt <= kList) {
          if (tid < cnt) {
            const uint32_t mykey = s_list[tid];
            int gt = 0, ge = 0;
            for (int j = 0; j < cnt; ++j) {
              const uint32_t o = s_list[j];
              gt += o > mykey;
              ge += o >= mykey;
            }
            if (gt < need && need <= ge) { s_thr = mykey; s_need_eq = need - gt; }
          }
          __syncthreads();
          thr = s_thr;
          need_eq = s_need_eq;
          break;
        }
        lo = s_bmin;                            // heavy bin: its members are exactly the keys in [bmin, bmax]
        width = (uint64_t)(s_bmax - s_bmin) + 1;
        shift = max(0, (32 - __clz(s_bmax - s_bmin)) - kBinBits);
        fpass = false;
        __syncthreads();
        continue;
      }
      const uint32_t bin_lo = lo + ((uint32_t)bin << shift);
      if (shift == 0) {                         // the bin is one key value: take the first `need` by index
        thr = bin_lo;
        need_eq = need;
        break;
      }
      if (cnt <= kList) {                       // rank the few members of the bin directly
        const uint64_t bin_w = (uint64_t)1 << shift;
        for (int j = tid; j < n_pages; j += THREADS) {
          const uint32_t key = key_at(j);
          if (key != kForcedKey && key >= bin_lo && (uint64_t)(key - bin_lo) < bin_w && (uint64_t)(key - lo) < width)
            s_list[atomicAdd(&s_nlist, 1)] = key;
        }
        __syncthreads();
        if (tid < cnt) {
          const uint32_t mykey = s_list[tid];
          int gt = 0, ge = 0;
          for (int j = 0; j < cnt; ++j) {
            const uint32_t o = s_list[j];
            gt += o > mykey;
            ge += o >= mykey;
          }
          if (gt < need && need <= ge) { s_thr = mykey; s_need_eq = need - gt; }   // same values from every tie
        }
        __syncthreads();
        thr = s_thr;
        need_eq = s_need_eq;
        break;
      }
      // heavy ties: recurse into the bin, 11 more bits.  The window stays inside [lo, lo + width): after a float pass the
      // interval [bmin, bmax] is unaligned, so its last sub-bin ends at bmax, not at bin_lo + 2^shift (keys above bmax
      // belong to a higher float bin and are already counted)
      width = min((uint64_t)1 << shift, (uint64_t)lo + width - bin_lo);
      lo = bin_lo;
      shift = max(0, shift - kBinBits);
    }
  }

  pdl_trigger();
  // ---- ordered emission: warp w owns a contiguous run of pages, 32 at a time ------------------
  // class of a page: sure (forced or key > thr) / tie (key == thr, the first need_eq by index are taken)
  const int per_warp = ((n_pages + WARPS - 1) / WARPS + kWarp - 1) / kWarp * kWarp;
  const int j_begin = min(warp * per_warp, n_pages), j_end = min(j_begin + per_warp, n_pages);
  int n_sure = 0, n_tie = 0;                    // warp-uniform
  for (int base = j_begin; base < j_end; base += kWarp) {
    const int j = base + lane;
    const uint32_t key = j < j_end ? key_at(j) : 0u;
    const bool sure = j < j_end && (key == kForcedKey || key > thr);
    const bool tie = j < j_end && key != kForcedKey && key == thr;
    n_sure += __popc(__ballot_sync(0xffffffffu, sure));
    n_tie += __popc(__ballot_sync(0xffffffffu, tie));
  }
  if (lane == 0) s_wcnt[warp] = make_int2(n_sure, n_tie);
  __syncthreads();
  int gt = 0, eq = 0;                           // sure / tie pages before this warp's run
#pragma unroll
  for (int w = 0; w < WARPS; ++w) {
    const int2 c = s_wcnt[w];
    gt += (w < warp) ? c.x : 0;
    eq += (w < warp) ? c.y : 0;
  }
  const unsigned lt_mask = (1u << lane) - 1u;
  const bool staged = n_sel <= kBins;           // the histogram is free now: stage the selected logical ids in it
  for (int base = j_begin; base < j_end; base += kWarp) {
    const int j = base + lane;
    const uint32_t key = j < j_end ? key_at(j) : 0u;
    const bool sure = j < j_end && (key == kForcedKey || key > thr);
    const bool tie = j < j_end && key != kForcedKey && key == thr;
    const unsigned b_sure = __ballot_sync(0xffffffffu, sure), b_tie = __ballot_sync(0xffffffffu, tie);
    const int my_gt = gt + __popc(b_sure & lt_mask), my_eq = eq + __popc(b_tie & lt_mask);
    const bool take = sure || (tie && my_eq < need_eq);
    const int pos = my_gt + min(my_eq, need_eq);
    if (take && pos < n_sel) {
      if (staged) s_hist[pos] = j;                // logical ids first; the page-table gather runs as one parallel pass
      else {
        sel_phys[out0 + pos] = page_indices[row0 + j];
        if (sel_logical) sel_logical[out0 + pos] = j;
      }
    }
    gt += __popc(b_sure);
    eq += __popc(b_tie);
  }
  if (staged) {                                   // every selected page: one independent gather + two stores
    __syncthreads();
    const int per_split = (n_sel + pf.splits - 1) / pf.splits;
    for (int r = tid; r < n_sel; r += THREADS) {
      const int j = s_hist[r];
      const int phys = page_indices[row0 + j];
      sel_phys[out0 + r] = phys;
      if (sel_logical) sel_logical[out0 + r] = j;
      // the decode kernel starts every split at its first pages: pull those into L2 while HBM is idle
      if (pf.k != nullptr && r % per_split < pf.pages_per_split) {
        const int64_t off = (int64_t)phys * pf.page_bytes + (int64_t)kvh * pf.head_bytes;
        l2_prefetch(static_cast<const uint8_t*>(pf.k) + off, pf.chunk_bytes);
        if (pf.v != nullptr) l2_prefetch(static_cast<const uint8_t*>(pf.v) + off, pf.chunk_bytes);
      }
    }
  }
  for (int r = n_sel + tid; r < max_budget; r += THREADS) {
    sel_phys[out0 + r] = -1;
    if (sel_logical) sel_logical[out0 + r] = -1;
  }
}

template <int THREADS>
static cudaError_t launch_topk_t(vx_ctx* c, const float* scores, const vx_page_table& pt, const int32_t* budget,
                                 int32_t max_budget, int32_t* sel_phys, int32_t* sel_logical, int32_t* sel_count,
                                 cudaStream_t s, bool pdl, const ReqRange& rr, const PrefetchPlan& pf,
                                 const ApproxPlan& ap = ApproxPlan()) {
  const vx_geom& g = c->g;
  const int keys = pt.max_pages_per_req <= kTopkSmemKeys ? pt.max_pages_per_req : 0;
  const size_t smem = (size_t)(keys > 0 ? keys : 1) * sizeof(uint32_t);
  if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(topk_kernel<THREADS>), c->device, kTopkSmemKeys * (int)sizeof(uint32_t))) return e;
  dim3 grid(g.num_kv_heads, rr.count < 0 ? pt.batch : rr.count);
  cudaError_t e = launch_kernel(topk_kernel<THREADS>, grid, dim3(THREADS), smem, s, pdl, scores, g.num_kv_heads,
                                pt.total_pages, pt.page_indptr, pt.page_indices, pt.seq_lens, g.page_size, budget,
                                g.n_sink, g.n_local, max_budget, keys, sel_phys, sel_logical, sel_count, rr.begin, pf, ap);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

// ---- register-resident variant: requests of at most kKpt * THREADS pages ---------------------------------------
// Same algorithm, but every thread keeps its kKpt keys in registers for all passes (no shared-memory key array, no
// re-reads): warp w owns the contiguous run [w * 32 * kKpt, (w+1) * 32 * kKpt) of logical pages, lane-strided inside
// it (coalesced score loads), so the ordered emission is one ballot per 32 pages.  Fewer, cheaper block-wide phases:
// this kernel is latency-bound ("top-k selection becomes a bottleneck").
// kApprox: the stochastic early termination of PAPER.md:196 (G20-G23): once the pages still to
// take from the threshold bin number at most floor(tolerate_ratio * k), they are drawn from the bin's members as a
// random cyclic window in page order instead of refining the bin (no member list, no ranking).
template <int THREADS, int kKpt, bool kApprox>
__global__ void __launch_bounds__(THREADS)
topk_reg_kernel(const float* __restrict__ scores, int num_kv_heads, int total_pages,
                const int32_t* __restrict__ page_indptr, const int32_t* __restrict__ page_indices,
                const int32_t* __restrict__ seq_lens, int page_size, const int32_t* __restrict__ budget,
                int n_sink, int n_local, int max_budget, int32_t* __restrict__ sel_phys,
                int32_t* __restrict__ sel_logical, int32_t* __restrict__ sel_count, int req0, const PrefetchPlan pf,
                const ApproxPlan ap) {
  constexpr int WARPS = THREADS / kWarp;
  constexpr int BPT = kBins / THREADS;          // bins per thread in the suffix scan
  static_assert(kBins % THREADS == 0, "shape");
  __shared__ int s_hist[kBins];
  __shared__ uint32_t s_list[kList];
  __shared__ uint32_t s_wmin[WARPS], s_wmax[WARPS];
  __shared__ int s_wsum[WARPS];
  __shared__ int2 s_wcnt[WARPS];
  __shared__ int s_bin, s_above, s_cnt, s_nlist, s_need_eq;
  __shared__ uint32_t s_thr, s_bmin, s_bmax;
  __shared__ float s_knot[kApprox ? kTopkRemapMaxKnots : 1];      // the remap's knot table (reading G29)

  const int kvh = blockIdx.x, i = blockIdx.y + req0;
  const int tid = threadIdx.x, lane = tid % kWarp, warp = tid / kWarp;
  [[maybe_unused]] const int cta = blockIdx.y * gridDim.x + blockIdx.x;
  const int rn = kApprox ? ap.remap_n : 0;
  if constexpr (kApprox)
    for (int t = tid; t < rn; t += THREADS) s_knot[t] = ap.remap[t];   // (an input of the call: read before the wait)
  if (tid == 0) { VX_TRACE_STAMP(cta, 0); VX_TRACE_SMID(cta); }
  const int n_pages = (seq_lens[i] + page_size - 1) / page_size;
  const int k = max(0, min(budget[i], max_budget));   // a negative budget selects nothing (never indexes below the row)
  const int row0 = page_indptr[i];
  for (int b = tid; b < kBins; b += THREADS) s_hist[b] = 0;      // first pass's histogram, zeroed under the loads
  if (tid == 0) VX_TRACE_STAMP(cta, 1);
  pdl_wait();                                   // the scores (and, in a step, nothing else) come from the predecessor
  if (tid == 0) VX_TRACE_STAMP(cta, 2);
  const int64_t out0 = ((int64_t)i * num_kv_heads + kvh) * max_budget;
  const int n_sel = min(k, n_pages);
  if (tid == 0) sel_count[i * num_kv_heads + kvh] = n_sel;

  if (k >= n_pages) {                           // G6: budget covers the request -> every page
    for (int r = tid; r < max_budget; r += THREADS) {
      const bool ok = r < n_pages;
      sel_phys[out0 + r] = ok ? page_indices[row0 + r] : -1;
      if (sel_logical) sel_logical[out0 + r] = ok ? r : -1;
    }
    return;
  }

  // ---- my keys: logical pages jbase + 32 u + lane ---------------------------------------------------------------
  const float* sc = scores + (int64_t)kvh * total_pages + row0;
  const int jbase = warp * kWarp * kKpt;
  uint32_t key[kKpt];                           // 0 for pages past the request (never forced, never counted: see `live`)
  float v[kKpt];
#pragma unroll
  for (int u = 0; u < kKpt; ++u) {
    const int j = jbase + u * kWarp + lane;
    v[u] = j < n_pages ? sc[j] : 0.f;
  }
  uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
  unsigned live = 0;                            // bit u: my u-th page exists and is not forced
#pragma unroll
  for (int u = 0; u < kKpt; ++u) {
    const int j = jbase + u * kWarp + lane;
    const bool forced = j < n_pages && page_forced(j, n_pages, n_sink, n_local);
    key[u] = forced ? kForcedKey : float_to_key(v[u]);
    if (j < n_pages && !forced) { live |= 1u << u; kmin = min(kmin, key[u]); kmax = max(kmax, key[u]); }
  }
  kmin = __reduce_min_sync(0xffffffffu, kmin);
  kmax = __reduce_max_sync(0xffffffffu, kmax);
  if (lane == 0) { s_wmin[warp] = kmin; s_wmax[warp] = kmax; }
  __syncthreads();
  if (tid == 0) VX_TRACE_STAMP(cta, 3);
#pragma unroll
  for (int w = 0; w < WARPS; ++w) { kmin = min(kmin, s_wmin[w]); kmax = max(kmax, s_wmax[w]); }

  const int sink = min(n_sink, n_pages), local = min(n_local, n_pages);
  const int n_forced = min(n_pages, sink + local);
  int need = k - n_forced;                      // non-forced pages still to take (precondition: >= 0)
  uint32_t thr = kForcedKey;                    // take keys > thr, and the first need_eq keys == thr
  int need_eq = 0;
  // early termination (kApprox): ties = the members of the threshold bin (key interval [m_lo, m_hi], or float bin
  // t_bin), taken as the cyclic window of need_eq member ranks that starts at rot
  bool early = false, fterm = false;
  uint32_t m_lo = 0u, m_hi = 0u;
  int t_bin = 0, rot = 0, wrap = 0;
  const float smin = key_to_float(kmin), smax = key_to_float(kmax);
  const float fscale = (float)kBins / (smax - smin);
  const float tscale = (float)(rn - 1) / (smax - smin);
  // first-pass bin of a key: linear in the score, or (remap installed) through the knot table -- x = the score's place
  // among the knots, u = f there, every product and sum rounded on its own as the oracle does (no fused multiply-add);
  // the min with the upper knot keeps the bin from ever decreasing with the score (reading G29)
  auto fbin = [&](uint32_t kk) -> int {
    const float d0 = key_to_float(kk) - smin;
    if (kApprox && rn > 0) {
      const float x = __fmul_rn(d0, tscale);
      const int i0 = max(0, min(rn - 2, (int)x));      // (>= 0 for every candidate; the emission also asks for absent pages)
      const float k0 = s_knot[i0], k1 = s_knot[i0 + 1];
      const float u = fminf(k1, __fadd_rn(__fmul_rn(__fsub_rn(x, (float)i0), __fsub_rn(k1, k0)), k0));
      return min(kBins - 1, (int)__fmul_rn(u, (float)kBins));
    }
    return min(kBins - 1, (int)(d0 * fscale));
  };

  if (need > 0) {
    uint32_t lo = kmin;
    uint64_t width = (uint64_t)(kmax - kmin) + 1;
    int shift = max(0, (32 - __clz(kmax - kmin)) - kBinBits);     // ((kmax - kmin) >> shift) < kBins
    bool fpass = (kmax - kmin >= (1u << 25) || rn > 0) && isfinite(fscale) && fscale > 0.f;   // float-domain first pass (see topk_kernel)
    [[maybe_unused]] const int tol = kApprox ? (int)(ap.tolerate_ratio * (float)k) : 0;   // floor: both factors >= 0
    bool first = true;
#pragma unroll 1
    while (true) {
      if (!first) {
        for (int b = tid; b < kBins; b += THREADS) s_hist[b] = 0;
        __syncthreads();
      }
      first = false;
#pragma unroll
      for (int u = 0; u < kKpt; ++u)
        if (((live >> u) & 1u) && key[u] >= lo && (uint64_t)(key[u] - lo) < width)
          atomicAdd(&s_hist[fpass ? fbin(key[u]) : (int)((key[u] - lo) >> shift)], 1);
      __syncthreads();
      if (tid == 0) VX_TRACE_STAMP(cta, 4);           // (the last pass's, if the select recurses)
      // threshold bin: the highest b with  #keys in bins > b  <  need  <=  #keys in bins >= b
      int h[BPT], mine = 0;
#pragma unroll
      for (int e = 0; e < BPT; ++e) { h[e] = s_hist[tid * BPT + e]; mine += h[e]; }
      int inc = mine;                           // inclusive suffix sum over threads (tid' >= tid)
#pragma unroll
      for (int o = 1; o < kWarp; o <<= 1) {
        const int a = __shfl_down_sync(0xffffffffu, inc, o);
        if (lane + o < kWarp) inc += a;
      }
      if (lane == 0) s_wsum[warp] = inc;
      __syncthreads();
      int run = inc - mine;                     // keys in bins owned by higher threads
#pragma unroll
      for (int w = 0; w < WARPS; ++w) run += (w > warp) ? s_wsum[w] : 0;
#pragma unroll
      for (int e = BPT - 1; e >= 0; --e) {
        if (run < need && run + h[e] >= need) { s_bin = tid * BPT + e; s_above = run; s_cnt = h[e]; }
        run += h[e];
      }
      if (tid == 0) { s_nlist = 0; s_bmin = 0xFFFFFFFFu; s_bmax = 0u; }
      __syncthreads();
      if (tid == 0) VX_TRACE_STAMP(cta, 5);
      const int bin = s_bin, cnt = s_cnt;
      need -= s_above;                          // still to take from the threshold bin
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
          uint64_t z = ap.seed + 0x9E3779B97F4A7C15ull * (uint64_t)(i * num_kv_heads + kvh + 1);   // SplitMix64 draw
          z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
          z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
          z ^= z >> 31;
          rot = (int)((uint32_t)(z >> 32) % (uint32_t)cnt);
          wrap = max(0, rot + need - cnt);      // member ranks [0, wrap) and [rot, rot + need - wrap) are taken
          break;
        }
      }
#pragma unroll
      for (int u = 0; u < kKpt; ++u) {
        const uint32_t kk = key[u];
        const bool in_range = ((live >> u) & 1u) && kk >= lo && (uint64_t)(kk - lo) < width;
        const bool member = in_range && (fpass ? fbin(kk) == bin : (kk >= bin_lo && (uint64_t)(kk - bin_lo) < bin_w));
        if (member) {
          if (cnt <= kList) s_list[atomicAdd(&s_nlist, 1)] = kk;
          else if (fpass) { atomicMin(&s_bmin, kk); atomicMax(&s_bmax, kk); }
        }
      }
      __syncthreads();
      if (cnt <= kList) {
        for (int m = tid; m < cnt; m += THREADS) {
          const uint32_t mykey = s_list[m];
          int gt = 0, ge = 0;
          for (int j = 0; j < cnt; ++j) {
            const uint32_t o = s_list[j];
            gt += o > mykey;
            ge += o >= mykey;
          }
          if (gt < need && need <= ge) { s_thr = mykey; s_need_eq = need - gt; }   // same values from every tie
        }
        __syncthreads();
        thr = s_thr;
        need_eq = s_need_eq;
        break;
      }
      if (fpass) {                              // heavy float bin: its members are exactly the keys in [bmin, bmax]
        lo = s_bmin;
        width = (uint64_t)(s_bmax - s_bmin) + 1;
        shift = max(0, (32 - __clz(s_bmax - s_bmin)) - kBinBits);
        fpass = false;
      } else {                                  // heavy ties: recurse into the bin, 11 more bits
        width = min(bin_w, (uint64_t)lo + width - bin_lo);   // never past the live window (unaligned after a float pass)
        lo = bin_lo;
        shift = max(0, shift - kBinBits);
      }
      __syncthreads();                          // s_bmin / s_bmax / s_bin are read before the next pass rewrites them
    }
  }

  if (tid == 0) VX_TRACE_STAMP(cta, 6);
  pdl_trigger();
  // ---- ordered emission: class of a page = sure (forced or key > thr) / tie (key == thr, first need_eq by index) --
  unsigned m_sure[kKpt], m_tie[kKpt];
  int n_sure = 0, n_tie = 0;                    // warp-uniform
  // (the three rules are separate warp-uniform code paths: with 32 warps per SM every predicated-off instruction of
  //  an unused rule would still cost an issue slot per warp)
  auto classify = [&](auto rule) {                // rule 0: exact threshold key; 1: key interval of the bin; 2: float bin
#pragma unroll
    for (int u = 0; u < kKpt; ++u) {
      const bool exists = jbase + u * kWarp + lane < n_pages;
      const bool forced = key[u] == kForcedKey;
      bool sure, tie;
      if constexpr (decltype(rule)::value == 0) {
        sure = exists && (forced || key[u] > thr);
        tie = exists && !forced && key[u] == thr;
      } else if constexpr (decltype(rule)::value == 1) {
        sure = exists && (forced || key[u] > m_hi);
        tie = exists && !forced && key[u] >= m_lo && key[u] <= m_hi;
      } else {
        const int fb = forced ? kBins : fbin(key[u]);
        sure = exists && fb > t_bin;
        tie = exists && fb == t_bin;
      }
      m_sure[u] = __ballot_sync(0xffffffffu, sure);
      m_tie[u] = __ballot_sync(0xffffffffu, tie);
      n_sure += __popc(m_sure[u]);
      n_tie += __popc(m_tie[u]);
    }
  };
  if (!kApprox || !early) classify(std::integral_constant<int, 0>());
  else if (!fterm) classify(std::integral_constant<int, 1>());
  else classify(std::integral_constant<int, 2>());
  if (lane == 0) s_wcnt[warp] = make_int2(n_sure, n_tie);
  __syncthreads();
  if (tid == 0) VX_TRACE_STAMP(cta, 7);
  int gt = 0, eq = 0;                           // sure / tie pages before this warp's run
#pragma unroll
  for (int w = 0; w < WARPS; ++w) {
    const int2 c = s_wcnt[w];
    gt += (w < warp) ? c.x : 0;
    eq += (w < warp) ? c.y : 0;
  }
  const unsigned lt_mask = (1u << lane) - 1u;
  const bool staged = n_sel <= kBins;           // the histogram is free now: stage the selected logical ids in it
  auto emit = [&](auto rotated) {                 // rotated: the taken ties are a cyclic window of tie ranks
#pragma unroll
    for (int u = 0; u < kKpt; ++u) {
      const int j = jbase + u * kWarp + lane;
      const bool sure = (m_sure[u] >> lane) & 1u, tie = (m_tie[u] >> lane) & 1u;
      const int my_gt = gt + __popc(m_sure[u] & lt_mask), my_eq = eq + __popc(m_tie[u] & lt_mask);
      bool take;
      int pos;
      if constexpr (decltype(rotated)::value) {   // ranks [0, wrap) and [rot, rot + need_eq - wrap)
        const int span = need_eq - wrap;
        take = sure || (tie && (my_eq < wrap || (my_eq >= rot && my_eq < rot + span)));
        pos = my_gt + min(my_eq, wrap) + min(max(my_eq - rot, 0), span);
      } else {
        take = sure || (tie && my_eq < need_eq);
        pos = my_gt + min(my_eq, need_eq);
      }
      if (take && pos < n_sel) {
        if (staged) s_hist[pos] = j;
        else {
          sel_phys[out0 + pos] = page_indices[row0 + j];
          if (sel_logical) sel_logical[out0 + pos] = j;
        }
      }
      gt += __popc(m_sure[u]);
      eq += __popc(m_tie[u]);
    }
  };
  if (kApprox && early) emit(std::true_type());
  else emit(std::false_type());
  if (staged) {                                   // every selected page: one independent gather + two stores
    __syncthreads();
    if (tid == 0) VX_TRACE_STAMP(cta, 8);
    const int per_split = (n_sel + pf.splits - 1) / pf.splits;
    for (int r = tid; r < n_sel; r += THREADS) {
      const int j = s_hist[r];
      const int phys = page_indices[row0 + j];
      sel_phys[out0 + r] = phys;
      if (sel_logical) sel_logical[out0 + r] = j;
      if (pf.k != nullptr && r % per_split < pf.pages_per_split) {
        const int64_t off = (int64_t)phys * pf.page_bytes + (int64_t)kvh * pf.head_bytes;
        l2_prefetch(static_cast<const uint8_t*>(pf.k) + off, pf.chunk_bytes);
        if (pf.v != nullptr) l2_prefetch(static_cast<const uint8_t*>(pf.v) + off, pf.chunk_bytes);
      }
    }
  }
  for (int r = n_sel + tid; r < max_budget; r += THREADS) {
    sel_phys[out0 + r] = -1;
    if (sel_logical) sel_logical[out0 + r] = -1;
  }
  if (tid == 0) VX_TRACE_STAMP(cta, 9);
}

VX_TRACE_SETTER(vx_trace_set_topk)

template <int THREADS, int kKpt>
static cudaError_t launch_topk_reg(vx_ctx* c, const float* scores, const vx_page_table& pt, const int32_t* budget,
                                   int32_t max_budget, int32_t* sel_phys, int32_t* sel_logical, int32_t* sel_count,
                                   cudaStream_t s, bool pdl, const ReqRange& rr, const PrefetchPlan& pf,
                                   const ApproxPlan& ap) {
  const vx_geom& g = c->g;
  dim3 grid(g.num_kv_heads, rr.count < 0 ? pt.batch : rr.count);
  auto kernel = ap.active() ? topk_reg_kernel<THREADS, kKpt, true> : topk_reg_kernel<THREADS, kKpt, false>;
  cudaError_t e = launch_kernel(kernel, grid, dim3(THREADS), 0, s, pdl, scores, g.num_kv_heads,
                                pt.total_pages, pt.page_indptr, pt.page_indices, pt.seq_lens, g.page_size, budget,
                                g.n_sink, g.n_local, max_budget, sel_phys, sel_logical, sel_count, rr.begin, pf, ap);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_topk_pages(vx_ctx* c, const float* scores, const vx_page_table& pt,
                              const int32_t* budget, int32_t max_budget, int32_t* sel_phys,
                              int32_t* sel_logical, int32_t* sel_count, cudaStream_t s, bool pdl, const ReqRange& rr,
                              const PrefetchPlan& pf, const ApproxPlan& ap) {
  if (pt.batch == 0) return cudaSuccess;
  // the lossy selection runs in the register kernel (<= 8,192 pages) and in the shared-memory-key kernel (<= 49,152 pages,
  // budgets of at most 2,048 pages)
  static_assert(kTopkApproxMaxPages == kTopkSmemKeys && kTopkApproxMaxBudgetLong == kBins, "vx_internal.h states the kernel's limits");
  if (ap.active() && !approx_topk_supported(pt.max_pages_per_req, max_budget)) return cudaErrorNotSupported;
  // block size by problem size
  const int n = pt.max_pages_per_req;
  if (!ap.active() && topk_pair_applies(c, c->g.num_kv_heads * (rr.count < 0 ? pt.batch : rr.count), n))
    return launch_topk_pair(c, scores, pt, budget, max_budget, sel_phys, sel_logical, sel_count, s, pdl, rr, pf);
  if (n <= kTopkRegMaxPages) {                   // keys fit the registers of one CTA
#define VX_REG(T, K) return launch_topk_reg<T, K>(c, scores, pt, budget, max_budget, sel_phys, sel_logical, sel_count, s, pdl, rr, pf, ap)
    // short requests: 4 keys per thread on twice the threads (measured: C4 71.5 -> 70.9 us, C2 106.8 -> 106.2 against 8
    // keys per thread; 2 keys on four times the threads and 16 keys per thread were slower)
    if (n <= 1024) VX_REG(256, 4);
    if (n <= 2048) VX_REG(512, 4);
    if (n <= 4096) VX_REG(512, 8);
    VX_REG(1024, 8);
#undef VX_REG
  }
  const int th = n <= 1024 ? 256 : n <= 4096 ? 512 : 1024;
  if (th <= 256) return launch_topk_t<256>(c, scores, pt, budget, max_budget, sel_phys, sel_logical, sel_count, s, pdl, rr, pf, ap);
  if (th <= 512) return launch_topk_t<512>(c, scores, pt, budget, max_budget, sel_phys, sel_logical, sel_count, s, pdl, rr, pf, ap);
  return launch_topk_t<1024>(c, scores, pt, budget, max_budget, sel_phys, sel_logical, sel_count, s, pdl, rr, pf, ap);
}

}  // namespace vx
