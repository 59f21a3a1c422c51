// vx_topk_pair.cu -- (a3) the exact selection of vx_topk.cu with one (request, KV head) spread over a CLUSTER OF
// TWO CTAs (PAPER.md:92 Eq.3, :194, :280; same readings G4-G6, same result bit for bit).
//
// Why: the selection kernel is issue-bound, not bandwidth-bound -- a long-context batch has few problems (C3: 8
// requests x 8 KV heads = 64 CTAs of 1,024 threads on 148 SMs), every thread carries 8 keys through ~10 block-wide
// phases, and with 32 warps on an SM every instruction costs an issue slot per warp while 84 SMs idle.  Two CTAs of
// half the threads halve the per-SM instruction stream of every per-key phase.  What the pair shares goes through
// distributed shared memory: the warps' min / max keys and emission counts are stored into both CTAs, every
// CTA histograms its own keys and the suffix scan adds the peer's bins read remotely, so each CTA scans the full
// histogram on its own and both reach the same threshold bin without a broadcast (per-key remote increments,
// red.shared::cluster, measured far slower); the threshold bin's few members are
// collected per CTA and the peer's list is appended by reading it remotely.  Cluster barriers replace the block
// barriers at those hand-overs (2 per select pass, 2 per kernel).  CTA 0 owns the lower half of the logical pages, so the
// ascending emission is CTA 0's ids followed by CTA 1's.
#include <type_traits>

#include "vx_common.cuh"
#include "vx_internal.h"
#include "vx_select.cuh"

namespace vx {

template <int THREADS, int kKpt>
__global__ void __launch_bounds__(THREADS)
topk_pair_kernel(const float* __restrict__ scores, int num_kv_heads, int total_pages,
                 const int32_t* __restrict__ page_indptr, const int32_t* __restrict__ page_indices,
                 const int32_t* __restrict__ seq_lens, int page_size, const int32_t* __restrict__ budget,
                 int n_sink, int n_local, int max_budget, int32_t* __restrict__ sel_phys,
                 int32_t* __restrict__ sel_logical, int32_t* __restrict__ sel_count, int req0, const PrefetchPlan pf) {
  constexpr int WARPS = THREADS / kWarp;
  constexpr int GW = 2 * WARPS;                 // warps of the pair, CTA 0's first
  constexpr int BPT = kBins / THREADS;          // bins per thread in the suffix scan
  static_assert(kBins % THREADS == 0, "shape");
  __shared__ int s_hist[kBins];
  __shared__ uint32_t s_list[kList];
  __shared__ uint32_t s_wmin[GW], s_wmax[GW];
  __shared__ int s_wsum[WARPS];
  __shared__ int s_wsure[GW], s_wtie[GW];
  __shared__ int s_bin, s_above, s_cnt, s_nlist, s_need_eq;
  __shared__ uint32_t s_thr, s_bmin, s_bmax;

  const int crank = blockIdx.x & 1, peer = crank ^ 1;           // cluster = (2, 1, 1) along x
  const int kvh = blockIdx.x >> 1, i = blockIdx.y + req0;
  const int tid = threadIdx.x, lane = tid % kWarp, warp = tid / kWarp;
  const int gw = crank * WARPS + warp;
  const int n_pages = (seq_lens[i] + page_size - 1) / page_size;
  const int k = max(0, min(budget[i], max_budget));   // a negative budget selects nothing (never indexes below the row)
  const int row0 = page_indptr[i];
  for (int b = tid; b < kBins; b += THREADS) s_hist[b] = 0;      // first pass's histogram, zeroed under the loads
  pdl_wait();                                   // the scores come from the predecessor
  const int64_t out0 = ((int64_t)i * num_kv_heads + kvh) * max_budget;
  const int n_sel = min(k, n_pages);
  if (tid == 0 && crank == 0) sel_count[i * num_kv_heads + kvh] = n_sel;

  if (k >= n_pages) {                           // G6: budget covers the request -> every page (both CTAs leave)
    if (crank == 0)
      for (int r = tid; r < max_budget; r += THREADS) {
        const bool ok = r < n_pages;
        sel_phys[out0 + r] = ok ? page_indices[row0 + r] : -1;
        if (sel_logical) sel_logical[out0 + r] = ok ? r : -1;
      }
    return;
  }

  // ---- my keys: logical pages jbase + 32 u + lane ---------------------------------------------------------------
  const float* sc = scores + (int64_t)kvh * total_pages + row0;
  const int jbase = gw * kWarp * kKpt;
  uint32_t key[kKpt];
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
  if (lane == 0) {                              // into both CTAs
    s_wmin[gw] = kmin;
    s_wmax[gw] = kmax;
    dsmem_st_u32(dsmem_addr(smem_u32(&s_wmin[gw]), peer), kmin);
    dsmem_st_u32(dsmem_addr(smem_u32(&s_wmax[gw]), peer), kmax);
  }
  cluster_sync();                               // (also: both histograms are zeroed before any remote increment)
#pragma unroll
  for (int w = 0; w < GW; ++w) { kmin = min(kmin, s_wmin[w]); kmax = max(kmax, s_wmax[w]); }

  const int sink = min(n_sink, n_pages), local = min(n_local, n_pages);
  const int n_forced = min(n_pages, sink + local);
  int need = k - n_forced;                      // non-forced pages still to take (precondition: >= 0)
  uint32_t thr = kForcedKey;                    // take keys > thr, and the first need_eq keys == thr
  int need_eq = 0;

  if (need > 0) {
    const uint32_t peer_hist = dsmem_addr(smem_u32(s_hist), peer);
    uint32_t lo = kmin;
    uint64_t width = (uint64_t)(kmax - kmin) + 1;
    int shift = max(0, (32 - __clz(kmax - kmin)) - kBinBits);     // ((kmax - kmin) >> shift) < kBins
    const float smin = key_to_float(kmin), smax = key_to_float(kmax);
    const float fscale = (float)kBins / (smax - smin);
    bool fpass = kmax - kmin >= (1u << 25) && isfinite(fscale) && fscale > 0.f;   // float-domain first pass (see vx_topk.cu)
    auto fbin = [&](uint32_t kk) -> int { return min(kBins - 1, (int)((key_to_float(kk) - smin) * fscale)); };
    bool first = true;
#pragma unroll 1
    while (true) {
      if (!first) {
        for (int b = tid; b < kBins; b += THREADS) s_hist[b] = 0;
        __syncthreads();                        // (the peer read the old histogram before the barrier that followed the member pass)
      }
      first = false;
#pragma unroll
      for (int u = 0; u < kKpt; ++u)
        if (((live >> u) & 1u) && key[u] >= lo && (uint64_t)(key[u] - lo) < width) {
          const int b = fpass ? fbin(key[u]) : (int)((key[u] - lo) >> shift);
          atomicAdd(&s_hist[b], 1);
        }
      cluster_sync();                           // both CTAs' histograms are complete
      // threshold bin: the highest b with  #keys in bins > b  <  need  <=  #keys in bins >= b  (each CTA on its own)
      int h[BPT], mine = 0;
#pragma unroll
      for (int e = 0; e < BPT; ++e) {           // my bins of the pair's histogram = mine + the peer's (read remotely)
        h[e] = s_hist[tid * BPT + e] + (int)dsmem_ld_u32(peer_hist + 4u * (uint32_t)(tid * BPT + e));
        mine += h[e];
      }
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
      const int bin = s_bin, cnt = s_cnt;
      need -= s_above;                          // still to take from the threshold bin
      const uint32_t bin_lo = lo + ((uint32_t)bin << shift);
      if (!fpass && shift == 0) {               // the bin is one key value: take the first `need` by index
        thr = bin_lo;
        need_eq = need;
        break;
      }
      // my members of the threshold bin: listed if the bin is light, else only their key interval
      const uint64_t bin_w = (uint64_t)1 << shift;
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
      cluster_sync();                           // both CTAs' lists / intervals are complete
      if (cnt <= kList) {                       // append the peer's members to mine, rank all of them
        const int n_own = s_nlist;
        const int n_peer = (int)dsmem_ld_u32(dsmem_addr(smem_u32(&s_nlist), peer));
        const uint32_t peer_list = dsmem_addr(smem_u32(s_list), peer);
        for (int m = tid; m < n_peer; m += THREADS) s_list[n_own + m] = dsmem_ld_u32(peer_list + 4u * (uint32_t)m);
        __syncthreads();
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
        break;                                  // (the peer's reads of my list precede its arrival at the next cluster barrier)
      }
      if (fpass) {                              // heavy float bin: its members are exactly the keys in [bmin, bmax]
        const uint32_t bmin = min(s_bmin, dsmem_ld_u32(dsmem_addr(smem_u32(&s_bmin), peer)));
        const uint32_t bmax = max(s_bmax, dsmem_ld_u32(dsmem_addr(smem_u32(&s_bmax), peer)));
        lo = bmin;
        width = (uint64_t)(bmax - bmin) + 1;
        shift = max(0, (32 - __clz(bmax - bmin)) - kBinBits);
        fpass = false;
      } else {                                  // heavy ties: recurse into the bin, 11 more bits
        width = min(bin_w, (uint64_t)lo + width - bin_lo);   // never past the live window (unaligned after a float pass)
        lo = bin_lo;
        shift = max(0, shift - kBinBits);
      }
      // (the next pass starts with a cluster barrier after zeroing: the peer has read my s_bmin / s_bmax by then,
      //  and they are reset only after the barrier that follows the next histogram)
    }
  }

  pdl_trigger();                                // (at kernel entry instead: C3 step +0.8 us -- the early decode CTAs compete)
  // ---- ordered emission: class of a page = sure (forced or key > thr) / tie (key == thr, first need_eq by index) --
  unsigned m_sure[kKpt], m_tie[kKpt];
  int n_sure = 0, n_tie = 0;                    // warp-uniform
#pragma unroll
  for (int u = 0; u < kKpt; ++u) {
    const bool exists = jbase + u * kWarp + lane < n_pages;
    const bool sure = exists && (key[u] == kForcedKey || key[u] > thr);
    const bool tie = exists && key[u] != kForcedKey && key[u] == thr;
    m_sure[u] = __ballot_sync(0xffffffffu, sure);
    m_tie[u] = __ballot_sync(0xffffffffu, tie);
    n_sure += __popc(m_sure[u]);
    n_tie += __popc(m_tie[u]);
  }
  if (lane == 0) {                              // into both CTAs
    s_wsure[gw] = n_sure;
    s_wtie[gw] = n_tie;
    dsmem_st_u32(dsmem_addr(smem_u32(&s_wsure[gw]), peer), (uint32_t)n_sure);
    dsmem_st_u32(dsmem_addr(smem_u32(&s_wtie[gw]), peer), (uint32_t)n_tie);
  }
  cluster_sync();                               // the last remote access of the kernel: either CTA may now finish alone
  int gt = 0, eq = 0;                           // sure / tie pages before this warp's run
  int gt0 = 0, eq0 = 0;                         // ... in CTA 0 altogether
#pragma unroll
  for (int w = 0; w < GW; ++w) {
    const int a = s_wsure[w], b = s_wtie[w];
    gt += (w < gw) ? a : 0;
    eq += (w < gw) ? b : 0;
    gt0 += (w < WARPS) ? a : 0;
    eq0 += (w < WARPS) ? b : 0;
  }
  const int split = min(n_sel, gt0 + min(eq0, need_eq));       // CTA 0 emits positions [0, split), CTA 1 [split, n_sel)
  const int base = crank == 0 ? 0 : split;
  const int count = crank == 0 ? split : n_sel - split;
  const unsigned lt_mask = (1u << lane) - 1u;
  const bool staged = n_sel <= kBins;           // the histogram is free now: stage my selected logical ids in it
#pragma unroll
  for (int u = 0; u < kKpt; ++u) {
    const int j = jbase + u * kWarp + lane;
    const bool sure = (m_sure[u] >> lane) & 1u, tie = (m_tie[u] >> lane) & 1u;
    const int my_gt = gt + __popc(m_sure[u] & lt_mask), my_eq = eq + __popc(m_tie[u] & lt_mask);
    const bool take = sure || (tie && my_eq < need_eq);
    const int pos = my_gt + min(my_eq, need_eq);
    if (take && pos < n_sel) {
      if (staged) s_hist[pos - base] = j;
      else {
        sel_phys[out0 + pos] = page_indices[row0 + j];
        if (sel_logical) sel_logical[out0 + pos] = j;
      }
    }
    gt += __popc(m_sure[u]);
    eq += __popc(m_tie[u]);
  }
  if (staged) {                                   // every selected page: one independent gather + two stores
    __syncthreads();
    const int per_split = (n_sel + pf.splits - 1) / pf.splits;
    for (int r = tid; r < count; r += THREADS) {
      const int j = s_hist[r];
      const int phys = page_indices[row0 + j];
      sel_phys[out0 + base + r] = phys;
      if (sel_logical) sel_logical[out0 + base + r] = j;
      if (pf.k != nullptr && (base + r) % per_split < pf.pages_per_split) {
        const int64_t off = (int64_t)phys * pf.page_bytes + (int64_t)kvh * pf.head_bytes;
        l2_prefetch(static_cast<const uint8_t*>(pf.k) + off, pf.chunk_bytes);
        if (pf.v != nullptr) l2_prefetch(static_cast<const uint8_t*>(pf.v) + off, pf.chunk_bytes);
      }
    }
  }
  if (crank == 1)
    for (int r = n_sel + tid; r < max_budget; r += THREADS) {
      sel_phys[out0 + r] = -1;
      if (sel_logical) sel_logical[out0 + r] = -1;
    }
}

template <int THREADS, int kKpt>
static cudaError_t launch_pair(vx_ctx* c, const float* scores, const vx_page_table& pt, const int32_t* budget,
                               int32_t max_budget, int32_t* sel_phys, int32_t* sel_logical, int32_t* sel_count,
                               cudaStream_t s, bool pdl, const ReqRange& rr, const PrefetchPlan& pf) {
  const vx_geom& g = c->g;
  dim3 grid(2 * g.num_kv_heads, rr.count < 0 ? pt.batch : rr.count);
  cudaError_t e = launch_kernel_cluster(topk_pair_kernel<THREADS, kKpt>, grid, dim3(THREADS), 0, s, pdl, 2, scores,
                                        g.num_kv_heads, pt.total_pages, pt.page_indptr, pt.page_indices, pt.seq_lens,
                                        g.page_size, budget, g.n_sink, g.n_local, max_budget, sel_phys, sel_logical,
                                        sel_count, rr.begin, pf);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

// requests of 2,049 .. 8,192 pages, few enough problems that every pair is resident at once
bool topk_pair_applies(const vx_ctx* c, int n_problems, int max_pages_per_req) {
  return max_pages_per_req > 2048 && max_pages_per_req <= kTopkRegMaxPages && 2 * n_problems <= c->num_sms;
}

cudaError_t launch_topk_pair(vx_ctx* c, const float* scores, const vx_page_table& pt, const int32_t* budget,
                             int32_t max_budget, int32_t* sel_phys, int32_t* sel_logical, int32_t* sel_count,
                             cudaStream_t s, bool pdl, const ReqRange& rr, const PrefetchPlan& pf) {
  // (4 keys per thread on twice the threads, which pays for short requests in topk_reg_kernel, measured worse here:
  //  C3 step 91.1 us against 89.5)
  if (pt.max_pages_per_req <= 4096)
    return launch_pair<256, 8>(c, scores, pt, budget, max_budget, sel_phys, sel_logical, sel_count, s, pdl, rr, pf);
  return launch_pair<512, 8>(c, scores, pt, budget, max_budget, sel_phys, sel_logical, sel_count, s, pdl, rr, pf);
}

}  // namespace vx
