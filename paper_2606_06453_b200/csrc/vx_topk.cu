// vx_topk.cu -- (a3) exact top-k page selection per (request, KV head).
// PAPER.md:92 Eq.3 (arg-top-k of the block scores), :194 (radix top-k), :280 (first block and last
// blocks always attended; readings G4-G6: budget includes the forced pages, ties go to the
// lower logical page, k >= P selects everything).
//
// One CTA per (request, KV head).  Scores become order-preserving uint32 keys held in shared memory
// (forced pages get the reserved key 0xFFFFFFFF so they always win); a 4-pass, 8-bit MSB radix
// select finds the k-th largest key and how many pages equal to it are still needed; a final
// ordered pass emits the selection in ascending logical order (so ties resolve to the lowest
// index and the partial last page comes last) together with the physical page ids.
// Integer work on a few KB per problem -- latency-bound, not bandwidth-bound.
#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

constexpr int kTopkThreads = 512;
constexpr int kTopkWarps = kTopkThreads / kWarp;
constexpr int kTopkSmemKeys = 48 * 1024;        // keys cached in shared memory (192 KB); more -> re-read scores

__device__ __forceinline__ uint32_t page_key(const float* __restrict__ sc, int j, int n_pages, int n_sink,
                                             int n_local) {
  const bool forced = (j < n_sink) || (j >= n_pages - n_local);
  return forced ? 0xFFFFFFFFu : float_to_key(sc[j]);
}

// inclusive block scan of two counters; returns exclusive prefix, totals via smem
__device__ __forceinline__ int2 block_exclusive_scan2(int2 v, int2* s_warp /*[kTopkWarps]*/, int2* total) {
  const int lane = threadIdx.x % kWarp, warp = threadIdx.x / kWarp;
  int2 inc = v;
#pragma unroll
  for (int o = 1; o < kWarp; o <<= 1) {
    const int ax = __shfl_up_sync(0xffffffffu, inc.x, o), ay = __shfl_up_sync(0xffffffffu, inc.y, o);
    if (lane >= o) { inc.x += ax; inc.y += ay; }
  }
  if (lane == kWarp - 1) s_warp[warp] = inc;
  __syncthreads();
  int2 base = make_int2(0, 0), tot = make_int2(0, 0);
  for (int w = 0; w < kTopkWarps; ++w) {
    const int2 t = s_warp[w];
    if (w < warp) { base.x += t.x; base.y += t.y; }
    tot.x += t.x; tot.y += t.y;
  }
  *total = tot;
  return make_int2(base.x + inc.x - v.x, base.y + inc.y - v.y);
}

__global__ void __launch_bounds__(kTopkThreads)
topk_kernel(const float* __restrict__ scores, int num_kv_heads, int total_pages,
            const int32_t* __restrict__ page_indptr, const int32_t* __restrict__ page_indices,
            const int32_t* __restrict__ seq_lens, int page_size, const int32_t* __restrict__ budget,
            int n_sink, int n_local, int max_budget, int smem_keys, int32_t* __restrict__ sel_phys,
            int32_t* __restrict__ sel_logical, int32_t* __restrict__ sel_count) {
  extern __shared__ uint32_t s_keys[];
  __shared__ int s_hist[256];
  __shared__ int s_suffix[257];
  __shared__ int s_bin, s_need;
  __shared__ int2 s_warp[kTopkWarps];

  const int kvh = blockIdx.x, i = blockIdx.y;
  const int tid = threadIdx.x;
  const int n_pages = (seq_lens[i] + page_size - 1) / page_size;
  const int k = min(budget[i], max_budget);
  const int row0 = page_indptr[i];
  const int64_t out0 = ((int64_t)i * num_kv_heads + kvh) * max_budget;
  const int n_sel = min(k, n_pages);
  if (tid == 0) sel_count[i * num_kv_heads + kvh] = n_sel;

  if (k >= n_pages) {                           // G6: budget covers the request -> every page
    for (int r = tid; r < max_budget; r += kTopkThreads) {
      const bool ok = r < n_pages;
      sel_phys[out0 + r] = ok ? page_indices[row0 + r] : -1;
      if (sel_logical) sel_logical[out0 + r] = ok ? r : -1;
    }
    return;
  }

  const float* sc = scores + (int64_t)kvh * total_pages + row0;
  const bool cached = n_pages <= smem_keys;
  if (cached) {
    for (int j = tid; j < n_pages; j += kTopkThreads) s_keys[j] = page_key(sc, j, n_pages, n_sink, n_local);
  }
  __syncthreads();
  auto key_at = [&](int j) -> uint32_t {
    return cached ? s_keys[j] : page_key(sc, j, n_pages, n_sink, n_local);
  };

  // ---- radix select: find thr = k-th largest key; `need` = how many keys == thr are taken ----
  uint32_t prefix = 0, mask = 0;
  int need = k;
#pragma unroll 1
  for (int shift = 24; shift >= 0; shift -= 8) {
    if (tid < 256) s_hist[tid] = 0;
    __syncthreads();
    for (int j0 = 0; j0 < n_pages; j0 += kTopkThreads) {
      const int j = j0 + tid;
      const bool act = j < n_pages;
      const uint32_t key = act ? key_at(j) : 0u;
      const bool in = act && ((key & mask) == prefix);
      const unsigned bin = (key >> shift) & 255u;
      // warp-aggregated histogram: one atomic per distinct bin per warp (scores are often clustered
      // in a few exponent bins, "highly sensitive to the score distribution")
      const unsigned active = __ballot_sync(0xffffffffu, in);
      if (in) {
        const unsigned peers = __match_any_sync(active, bin);
        if ((tid % kWarp) == __ffs(peers) - 1) atomicAdd(&s_hist[bin], __popc(peers));
      }
    }
    __syncthreads();
    // suffix counts: s_suffix[b] = #keys in bins >= b
    if (tid < 256) s_suffix[tid] = s_hist[tid];
    if (tid == 0) s_suffix[256] = 0;
    __syncthreads();
    for (int o = 1; o < 256; o <<= 1) {
      int add = 0;
      if (tid < 256 && tid + o < 256) add = s_suffix[tid + o];
      __syncthreads();
      if (tid < 256) s_suffix[tid] += add;
      __syncthreads();
    }
    if (tid < 256 && s_suffix[tid] >= need && s_suffix[tid + 1] < need) {
      s_bin = tid;
      s_need = need - s_suffix[tid + 1];
    }
    __syncthreads();
    prefix |= (uint32_t)s_bin << shift;
    mask |= 255u << shift;
    need = s_need;
    __syncthreads();
  }
  const uint32_t thr = prefix;                  // k-th largest key; take all > thr and the first `need` == thr

  // ---- ordered emission ------------------------------------------------------------------
  const int per = (n_pages + kTopkThreads - 1) / kTopkThreads;
  const int j_begin = min(tid * per, n_pages), j_end = min(j_begin + per, n_pages);
  int2 cnt = make_int2(0, 0);                   // x: keys > thr, y: keys == thr in my chunk
  for (int j = j_begin; j < j_end; ++j) {
    const uint32_t key = key_at(j);
    cnt.x += key > thr;
    cnt.y += key == thr;
  }
  int2 total;
  const int2 before = block_exclusive_scan2(cnt, s_warp, &total);
  int gt = before.x, eq = before.y;
  for (int j = j_begin; j < j_end; ++j) {
    const uint32_t key = key_at(j);
    const bool take = key > thr || (key == thr && eq < need);
    if (take) {
      const int pos = gt + min(eq, need);
      sel_phys[out0 + pos] = page_indices[row0 + j];
      if (sel_logical) sel_logical[out0 + pos] = j;
    }
    gt += key > thr;
    eq += key == thr;
  }
  for (int r = n_sel + tid; r < max_budget; r += kTopkThreads) {
    sel_phys[out0 + r] = -1;
    if (sel_logical) sel_logical[out0 + r] = -1;
  }
}

cudaError_t launch_topk_pages(vx_ctx* c, const float* scores, const vx_page_table& pt,
                              const int32_t* budget, int32_t max_budget, int32_t* sel_phys,
                              int32_t* sel_logical, int32_t* sel_count, cudaStream_t s) {
  if (pt.batch == 0) return cudaSuccess;
  const vx_geom& g = c->g;
  const int keys = pt.max_pages_per_req <= kTopkSmemKeys ? pt.max_pages_per_req : 0;
  const size_t smem = (size_t)(keys > 0 ? keys : 1) * sizeof(uint32_t);
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         kTopkSmemKeys * (int)sizeof(uint32_t));
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  dim3 grid(g.num_kv_heads, pt.batch);
  topk_kernel<<<grid, kTopkThreads, smem, s>>>(scores, g.num_kv_heads, pt.total_pages, pt.page_indptr,
                                               pt.page_indices, pt.seq_lens, g.page_size, budget,
                                               g.n_sink, g.n_local, max_budget, keys, sel_phys,
                                               sel_logical, sel_count);
  c->launches += 1;
  return cudaGetLastError();
}

}  // namespace vx
