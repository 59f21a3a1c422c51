// vx_summary.cu -- (a1) page summaries: channel-wise min / max of the keys of a page (Quest envelope),
// or their mean rounded once to the KV dtype (block top-k centroid, Eq.1).
// PAPER.md:546 "feature-wise key envelope k_j^max, k_j^min"; :89 query-independent; :529 per block.
//
// HBM-bound streaming kernel.  One thread owns one 16-byte channel vector of one (page, KV head)
// and walks the page's valid tokens; consecutive threads own consecutive vectors, so a warp
// reads whole contiguous rows (256 B per token row at d=128 bf16).  Algorithmic bytes per
// (page, head): valid_tokens*d*esz read + 2*d*esz written.
#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

template <typename T, int UNROLL, int KIND>
__global__ void __launch_bounds__(256)
summary_kernel(const T* __restrict__ k, int64_t stride_page, int64_t stride_token, int64_t stride_head,
               int num_kv_heads, int qk_dim, int page_size, int batch,
               const int32_t* __restrict__ page_indptr, const int32_t* __restrict__ page_indices,
               const int32_t* __restrict__ seq_lens, const int32_t* __restrict__ first_new_pos,
               int append_only, int64_t num_slots, T* __restrict__ summary, int bpp) {
  constexpr int PER = Elem<T>::kPerVec;
  const int nvec = qk_dim / PER;
  const int64_t items = num_slots * num_kv_heads * nvec;
  for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < items;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int v = (int)(idx % nvec);
    const int h = (int)((idx / nvec) % num_kv_heads);
    const int64_t slot = idx / ((int64_t)nvec * num_kv_heads);
    int i, j;
    if (append_only) {            // one page per request: the page holding the newest token
      i = (int)slot;
      j = (seq_lens[i] - 1) / page_size;
    } else {                      // slot = flat index into page_indices; find its request
      int lo = 0, hi = batch;     // largest i with page_indptr[i] <= slot
      while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (page_indptr[mid] <= slot) lo = mid; else hi = mid;
      }
      i = lo;
      j = (int)(slot - page_indptr[i]);
      if (first_new_pos != nullptr && j < first_new_pos[i] / page_size) continue;
    }
    const int n = seq_lens[i];
    const int n_pages = (n + page_size - 1) / page_size;
    if (j >= n_pages) continue;   // slack entries of an over-allocated table
    const int valid = min(page_size, n - j * page_size);
    const int64_t phys = page_indices[page_indptr[i] + j];
    const T* src = k + pool_block_base(phys, stride_page, bpp, page_size * stride_token) + h * stride_head + (int64_t)v * PER;

    if constexpr (KIND == VX_SUMMARY_CENTROID) {       // mean of the valid keys, one rounding (exact double sums)
      double sum[PER];
#pragma unroll
      for (int e = 0; e < PER; ++e) sum[e] = 0.0;
      int t = 0;
      for (; t + UNROLL <= valid; t += UNROLL) {
        uint4 raw[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) raw[u] = ldg_stream(src + (int64_t)(t + u) * stride_token);
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
          float f[PER];
          Elem<T>::unpack(raw[u], f);
#pragma unroll
          for (int e = 0; e < PER; ++e) sum[e] += (double)f[e];
        }
      }
      for (; t < valid; ++t) {
        float f[PER];
        Elem<T>::unpack(ldg_stream(src + (int64_t)t * stride_token), f);
#pragma unroll
        for (int e = 0; e < PER; ++e) sum[e] += (double)f[e];
      }
      T* dst = summary + (phys * num_kv_heads + h) * (int64_t)qk_dim + (int64_t)v * PER;
      alignas(16) T outv[PER];
#pragma unroll
      for (int e = 0; e < PER; ++e) outv[e] = round_double<T>(sum[e] / (double)valid);
      *reinterpret_cast<uint4*>(dst) = *reinterpret_cast<const uint4*>(outv);
      continue;
    }
    float lo_v[PER], hi_v[PER];
#pragma unroll
    for (int e = 0; e < PER; ++e) { lo_v[e] = INFINITY; hi_v[e] = -INFINITY; }
    int t = 0;
    for (; t + UNROLL <= valid; t += UNROLL) {
      uint4 raw[UNROLL];
#pragma unroll
      for (int u = 0; u < UNROLL; ++u) raw[u] = ldg_stream(src + (int64_t)(t + u) * stride_token);
#pragma unroll
      for (int u = 0; u < UNROLL; ++u) {
        float f[PER];
        Elem<T>::unpack(raw[u], f);
#pragma unroll
        for (int e = 0; e < PER; ++e) { lo_v[e] = fminf(lo_v[e], f[e]); hi_v[e] = fmaxf(hi_v[e], f[e]); }
      }
    }
    for (; t < valid; ++t) {
      float f[PER];
      Elem<T>::unpack(ldg_stream(src + (int64_t)t * stride_token), f);
#pragma unroll
      for (int e = 0; e < PER; ++e) { lo_v[e] = fminf(lo_v[e], f[e]); hi_v[e] = fmaxf(hi_v[e], f[e]); }
    }
    T* dst = summary + ((phys * num_kv_heads + h) * 2) * (int64_t)qk_dim + (int64_t)v * PER;
    alignas(16) T out_lo[PER], out_hi[PER];
#pragma unroll
    for (int e = 0; e < PER; ++e) { out_lo[e] = Elem<T>::from_float(lo_v[e]); out_hi[e] = Elem<T>::from_float(hi_v[e]); }
    *reinterpret_cast<uint4*>(dst) = *reinterpret_cast<const uint4*>(out_lo);
    *reinterpret_cast<uint4*>(dst + qk_dim) = *reinterpret_cast<const uint4*>(out_hi);
  }
}

template <typename T>
static cudaError_t launch_summary_t(vx_ctx* c, const vx_kv_pool& pool, const vx_page_table& pt,
                                    const int32_t* first_new_pos, void* summary, cudaStream_t s) {
  const vx_geom& g = c->g;
  const int append_only = first_new_pos == nullptr;
  const int64_t slots = append_only ? pt.batch : pt.total_pages;
  const int nvec = g.qk_dim / Elem<T>::kPerVec;
  const int64_t items = slots * g.num_kv_heads * nvec;
  if (items == 0) return cudaSuccess;
  const int threads = 256;
  int64_t blocks = (items + threads - 1) / threads;
  const int64_t cap = (int64_t)c->num_sms * 32;       // grid-stride beyond 32 CTAs per SM
  if (blocks > cap) blocks = cap;
  if (g.summary_kind == VX_SUMMARY_CENTROID)
    summary_kernel<T, 8, VX_SUMMARY_CENTROID><<<(unsigned)blocks, threads, 0, s>>>(
        static_cast<const T*>(pool.k), pool.stride_page, pool.stride_token, pool.stride_head,
        g.num_kv_heads, g.qk_dim, g.page_size, pt.batch, pt.page_indptr, pt.page_indices, pt.seq_lens,
        first_new_pos, append_only, slots, static_cast<T*>(summary), c->bpp);
  else
    summary_kernel<T, 8, VX_SUMMARY_ENVELOPE><<<(unsigned)blocks, threads, 0, s>>>(
        static_cast<const T*>(pool.k), pool.stride_page, pool.stride_token, pool.stride_head,
        g.num_kv_heads, g.qk_dim, g.page_size, pt.batch, pt.page_indptr, pt.page_indices, pt.seq_lens,
        first_new_pos, append_only, slots, static_cast<T*>(summary), c->bpp);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_summary_update(vx_ctx* c, const vx_kv_pool& pool, const vx_page_table& pt,
                                  const int32_t* first_new_pos, void* summary, cudaStream_t s) {
  if (c->g.kv_format == VX_KV_FP8_E4M3) return launch_summary_t<fp8_e4m3>(c, pool, pt, first_new_pos, summary, s);
  if (c->g.kv_format == VX_KV_FP8_E5M2) return launch_summary_t<fp8_e5m2>(c, pool, pt, first_new_pos, summary, s);
  if (c->g.dtype == VX_DT_BF16) return launch_summary_t<__nv_bfloat16>(c, pool, pt, first_new_pos, summary, s);
  return launch_summary_t<float>(c, pool, pt, first_new_pos, summary, s);
}

}  // namespace vx
