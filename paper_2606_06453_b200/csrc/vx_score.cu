// vx_score.cu -- (a2) query-to-page scores from the min/max summaries.
// PAPER.md:552  u[h,j] = sum_c max(q_h[c]*M_j[c], q_h[c]*m_j[c]);  :92 / :119 aggregated over the
// query heads of one KV head by SUM (reading G2).
//
// With SUM the per-head maxima collapse exactly (max(q*M, q*m) = max(q,0)*M + min(q,0)*m, M >= m):
//     S[kvh,j] = Qp . M_j + Qm . m_j,   Qp = sum_h max(q_h,0),  Qm = sum_h min(q_h,0)
// so the kernel is one fp32 dot product per summary row: 1 flop per byte, a pure HBM stream
// (2*d*esz bytes per (page, KV head), gathered through the page table in >=512 B rows).
//
// Mapping: a CTA takes PB consecutive logical pages of one request for all KV heads; a warp takes
// one KV head and 32 pages; G lanes share one summary row, each lane reading 16-byte vectors
// l, l+G, .. of the min half and of the max half (128 B contiguous per G=8 lanes per load).
// Qp/Qm live in registers (fp32), page ids are fetched 32 at a time and shuffled out.
#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

constexpr int kScoreThreads = 256;
constexpr int kScorePagesPerWarp = 32;

template <typename T, int D, int G, int PB>
__global__ void __launch_bounds__(kScoreThreads)
score_kernel(const T* __restrict__ q, const T* __restrict__ summary, int num_q_heads, int num_kv_heads,
             const int32_t* __restrict__ page_indptr, const int32_t* __restrict__ page_indices,
             const int32_t* __restrict__ seq_lens, int page_size, int total_pages,
             float* __restrict__ scores) {
  constexpr int PER = Elem<T>::kPerVec;
  constexpr int NVEC = D / PER;                 // 16-byte vectors per half row
  constexpr int NI = (NVEC + G - 1) / G;        // vectors per lane per half row
  constexpr int RW = kWarp / G;                 // summary rows per warp pass
  constexpr int NPASS = kScorePagesPerWarp / RW;
  constexpr int NWARPS = kScoreThreads / kWarp;
  static_assert(D % PER == 0 && kWarp % G == 0 && PB % kScorePagesPerWarp == 0, "shape");

  extern __shared__ float s_q[];                // [Hkv][2][D]: Qm (pairs with min), Qp (pairs with max)
  const int i = blockIdx.y;
  const int n_pages = (seq_lens[i] + page_size - 1) / page_size;
  const int page0 = blockIdx.x * PB;
  if (page0 >= n_pages) return;
  const int grp = num_q_heads / num_kv_heads;

  for (int e = threadIdx.x; e < num_kv_heads * D; e += kScoreThreads) {
    const int kvh = e / D, c = e % D;
    const T* qrow = q + ((int64_t)i * num_q_heads + kvh * grp) * D + c;
    float qp = 0.f, qm = 0.f;
    for (int r = 0; r < grp; ++r) {
      const float x = Elem<T>::to_float(qrow[(int64_t)r * D]);
      qp += fmaxf(x, 0.f);
      qm += fminf(x, 0.f);
    }
    s_q[(kvh * 2 + 0) * D + c] = qm;
    s_q[(kvh * 2 + 1) * D + c] = qp;
  }
  __syncthreads();

  const int warp = threadIdx.x / kWarp, lane = threadIdx.x % kWarp;
  const int sub = lane % G, row_in_pass = lane / G;
  const int row_base = page_indptr[i];
  constexpr int NSUB = PB / kScorePagesPerWarp;
  int cur_kvh = -1;
  float qm[NI][PER], qp[NI][PER];

  for (int u = warp; u < num_kv_heads * NSUB; u += NWARPS) {
    const int kvh = u % num_kv_heads;
    const int p_first = page0 + (u / num_kv_heads) * kScorePagesPerWarp;
    if (p_first >= n_pages) continue;
    if (kvh != cur_kvh) {
      cur_kvh = kvh;
#pragma unroll
      for (int it = 0; it < NI; ++it) {
        const int v = sub + it * G;
#pragma unroll
        for (int e = 0; e < PER; ++e) {
          qm[it][e] = v < NVEC ? s_q[(kvh * 2 + 0) * D + v * PER + e] : 0.f;
          qp[it][e] = v < NVEC ? s_q[(kvh * 2 + 1) * D + v * PER + e] : 0.f;
        }
      }
    }
    const int my_page = p_first + lane;
    const int my_phys = my_page < n_pages ? page_indices[row_base + my_page] : -1;
    float mine = 0.f;
#pragma unroll 2
    for (int pass = 0; pass < NPASS; ++pass) {
      const int phys = __shfl_sync(0xffffffffu, my_phys, pass * RW + row_in_pass);
      float acc = 0.f;
      if (phys >= 0) {
        const T* row = summary + ((int64_t)phys * num_kv_heads + kvh) * 2 * D;
        uint4 lo[NI], hi[NI];
#pragma unroll
        for (int it = 0; it < NI; ++it) {
          const int v = sub + it * G;
          if (NVEC % G == 0 || v < NVEC) {
            lo[it] = ldg_stream(row + v * PER);
            hi[it] = ldg_stream(row + D + v * PER);
          } else {
            lo[it] = make_uint4(0, 0, 0, 0);
            hi[it] = make_uint4(0, 0, 0, 0);
          }
        }
#pragma unroll
        for (int it = 0; it < NI; ++it) {
          float a[PER], b[PER];
          Elem<T>::unpack(lo[it], a);
          Elem<T>::unpack(hi[it], b);
#pragma unroll
          for (int e = 0; e < PER; ++e) acc = fmaf(qm[it][e], a[e], fmaf(qp[it][e], b[e], acc));
        }
      }
      acc = warp_sum<G>(acc);                    // every lane of the row's group holds the row score
      const float s_r = __shfl_sync(0xffffffffu, acc, (lane % RW) * G);
      if (lane / RW == pass) mine = s_r;         // lane r keeps the score of page p_first + r
    }
    if (my_page < n_pages) scores[(int64_t)kvh * total_pages + row_base + my_page] = mine;
  }
}

bool score_geometry_supported(const vx_geom& g) {
  if (g.agg != VX_AGG_SUM) return false;
  if (g.dtype == VX_DT_BF16) return g.qk_dim == 128 || g.qk_dim == 64 || g.qk_dim == 576 || g.qk_dim == 256;
  return g.qk_dim == 64 || g.qk_dim == 128;
}

template <typename T, int D, int G>
static cudaError_t launch_score_t(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt,
                                  float* scores, cudaStream_t s) {
  constexpr int PB = 64;
  const vx_geom& g = c->g;
  dim3 grid((pt.max_pages_per_req + PB - 1) / PB, pt.batch);
  const size_t smem = (size_t)g.num_kv_heads * 2 * D * sizeof(float);
  score_kernel<T, D, G, PB><<<grid, kScoreThreads, smem, s>>>(
      static_cast<const T*>(q), static_cast<const T*>(summary), g.num_q_heads, g.num_kv_heads,
      pt.page_indptr, pt.page_indices, pt.seq_lens, g.page_size, pt.total_pages, scores);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_page_score(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt,
                              float* scores, cudaStream_t s) {
  if (pt.batch == 0 || pt.max_pages_per_req == 0) return cudaSuccess;
  const vx_geom& g = c->g;
  if (g.dtype == VX_DT_BF16) {
    switch (g.qk_dim) {
      case 64: return launch_score_t<__nv_bfloat16, 64, 8>(c, q, summary, pt, scores, s);
      case 128: return launch_score_t<__nv_bfloat16, 128, 8>(c, q, summary, pt, scores, s);
      case 256: return launch_score_t<__nv_bfloat16, 256, 16>(c, q, summary, pt, scores, s);
      case 576: return launch_score_t<__nv_bfloat16, 576, 32>(c, q, summary, pt, scores, s);
    }
  } else {
    switch (g.qk_dim) {
      case 64: return launch_score_t<float, 64, 8>(c, q, summary, pt, scores, s);
      case 128: return launch_score_t<float, 128, 16>(c, q, summary, pt, scores, s);
    }
  }
  return cudaErrorInvalidValue;
}

}  // namespace vx
