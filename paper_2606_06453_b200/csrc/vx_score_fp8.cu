// vx_score_fp8.cu -- (a2) page scores over an fp8 summary pool (PAPER.md:200 / :520 / :525 fp8 KV cache; :552 envelope score,
// :92 group aggregate; readings G25-G27).
//
// With SUM aggregation the envelope score of a page collapses exactly to one dot product per summary row,
//     S[kvh, j] = [Qm | Qp] . [m_j | M_j],   Qp = sum_h max(q_h, 0),  Qm = sum_h min(q_h, 0)
// (vx_score.cu), and the rows here are one-byte codes: 2 d bytes per (page, KV head) -- half the bf16 stream.  The codes
// are decoded to fp32 by the hardware conversion (exact) and k_scale is NOT applied (a positive factor common to all
// pages changes no selection, G27).  HBM-bound streaming kernel, 1 flop per byte plus the conversion:
//   * qvec_fp8_kernel builds [Qm | Qp] per (request, KV head) once into the workspace (fp32);
//   * score_fp8_kernel: persistent CTAs, each a contiguous share of the batch's flat page list; a warp takes whole pages
//     (all KV heads of a page are one contiguous chunk of Hkv * 2 d bytes), two pages in flight, every lane 16-byte
//     loads; the lane's slice of the query vector lives in registers and is reloaded (from L2) only when the warp's
//     pages cross into another request.
#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

// [Qm | Qp] fp32 per (request, KV head): thread = one channel of one (request, KV head)
__global__ void __launch_bounds__(256)
qvec_fp8_kernel(const __nv_bfloat16* __restrict__ q, int batch, int num_q_heads, int num_kv_heads, int d, float* __restrict__ qvec) {
  const int grp = num_q_heads / num_kv_heads;
  const int64_t n = (int64_t)batch * num_kv_heads * d;
  for (int64_t x = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; x < n; x += (int64_t)gridDim.x * blockDim.x) {
    const int c = (int)(x % d);
    const int64_t rk = x / d;                            // request * Hkv + kvh
    const int i = (int)(rk / num_kv_heads), kvh = (int)(rk % num_kv_heads);
    float qp = 0.f, qm = 0.f;
    for (int h = 0; h < grp; ++h) {
      const float v = __bfloat162float(q[((int64_t)i * num_q_heads + kvh * grp + h) * d + c]);
      qp += fmaxf(v, 0.f);
      qm += fminf(v, 0.f);
    }
    qvec[rk * 2 * d + c] = qm;
    qvec[rk * 2 * d + d + c] = qp;
  }
}

// NT16 = 16-byte vectors per lane per page = ceil(Hkv * (2 d / 16) / 32)
template <typename T, int NT16>
__global__ void __launch_bounds__(256)
score_fp8_kernel(const uint8_t* __restrict__ summary, const float* __restrict__ qvec, const int32_t* __restrict__ page_indptr,
                 const int32_t* __restrict__ page_indices, int batch, int total_pages, int num_kv_heads, int d,
                 float* __restrict__ scores) {
  const int lane = threadIdx.x % kWarp, warp = threadIdx.x / kWarp, nwarp = blockDim.x / kWarp;
  const int rowv = 2 * d / 16;                           // vectors per (page, head) row
  const int pagev = num_kv_heads * rowv;                 // vectors per page
  const int64_t page_bytes = (int64_t)pagev * 16;
  const int begin = (int)((int64_t)total_pages * blockIdx.x / gridDim.x);
  const int end = (int)((int64_t)total_pages * (blockIdx.x + 1) / gridDim.x);
  float qreg[NT16][16];
  int cur_req = -1, cur_end = 0;                         // the request whose query vector is in qreg; its last flat page + 1
  auto load_qreg = [&](int flat) {
    int lo = 0, hi = batch;                              // largest r with page_indptr[r] <= flat
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (page_indptr[mid] <= flat) lo = mid; else hi = mid;
    }
    cur_req = lo;
    cur_end = page_indptr[lo + 1];
#pragma unroll
    for (int t = 0; t < NT16; ++t) {
      const int v = lane + t * kWarp;                    // vector v of the page: head v / rowv, channels 16 (v % rowv) ..
      if (v < pagev) {
        const float4* src = reinterpret_cast<const float4*>(qvec + ((int64_t)lo * num_kv_heads + v / rowv) * 2 * d + (v % rowv) * 16);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float4 x = src[e];
          qreg[t][4 * e] = x.x; qreg[t][4 * e + 1] = x.y; qreg[t][4 * e + 2] = x.z; qreg[t][4 * e + 3] = x.w;
        }
      } else {
#pragma unroll
        for (int e = 0; e < 16; ++e) qreg[t][e] = 0.f;
      }
    }
  };
  auto load_page = [&](int flat, uint4 (&v)[NT16]) {
    const uint8_t* src = summary + (int64_t)page_indices[flat] * page_bytes;
#pragma unroll
    for (int t = 0; t < NT16; ++t)
      v[t] = lane + t * kWarp < pagev ? ldg_stream(src + (lane + t * kWarp) * 16) : make_uint4(0, 0, 0, 0);
  };
  auto finish_page = [&](int flat, const uint4 (&v)[NT16]) {
    if (flat >= cur_end || cur_req < 0) load_qreg(flat);         // (warp-uniform)
    float part[NT16];
#pragma unroll
    for (int t = 0; t < NT16; ++t) {
      float f[16];
      Elem<T>::unpack(v[t], f);
      float acc = 0.f;
#pragma unroll
      for (int e = 0; e < 16; ++e) acc = fmaf(qreg[t][e], f[e], acc);
      part[t] = acc;
    }
    if (num_kv_heads == 1) {                             // one (latent) head: the whole page is one row
      float tot = 0.f;
#pragma unroll
      for (int t = 0; t < NT16; ++t) tot += part[t];
      tot = warp_sum(tot);
      if (lane == 0) scores[flat] = tot;
    } else {                                             // rowv in {8, 16, 32}: lanes [k rowv, (k + 1) rowv) hold one head's row
#pragma unroll
      for (int t = 0; t < NT16; ++t) {
        float x = part[t];
        for (int o = min(rowv, kWarp) / 2; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        const int v0 = lane + t * kWarp;
        if (v0 < pagev && v0 % rowv == 0) scores[(int64_t)(v0 / rowv) * total_pages + flat] = x;
      }
    }
  };
  for (int p0 = begin + warp; p0 < end; p0 += 2 * nwarp) {       // two pages in flight per warp
    const int p1 = p0 + nwarp;
    uint4 va[NT16], vb[NT16];
    load_page(p0, va);
    if (p1 < end) load_page(p1, vb);
    finish_page(p0, va);
    if (p1 < end) finish_page(p1, vb);
  }
}

bool fp8_geometry_supported(const vx_geom& g) {
  if (g.dtype != VX_DT_BF16 || g.agg != VX_AGG_SUM || g.summary_kind != VX_SUMMARY_ENVELOPE) return false;
  const int grp = g.num_kv_heads > 0 ? g.num_q_heads / g.num_kv_heads : 0;
  const int rowv = 2 * g.qk_dim / 16;
  if (g.kv_shared)                                       // the MLA latent head
    return g.num_kv_heads == 1 && g.qk_dim == 576 && g.v_dim == 512 && g.num_q_heads <= 32 && g.num_q_heads % 4 == 0;
  if (grp < 1 || grp > 8 || g.qk_dim != g.v_dim || (g.qk_dim != 64 && g.qk_dim != 128)) return false;
  return g.num_kv_heads * rowv <= 4 * kWarp;             // a lane holds at most four 16-byte vectors of a page
}

template <typename T>
static cudaError_t launch_score_fp8_t(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt, float* scores,
                                      cudaStream_t s) {
  const vx_geom& g = c->g;
  const int64_t n = (int64_t)pt.batch * g.num_kv_heads * g.qk_dim;
  int qb = (int)((n + 255) / 256);
  if (qb > c->num_sms * 8) qb = c->num_sms * 8;
  qvec_fp8_kernel<<<qb, 256, 0, s>>>(static_cast<const __nv_bfloat16*>(q), pt.batch, g.num_q_heads, g.num_kv_heads, g.qk_dim,
                                     c->ws.fp8_qvec);
  c->launches += 1;
  if (cudaError_t e = cudaGetLastError()) return e;
  const int pagev = g.num_kv_heads * (2 * g.qk_dim / 16);
  const int nt16 = (pagev + kWarp - 1) / kWarp;
  int grid = c->num_sms * 4;                             // 4 CTAs of 8 warps per SM: 64 pages in flight per SM
  if (grid > pt.total_pages) grid = pt.total_pages;
  const uint8_t* sm = static_cast<const uint8_t*>(summary);
#define VX_GO(N) score_fp8_kernel<T, N><<<grid, 256, 0, s>>>(sm, c->ws.fp8_qvec, pt.page_indptr, pt.page_indices, pt.batch, \
                                                             pt.total_pages, g.num_kv_heads, g.qk_dim, scores)
  switch (nt16) {
    case 1: VX_GO(1); break;
    case 2: VX_GO(2); break;
    case 3: VX_GO(3); break;
    case 4: VX_GO(4); break;
    default: return cudaErrorInvalidValue;
  }
#undef VX_GO
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_score_fp8(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt, float* scores, cudaStream_t s) {
  if (pt.batch == 0 || pt.total_pages == 0) return cudaSuccess;
  return c->g.kv_format == VX_KV_FP8_E4M3 ? launch_score_fp8_t<fp8_e4m3>(c, q, summary, pt, scores, s)
                                           : launch_score_fp8_t<fp8_e5m2>(c, q, summary, pt, scores, s);
}

}  // namespace vx
