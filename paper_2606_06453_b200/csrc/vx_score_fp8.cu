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
  pdl_trigger();                                       // the score kernel may start streaming summaries under me
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

// NT16 = 16-byte vectors per lane per page = ceil(Hkv * (2 d / 16) / 32).  Every warp streams its own pages (begin + warp,
// + 8, ..) through a private ring of STAGES page slots filled by 16-byte cp.async copies -- the bytes in flight cost
// shared memory, not registers -- with the page ids fetched 32 at a time (one coalesced load per warp).
constexpr int kS8Warps = 8, kS8Stages = 4;
template <typename T, int NT16>
__global__ void __launch_bounds__(kS8Warps * kWarp, 3)
score_fp8_kernel(const uint8_t* __restrict__ summary, const float* __restrict__ qvec, const int32_t* __restrict__ page_indptr,
                 const int32_t* __restrict__ page_indices, int batch, int total_pages, int num_kv_heads, int d,
                 float* __restrict__ scores) {
  extern __shared__ __align__(128) uint8_t s8_smem[];
  const int lane = threadIdx.x % kWarp, warp = threadIdx.x / kWarp;
  const int rowv = 2 * d / 16;                           // vectors per (page, head) row
  const int pagev = num_kv_heads * rowv;                 // vectors per page
  const int64_t page_bytes = (int64_t)pagev * 16;
  constexpr int SLOT = NT16 * kWarp * 16;                // bytes of a page slot
  const int begin = (int)((int64_t)total_pages * blockIdx.x / gridDim.x);
  const int end = (int)((int64_t)total_pages * (blockIdx.x + 1) / gridDim.x);
  const int my_pages = end - begin > warp ? (end - begin - warp + kS8Warps - 1) / kS8Warps : 0;
  uint8_t* ring = s8_smem + (size_t)warp * kS8Stages * SLOT;
  int ids = 0;                                           // lane l: physical id of my (base + l)-th page
  auto fetch_ids = [&](int base) {
    const int p = base + lane;
    if (p < my_pages) ids = page_indices[begin + warp + p * kS8Warps];
  };
  // (no L2 evict-first hint on these copies, unlike the tensor-core kernel below: with the lane predicate on the copy the
  //  hinted form ran into "illegal instruction" on the full-size latent geometry)
  auto issue = [&](int p) {
    const int phys = __shfl_sync(0xffffffffu, ids, p & 31);
    const uint8_t* src = summary + (int64_t)phys * page_bytes + lane * 16;
#pragma unroll
    for (int t = 0; t < NT16; ++t)
      if (lane + t * kWarp < pagev) cp_async16(ring + (size_t)(p % kS8Stages) * SLOT + (lane + t * kWarp) * 16, src + t * kWarp * 16);
  };
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
  fetch_ids(0);
#pragma unroll
  for (int p = 0; p < kS8Stages - 1; ++p) {
    if (p < my_pages) issue(p);
    cp_async_commit();
  }
  for (int p = 0; p < my_pages; ++p) {
    const int flat = begin + warp + p * kS8Warps;
    if (cur_req < 0) pdl_wait();                         // the query vectors come from qvec_fp8_kernel, my predecessor (my copies are already in flight)
    if (flat >= cur_end || cur_req < 0) load_qreg(flat);          // (warp-uniform)
    cp_async_wait<kS8Stages - 2>();                      // page p has landed (this lane's copies; a lane reads only its own)
    float part[NT16];
#pragma unroll
    for (int t = 0; t < NT16; ++t) {
      const uint4 v = lane + t * kWarp < pagev ? *reinterpret_cast<const uint4*>(ring + (size_t)(p % kS8Stages) * SLOT + (lane + t * kWarp) * 16)
                                              : make_uint4(0, 0, 0, 0);
      float f[16];
      Elem<T>::unpack(v, f);
      float acc = 0.f;
#pragma unroll
      for (int e = 0; e < 16; ++e) acc = fmaf(qreg[t][e], f[e], acc);
      part[t] = acc;
    }
    {
      const int nxt = p + kS8Stages - 1;                 // refill the slot page p - 1 used (this lane read it an iteration ago)
      if ((nxt & 31) == 0 && nxt < my_pages) fetch_ids(nxt);
      if (nxt < my_pages) issue(nxt);
      cp_async_commit();
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
  }
  cp_async_wait<0>();
}

// ---- the same scores on the tensor cores, for the GQA geometry the configs use (8 KV heads, d = 128: a page's summary chunk
// is [8 heads][256 B]).  The CUDA-core kernel above is ISSUE-bound on this format (ncu: 67 % issue slots busy at 26 % of
// the DRAM peak -- every byte is an element that costs a conversion and an FMA), so the dot products go to
// mma.m16n8k16: an A tile is 16 rows = 2 pages x 8 heads of one 16-channel chunk (ldmatrix straight from the staged
// codes, widened to f16 by cvt.rn.f16x2.*: 0.5 LDSM + 4 F2FP + 2 HMMA per 256 elements against ~20 instructions), the B
// operand holds the 8 heads' query vectors as the 8 columns, split into an f16 high and low part (q = hi + lo to 2^-22;
// a power-of-two pre-scale keeps it inside the f16 range), and row r reads its score from column r % 8 of fp32 D.
constexpr int kM8Warps = 8, kM8Stages = 3, kM8TileBytes = 2 * 2048;
template <typename T> __device__ __forceinline__ void s8_cvt4(uint32_t four, uint32_t& lo, uint32_t& hi);
template <> __device__ __forceinline__ void s8_cvt4<fp8_e4m3>(uint32_t four, uint32_t& lo, uint32_t& hi) {
  asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %2;\n\tcvt.rn.f16x2.e4m3x2 %0, l;\n\tcvt.rn.f16x2.e4m3x2 %1, h;\n\t}"
      : "=r"(lo), "=r"(hi) : "r"(four));
}
template <> __device__ __forceinline__ void s8_cvt4<fp8_e5m2>(uint32_t four, uint32_t& lo, uint32_t& hi) {
  asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %2;\n\tcvt.rn.f16x2.e5m2x2 %0, l;\n\tcvt.rn.f16x2.e5m2x2 %1, h;\n\t}"
      : "=r"(lo), "=r"(hi) : "r"(four));
}
template <typename T>
__global__ void __launch_bounds__(kM8Warps * kWarp, 2)
score_fp8_mma_kernel(const uint8_t* __restrict__ summary, const float* __restrict__ qvec, const int32_t* __restrict__ page_indptr,
                     const int32_t* __restrict__ page_indices, int batch, int total_pages, float* __restrict__ scores,
                     int stream_once) {
  constexpr int HKV = 8, ROW = 256, PAGEB = HKV * ROW, NCH = ROW / 16;      // 16 chunks of 16 codes per row
  extern __shared__ __align__(128) uint8_t s8_smem[];
  const int lane = threadIdx.x % kWarp, warp = threadIdx.x / kWarp;
  const int g = lane >> 2, j = lane & 3;
  const int begin = (int)((int64_t)total_pages * blockIdx.x / gridDim.x);
  const int end = (int)((int64_t)total_pages * (blockIdx.x + 1) / gridDim.x);
  const int n_tiles = (end - begin + 1) / 2;              // tiles of 2 consecutive flat pages
  const int my_tiles = n_tiles > warp ? (n_tiles - warp + kM8Warps - 1) / kM8Warps : 0;
  auto tile_page0 = [&](int p) -> int { return begin + 2 * (warp + kM8Warps * p); };
  const uint32_t ring = smem_u32(s8_smem) + (uint32_t)warp * kM8Stages * kM8TileBytes;
  const uint64_t stream_pol = l2_stream_policy(stream_once != 0);   // (vx_common.cuh)
  int ids = 0;                                            // lane l: page l % 2 of my (base + l / 2)-th tile
  auto fetch_ids = [&](int base) {
    const int flat = tile_page0(base + (lane >> 1)) + (lane & 1);
    ids = (base + (lane >> 1) < my_tiles && flat < end) ? page_indices[flat] : -1;
  };
  auto issue = [&](int p) {
    const uint32_t dst = ring + (uint32_t)(p % kM8Stages) * kM8TileBytes;
#pragma unroll
    for (int pg = 0; pg < 2; ++pg) {
      const int phys = __shfl_sync(0xffffffffu, ids, 2 * (p & 15) + pg);
      if (phys >= 0) {
        const uint8_t* src = summary + (int64_t)phys * PAGEB;
#pragma unroll
        for (int it = 0; it < 4; ++it) {                  // 128 granules of 16 B per page
          const int x = lane + it * kWarp, head = x >> 4, c = x & 15;
          cp_async16_hint(dst + pg * PAGEB + head * ROW + ((c ^ head) << 4), src + x * 16, stream_pol);
        }
      }
    }
  };
  // B operand: thread (column = head g, j) holds for chunk c the channels 16 c + 4 j .. + 3 of head g's [Qm | Qp]
  uint32_t qh[NCH][2], ql[NCH][2];
  float q_up = 1.f;
  int cur_req = -1, cur_end = 0;
  auto load_qreg = [&](int flat) {
    int lo = 0, hi = batch;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (page_indptr[mid] <= flat) lo = mid; else hi = mid;
    }
    cur_req = lo;
    cur_end = page_indptr[lo + 1];
    const float4* src = reinterpret_cast<const float4*>(qvec + ((int64_t)lo * HKV + g) * ROW) + j;
    float mx = 0.f;
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      const float4 x = src[4 * c];
      mx = fmaxf(fmaxf(mx, fmaxf(fabsf(x.x), fabsf(x.y))), fmaxf(fabsf(x.z), fabsf(x.w)));
    }
    mx = warp_max(mx);
    const int e2 = mx > 16384.f ? ilogbf(mx) - 13 : 0;
    const float down = exp2f((float)-e2);
    q_up = exp2f((float)e2);
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      const float4 x = src[4 * c];
      const float v[4] = {x.x * down, x.y * down, x.z * down, x.w * down};
      __half h[4], l[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        h[e] = __float2half_rn(v[e]);
        l[e] = __float2half_rn(v[e] - __half2float(h[e]));
      }
      qh[c][0] = (uint32_t)__half_as_ushort(h[0]) | ((uint32_t)__half_as_ushort(h[1]) << 16);
      qh[c][1] = (uint32_t)__half_as_ushort(h[2]) | ((uint32_t)__half_as_ushort(h[3]) << 16);
      ql[c][0] = (uint32_t)__half_as_ushort(l[0]) | ((uint32_t)__half_as_ushort(l[1]) << 16);
      ql[c][1] = (uint32_t)__half_as_ushort(l[2]) | ((uint32_t)__half_as_ushort(l[3]) << 16);
    }
  };
  // rows of the A tile: r = lane & 15 -> page r / 8, head r % 8; lanes 16..31 address the odd chunk of a pair
  const uint32_t row_off = (uint32_t)(((lane & 15) >> 3) * PAGEB + (lane & 7) * ROW);
  auto compute = [&](int p, float& s_page0, float& s_page1) {
    const uint32_t slot = ring + (uint32_t)(p % kM8Stages) * kM8TileBytes + row_off;
    float dh[4] = {0.f, 0.f, 0.f, 0.f}, dl[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int cc = 0; cc < NCH / 2; ++cc) {
      uint32_t r[4];
      const int c = 2 * cc + (lane >> 4);
      asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                   : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(slot + (uint32_t)((c ^ (lane & 7)) << 4)));
#pragma unroll
      for (int u = 0; u < 2; ++u) {                       // chunk 2 cc + u: r[2u] = rows 0..7, r[2u + 1] = rows 8..15
        uint32_t a0, a1, a2, a3;
        s8_cvt4<T>(r[2 * u], a0, a2);
        s8_cvt4<T>(r[2 * u + 1], a1, a3);
        asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                     : "+f"(dh[0]), "+f"(dh[1]), "+f"(dh[2]), "+f"(dh[3])
                     : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(qh[2 * cc + u][0]), "r"(qh[2 * cc + u][1]));
        asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                     : "+f"(dl[0]), "+f"(dl[1]), "+f"(dl[2]), "+f"(dl[3])
                     : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(ql[2 * cc + u][0]), "r"(ql[2 * cc + u][1]));
      }
    }
    // D[row][col]: this thread holds rows g, g + 8 x columns 2 j, 2 j + 1; row g / g + 8 = head g wants column g
    const bool odd = g & 1;
    s_page0 = ((odd ? dh[1] : dh[0]) + (odd ? dl[1] : dl[0])) * q_up;
    s_page1 = ((odd ? dh[3] : dh[2]) + (odd ? dl[3] : dl[2])) * q_up;
  };
  fetch_ids(0);
#pragma unroll
  for (int p = 0; p < kM8Stages - 1; ++p) {
    if (p < my_tiles) issue(p);
    cp_async_commit();
  }
  for (int p = 0; p < my_tiles; ++p) {
    const int flat0 = tile_page0(p), flat1 = flat0 + 1;
    if (cur_req < 0) pdl_wait();                          // the query vectors come from qvec_fp8_kernel, my predecessor (my copies are already in flight)
    if (flat0 >= cur_end || cur_req < 0) load_qreg(flat0);         // (warp-uniform)
    cp_async_wait<kM8Stages - 2>();
    __syncwarp();                                         // every lane's copies of tile p have landed
    float s0, s1;
    compute(p, s0, s1);
    const bool mine = j == (g >> 1);                      // the thread that holds column g of rows g, g + 8
    if (mine) scores[(int64_t)g * total_pages + flat0] = s0;
    if (flat1 < end) {
      if (flat1 >= cur_end) {                             // the tile straddles two requests: page 1 again with its own query
        load_qreg(flat1);
        compute(p, s0, s1);
      }
      if (mine) scores[(int64_t)g * total_pages + flat1] = s1;
    }
    __syncwarp();                                         // all lanes are done with tile p's slot group before it is refilled
    {
      const int nxt = p + kM8Stages - 1;
      if ((nxt & 15) == 0 && nxt < my_tiles) fetch_ids(nxt);
      if (nxt < my_tiles) issue(nxt);
      cp_async_commit();
    }
  }
  cp_async_wait<0>();
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
  if (g.num_kv_heads == 8 && g.qk_dim == 128) {         // the tensor-core kernel
    constexpr int smem_bytes = kM8Warps * kM8Stages * kM8TileBytes;
    if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(score_fp8_mma_kernel<T>), c->device, smem_bytes)) return e;
    int grid = c->num_sms * 2;
    if (grid > (pt.total_pages + 1) / 2) grid = (pt.total_pages + 1) / 2;
    cudaError_t e = launch_kernel(score_fp8_mma_kernel<T>, dim3(grid), dim3(kM8Warps * kWarp), (size_t)smem_bytes, s, true,
                                  static_cast<const uint8_t*>(summary), (const float*)c->ws.fp8_qvec, pt.page_indptr, pt.page_indices,
                                  pt.batch, pt.total_pages, scores, l2_stream_once(c, (int64_t)pt.total_pages * 2048) ? 1 : 0);
    c->launches += 1;
    return e != cudaSuccess ? e : cudaGetLastError();
  }
  const int pagev = g.num_kv_heads * (2 * g.qk_dim / 16);
  const int nt16 = (pagev + kWarp - 1) / kWarp;
  int grid = c->num_sms * 3;                             // 3 CTAs of 8 warps per SM, 3 pages in flight per warp
  if (grid > pt.total_pages) grid = pt.total_pages;
  const uint8_t* sm = static_cast<const uint8_t*>(summary);
#define VX_GO(N)                                                                                                            \
  do {                                                                                                                      \
    constexpr int smem_bytes = kS8Warps * kS8Stages * N * kWarp * 16;                                                       \
    if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(score_fp8_kernel<T, N>), c->device, smem_bytes)) return e; \
    if (cudaError_t e = launch_kernel(score_fp8_kernel<T, N>, dim3(grid), dim3(kS8Warps * kWarp), (size_t)smem_bytes, s, true, sm,  \
                                      (const float*)c->ws.fp8_qvec, pt.page_indptr, pt.page_indices, pt.batch, pt.total_pages,    \
                                      g.num_kv_heads, g.qk_dim, scores)) return e;                                                \
  } while (0)
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
