// vx_decode_generic.cu -- (a4) sparse paged decode, generic CUDA-core path, and (a5) LSE combine.
// PAPER.md:92 Eq.4  o = softmax(q K_I^T / sqrt(d)) V_I  over the tokens of the selected pages,
// reached through the sparse block table (:200); :75 Flash-Decoding split + merge.
//
// This is the geometry-agnostic path: fp32 pools (config C1) and any (d, dv, group) the tensor-core
// kernels are not built for.  A warp streams tokens one at a time: the 32 lanes split the channels
// of a K row (coalesced 128-byte loads), dot products for HPW query heads are reduced by shuffles,
// online softmax state and the output accumulators live in registers.  Work is split over
// (request, KV head, page split, token slice); every (split, slice) writes one partial (o, lse)
// that the combine kernel merges.
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

template <typename T> struct Pair;        // per-lane access granularity: 4 bytes
template <> struct Pair<__nv_bfloat16> {
  static constexpr int kElems = 2;
  __device__ __forceinline__ static void load(const __nv_bfloat16* p, float (&f)[2]) {
    const uint32_t w = *reinterpret_cast<const uint32_t*>(p);
    f[0] = __uint_as_float(w << 16);
    f[1] = __uint_as_float(w & 0xffff0000u);
  }
};
template <typename T> struct PairFp8 {       // fp8 KV cache: two one-byte codes per lane access (the same channels as a bf16 pair)
  static constexpr int kElems = 2;
  __device__ __forceinline__ static void load(const T* p, float (&f)[2]) {
    const float2 v = fp8x2_to_float2<T>(*reinterpret_cast<const uint16_t*>(p));
    f[0] = v.x;
    f[1] = v.y;
  }
};
template <> struct Pair<fp8_e4m3> : PairFp8<fp8_e4m3> {};
template <> struct Pair<fp8_e5m2> : PairFp8<fp8_e5m2> {};
template <> struct Pair<float> {
  static constexpr int kElems = 1;
  __device__ __forceinline__ static void load(const float* p, float (&f)[1]) { f[0] = *p; }
};

// block = WH head-groups x WT token slices (warps); HPW query heads per warp
// T = element type of q (and of out, through the combine kernel); TKV = element type of the pools (T, or an fp8 code type:
// then a code stands for k_scale / v_scale times its decoded value, G26)
template <typename T, typename TKV, int D, int DV, int HPW, int WT>
__global__ void __launch_bounds__(256)
decode_generic_kernel(const T* __restrict__ q, const TKV* __restrict__ kpool, const TKV* __restrict__ vpool,
                      int64_t stride_page, int64_t stride_token, int64_t stride_head, int num_q_heads,
                      int num_kv_heads, int page_size, float sm_scale,
                      const int32_t* __restrict__ seq_lens, const int32_t* __restrict__ sel_phys,
                      const int32_t* __restrict__ sel_logical, const int32_t* __restrict__ sel_count,
                      int max_budget, int num_splits, float* __restrict__ part_o,
                      float* __restrict__ part_lse, float k_scale, float v_scale, int bpp) {
  constexpr int E = Pair<T>::kElems;
  static_assert(Pair<TKV>::kElems == E, "q and the pools are read with the same channels per lane");
  sm_scale *= k_scale;                           // logits = sm_scale * q . (k_scale * decode(code))
  constexpr int NK = D / (kWarp * E);            // 4-byte loads per lane per K row
  constexpr int NV = DV / (kWarp * E);
  static_assert(D % (kWarp * E) == 0 && DV % (kWarp * E) == 0, "row width must be a multiple of 128 B / 64 B");

  const int split = blockIdx.x, kvh = blockIdx.y, i = blockIdx.z;
  const int warp = threadIdx.x / kWarp, lane = threadIdx.x % kWarp;
  const int wt = warp % WT, wh = warp / WT;
  const int grp = num_q_heads / num_kv_heads;
  const int h0 = kvh * grp + wh * HPW;           // first query head of this warp
  const int n_heads = min(HPW, grp - wh * HPW);
  const int n_tok = seq_lens[i];
  const int cnt = sel_count[i * num_kv_heads + kvh];
  const int per_split = (cnt + num_splits - 1) / num_splits;
  const int r_begin = min(split * per_split, cnt), r_end = min(r_begin + per_split, cnt);
  const int32_t* phys_list = sel_phys + ((int64_t)i * num_kv_heads + kvh) * max_budget;
  const int32_t* log_list = sel_logical + ((int64_t)i * num_kv_heads + kvh) * max_budget;

  float qr[HPW][NK * E];
#pragma unroll
  for (int h = 0; h < HPW; ++h)
#pragma unroll
    for (int r = 0; r < NK; ++r) {
      float f[E];
      if (h < n_heads) Pair<T>::load(q + ((int64_t)i * num_q_heads + h0 + h) * D + (r * kWarp + lane) * E, f);
#pragma unroll
      for (int e = 0; e < E; ++e) qr[h][r * E + e] = h < n_heads ? f[e] * sm_scale : 0.f;
    }

  float m[HPW], l[HPW], acc[HPW][NV * E];
#pragma unroll
  for (int h = 0; h < HPW; ++h) {
    m[h] = -INFINITY; l[h] = 0.f;
#pragma unroll
    for (int c = 0; c < NV * E; ++c) acc[h][c] = 0.f;
  }

  // tokens of the split, flattened; token slice wt takes tokens wt, wt+WT, ...
  for (int r = r_begin; r < r_end; ++r) {
    const int64_t phys = phys_list[r];
    const int valid = min(page_size, n_tok - log_list[r] * page_size);
    const int64_t pbase = pool_block_base(phys, stride_page, bpp, page_size * stride_token) + kvh * stride_head;
    const TKV* kbase = kpool + pbase;
    const TKV* vbase = vpool + pbase;
    for (int t = wt; t < valid; t += WT) {
      float kf[NK * E];
#pragma unroll
      for (int c = 0; c < NK; ++c) {
        float f[E];
        Pair<TKV>::load(kbase + t * stride_token + (c * kWarp + lane) * E, f);
#pragma unroll
        for (int e = 0; e < E; ++e) kf[c * E + e] = f[e];
      }
      float vf[NV * E];
#pragma unroll
      for (int c = 0; c < NV; ++c) {
        float f[E];
        Pair<TKV>::load(vbase + t * stride_token + (c * kWarp + lane) * E, f);
#pragma unroll
        for (int e = 0; e < E; ++e) vf[c * E + e] = f[e];
      }
#pragma unroll
      for (int h = 0; h < HPW; ++h) {
        float dot = 0.f;
#pragma unroll
        for (int c = 0; c < NK * E; ++c) dot = fmaf(qr[h][c], kf[c], dot);
        dot = warp_sum(dot);
        const float m_new = fmaxf(m[h], dot);
        const float alpha = __expf(m[h] - m_new);   // exp(-inf) = 0 on the first token
        const float p = __expf(dot - m_new);
        l[h] = l[h] * alpha + p;
#pragma unroll
        for (int c = 0; c < NV * E; ++c) acc[h][c] = fmaf(p, vf[c], acc[h][c] * alpha);
        m[h] = m_new;
      }
    }
  }

  const int part = split * WT + wt, n_part = num_splits * WT;
#pragma unroll
  for (int h = 0; h < HPW; ++h) {
    if (h >= n_heads) break;
    const int64_t row = ((int64_t)i * num_q_heads + h0 + h) * n_part + part;
    const float inv = l[h] > 0.f ? v_scale / l[h] : 0.f;
#pragma unroll
    for (int c = 0; c < NV; ++c)
#pragma unroll
      for (int e = 0; e < E; ++e) part_o[row * DV + (c * kWarp + lane) * E + e] = acc[h][c * E + e] * inv;
    if (lane == 0) part_lse[row] = l[h] > 0.f ? m[h] + __logf(l[h]) : -INFINITY;
  }
}

// (a5) combine: lse = log sum_s exp(lse_s); o = sum_s exp(lse_s - lse) o_s.  One CTA per (request, head).
template <typename T>
__global__ void __launch_bounds__(128)
combine_kernel(const float* __restrict__ part_o, const float* __restrict__ part_lse, int n_part, int v_dim,
               T* __restrict__ out, float* __restrict__ lse) {
  const int64_t row = blockIdx.x;
  const float* ls = part_lse + row * n_part;
  float mx = -INFINITY;
  for (int s = 0; s < n_part; ++s) mx = fmaxf(mx, ls[s]);
  float z = 0.f;
  for (int s = 0; s < n_part; ++s) z += mx == -INFINITY ? 0.f : __expf(ls[s] - mx);
  for (int c = threadIdx.x; c < v_dim; c += blockDim.x) {
    float o = 0.f;
    for (int s = 0; s < n_part; ++s) {
      const float w = mx == -INFINITY ? 0.f : __expf(ls[s] - mx);
      if (w != 0.f) o = fmaf(w, part_o[(row * n_part + s) * v_dim + c], o);
    }
    out[row * v_dim + c] = Elem<T>::from_float(z > 0.f ? o / z : 0.f);
  }
  if (threadIdx.x == 0 && lse != nullptr) lse[row] = z > 0.f ? mx + logf(z) : -INFINITY;
}

cudaError_t launch_combine(vx_ctx* c, int32_t batch, int n_part, void* out, float* lse, cudaStream_t s) {
  const vx_geom& g = c->g;
  const unsigned rows = (unsigned)batch * g.num_q_heads;
  if (rows == 0) return cudaSuccess;
  if (g.dtype == VX_DT_BF16)
    combine_kernel<__nv_bfloat16><<<rows, 128, 0, s>>>(c->ws.part_o, c->ws.part_lse, n_part, g.v_dim,
                                                       static_cast<__nv_bfloat16*>(out), lse);
  else
    combine_kernel<float><<<rows, 128, 0, s>>>(c->ws.part_o, c->ws.part_lse, n_part, g.v_dim,
                                               static_cast<float*>(out), lse);
  c->launches += 1;
  return cudaGetLastError();
}

// number of page splits so that the grid covers the SMs a few times over
static int pick_splits(const vx_ctx* c, int batch, int max_budget, int wt, int min_pages_per_split) {
  const int units = batch * c->g.num_kv_heads;
  int s = (c->num_sms * 4 + units - 1) / (units > 0 ? units : 1);
  const int cap_pages = (max_budget + min_pages_per_split - 1) / min_pages_per_split;
  if (s > cap_pages) s = cap_pages;
  if (s > kMaxSplits / wt) s = kMaxSplits / wt;
  return s < 1 ? 1 : s;
}

template <typename T, typename TKV, int D, int DV, int HPW, int WT>
static cudaError_t launch_generic_t(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                    const int32_t* sel_phys, const int32_t* sel_logical,
                                    const int32_t* sel_count, int32_t max_budget, void* out, float* lse,
                                    cudaStream_t s) {
  const vx_geom& g = c->g;
  const int grp = g.num_q_heads / g.num_kv_heads;
  const int wh = (grp + HPW - 1) / HPW;
  const int splits = pick_splits(c, pt.batch, max_budget, WT, 2);
  dim3 grid(splits, g.num_kv_heads, pt.batch);
  const void* v = g.kv_shared ? pool.k : pool.v;
  const bool fp8 = kv_is_fp8(g);
  decode_generic_kernel<T, TKV, D, DV, HPW, WT><<<grid, wh * WT * kWarp, 0, s>>>(
      static_cast<const T*>(q), static_cast<const TKV*>(pool.k), static_cast<const TKV*>(v), pool.stride_page,
      pool.stride_token, pool.stride_head, g.num_q_heads, g.num_kv_heads, g.page_size, g.sm_scale,
      pt.seq_lens, sel_phys, sel_logical, sel_count, max_budget, splits, c->ws.part_o, c->ws.part_lse,
      fp8 ? pool.k_scale : 1.f, fp8 ? (g.kv_shared ? pool.k_scale : pool.v_scale) : 1.f, c->bpp);
  c->launches += 1;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return launch_combine(c, pt.batch, splits * WT, out, lse, s);
}

bool gqa_geometry_supported(const vx_geom& g) {
  const int grp = g.num_kv_heads > 0 ? g.num_q_heads / g.num_kv_heads : 0;
  if (g.kv_shared || grp < 1 || grp > 8 || g.qk_dim != g.v_dim) return false;
  if (g.dtype == VX_DT_F32) return g.qk_dim == 64 || g.qk_dim == 128;
  return g.qk_dim == 64 || g.qk_dim == 128;
}

bool mla_geometry_supported(const vx_geom& g) {
  return g.kv_shared && g.dtype == VX_DT_BF16 && g.num_kv_heads == 1 && g.qk_dim == 576 && g.v_dim == 512 &&
         g.num_q_heads <= 32 && g.num_q_heads % 4 == 0;
}

cudaError_t launch_decode_gqa(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                              const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                              int32_t max_budget, void* out, float* lse, cudaStream_t s, const DecodeOpts& opt) {
  const vx_geom& g = c->g;
  if (gqa_mma_supported(g))
    return launch_decode_gqa_mma(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s, opt);
#define VX_GO(T, D, HPW, WT) \
  return launch_generic_t<T, T, D, D, HPW, WT>(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s)
  if (g.dtype == VX_DT_F32) {
    if (g.qk_dim == 64) VX_GO(float, 64, 8, 4);
    if (g.qk_dim == 128) VX_GO(float, 128, 8, 4);
  } else {
    if (g.qk_dim == 64) VX_GO(__nv_bfloat16, 64, 8, 4);
    if (g.qk_dim == 128) VX_GO(__nv_bfloat16, 128, 8, 4);
  }
#undef VX_GO
  return cudaErrorInvalidValue;
}

cudaError_t launch_decode_mla(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                              const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                              int32_t max_budget, void* out, float* lse, cudaStream_t s, const DecodeOpts& opt) {
  if (mla_tc_supported(c->g))
    return launch_decode_mla_tc(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s, opt);
  // CUDA-core fallback: 32 heads = 8 head-groups of 4 per CTA, one token slice: 8 warps
  return launch_generic_t<__nv_bfloat16, __nv_bfloat16, 576, 512, 4, 1>(c, q, pool, pt, sel_phys, sel_logical, sel_count,
                                                                        max_budget, out, lse, s);
}

// fp8 KV cache (vx_kv_format): the generic kernels with one-byte pool elements converted in registers
template <typename TKV>
static cudaError_t launch_decode_fp8_t(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                       const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                       int32_t max_budget, void* out, float* lse, cudaStream_t s) {
  const vx_geom& g = c->g;
  typedef __nv_bfloat16 B;
  if (g.kv_shared) return launch_generic_t<B, TKV, 576, 512, 4, 1>(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s);
  if (g.qk_dim == 64) return launch_generic_t<B, TKV, 64, 64, 8, 4>(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s);
  if (g.qk_dim == 128) return launch_generic_t<B, TKV, 128, 128, 8, 4>(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s);
  return cudaErrorInvalidValue;
}
cudaError_t launch_decode_fp8(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                              const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                              int32_t max_budget, void* out, float* lse, cudaStream_t s) {
  return c->g.kv_format == VX_KV_FP8_E4M3
             ? launch_decode_fp8_t<fp8_e4m3>(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s)
             : launch_decode_fp8_t<fp8_e5m2>(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s);
}


// ---- vx_sparse_paged_decode_static: (a4)+(a5) with NO allocation and no context ---------------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
// the split-KV partials of decode_generic_kernel / combine_kernel live in the file-scope device array below instead of a
// caller workspace.  Every GPU that loads the library holds the array (kStaticScratchBytes) until the process exits.
// Every call shares it and it keeps the last call's contents; nothing in it has to start at zero (each (split, slice)
// writes its whole partial, weight -inf when empty, before the combine kernel reads it), but two calls that overlap on
// the GPU (different streams) race on it.  Same arithmetic as the generic path of vx_sparse_paged_decode.
constexpr size_t kStaticScratchBytes = (size_t)8 << 20;          // 8 MiB: partial o + partial lse of one call
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kStaticMaxDevices = 64;
static std::mutex g_static_mu;
static void* g_static_ptr[kStaticMaxDevices];                   // device address of the array, per device
static int g_static_sms[kStaticMaxDevices];
static char g_static_err[512] = "";

static vx_status static_fail(vx_status st, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_static_err, sizeof g_static_err, fmt, ap);
  va_end(ap);
  return st;
}

// In host code `g_static_scratch` is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, once per device, with that device current.
static vx_status static_scratch_for_current_device(void** ptr, int* num_sms) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return static_fail(VX_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kStaticMaxDevices) return static_fail(VX_ERR_UNSUPPORTED, "device index %d beyond %d", dev, kStaticMaxDevices);
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (g_static_ptr[dev] == nullptr) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || p == nullptr)
      return static_fail(VX_ERR_CUDA, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return static_fail(VX_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
    g_static_sms[dev] = sms;
    g_static_ptr[dev] = p;
  }
  *ptr = g_static_ptr[dev];
  *num_sms = g_static_sms[dev];
  return VX_OK;
}

template <typename T, int D, int DV, int HPW, int WT>
static vx_status launch_generic_static_t(const vx_geom& g, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                         const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                         int32_t max_budget, void* out, float* lse, cudaStream_t s, void* scratch, int num_sms) {
  const int grp = g.num_q_heads / g.num_kv_heads;
  const int wh = (grp + HPW - 1) / HPW;
  const size_t rows = (size_t)pt.batch * g.num_q_heads;
  const size_t per_part = rows * ((size_t)DV + 1) * 4;           // bytes of partial o + lse per (split, slice)
  // splits: cover the SMs a few times over (as the workspace path), at least 2 pages per split, and within the array
  const int units = pt.batch * g.num_kv_heads;
  int splits = (num_sms * 4 + units - 1) / (units > 0 ? units : 1);
  if (splits > (max_budget + 1) / 2) splits = (max_budget + 1) / 2;
  if (splits > kMaxSplits / WT) splits = kMaxSplits / WT;
  if (splits < 1) splits = 1;
  const size_t fit = kStaticScratchBytes / (per_part * WT + 512);      // (+512: the lse block starts 256-byte aligned)
  if (fit < 1)
    return static_fail(VX_ERR_WORKSPACE, "batch %d x %d query heads x v_dim %d needs %zu bytes of split partials; the static "
                       "scratch of vx_sparse_paged_decode_static holds %zu (use vx_sparse_paged_decode with a workspace)",
                       pt.batch, g.num_q_heads, DV, per_part * WT, kStaticScratchBytes);
  if ((size_t)splits > fit) splits = (int)fit;
  const int n_part = splits * WT;
  float* part_o = static_cast<float*>(scratch);
  const size_t o_bytes = (rows * n_part * DV * 4 + 255) / 256 * 256;
  float* part_lse = reinterpret_cast<float*>(static_cast<unsigned char*>(scratch) + o_bytes);
  dim3 grid(splits, g.num_kv_heads, pt.batch);
  const void* v = g.kv_shared ? pool.k : pool.v;
  decode_generic_kernel<T, T, D, DV, HPW, WT><<<grid, wh * WT * kWarp, 0, s>>>(
      static_cast<const T*>(q), static_cast<const T*>(pool.k), static_cast<const T*>(v), pool.stride_page,
      pool.stride_token, pool.stride_head, g.num_q_heads, g.num_kv_heads, g.page_size, g.sm_scale,
      pt.seq_lens, sel_phys, sel_logical, sel_count, max_budget, splits, part_o, part_lse, 1.f, 1.f, 1);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) {
    combine_kernel<T><<<(unsigned)rows, 128, 0, s>>>(part_o, part_lse, n_part, g.v_dim, static_cast<T*>(out), lse);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) return static_fail(VX_ERR_CUDA, "vx_sparse_paged_decode_static: %s", cudaGetErrorString(e));
  return VX_OK;
}

}  // namespace vx

extern "C" {

size_t vx_static_scratch_bytes(void) { return vx::kStaticScratchBytes; }

const char* vx_static_last_error(void) { return vx::g_static_err; }

vx_status vx_sparse_paged_decode_static(const vx_geom* g, const void* q, const vx_kv_pool* pool, const vx_page_table* pt,
                                        const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                        int32_t max_budget, void* out, float* lse, vx_stream stream) {
  using namespace vx;
  if (!g || !q || !pool || !pool->k || !pt || !sel_phys || !sel_logical || !sel_count || !out)
    return static_fail(VX_ERR_INVALID_ARG, "geom / q / pool / page table / sel_* / out is NULL");
  if (g->num_q_heads <= 0 || g->num_kv_heads <= 0 || g->num_q_heads % g->num_kv_heads != 0 || g->page_size <= 0)
    return static_fail(VX_ERR_INVALID_ARG, "num_q_heads must be a positive multiple of num_kv_heads, page_size positive");
  if (!g->kv_shared && !pool->v) return static_fail(VX_ERR_INVALID_ARG, "kv pool v is NULL");
  if (pt->batch < 0 || (pt->batch > 0 && !pt->seq_lens)) return static_fail(VX_ERR_INVALID_ARG, "bad page table");
  if (max_budget <= 0) return static_fail(VX_ERR_INVALID_ARG, "max_budget must be positive");
  if (g->kv_format != VX_KV_SAME) return static_fail(VX_ERR_UNSUPPORTED, "vx_sparse_paged_decode_static takes pools of geom.dtype only");
  if (g->kv_shared ? !mla_geometry_supported(*g) : !gqa_geometry_supported(*g))
    return static_fail(VX_ERR_UNSUPPORTED, "(dtype, qk_dim, v_dim, heads) not supported by the decode kernels");
  if (pt->batch == 0) return VX_OK;
  void* scratch = nullptr;
  int sms = 0;
  if (vx_status st = static_scratch_for_current_device(&scratch, &sms)) return st;
  cudaStream_t s = (cudaStream_t)stream;
#define VX_GO(T, D, DV, HPW, WT) \
  return launch_generic_static_t<T, D, DV, HPW, WT>(*g, q, *pool, *pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s, scratch, sms)
  if (g->kv_shared) VX_GO(__nv_bfloat16, 576, 512, 4, 1);
  if (g->dtype == VX_DT_F32) {
    if (g->qk_dim == 64) VX_GO(float, 64, 64, 8, 4);
    if (g->qk_dim == 128) VX_GO(float, 128, 128, 8, 4);
  } else {
    if (g->qk_dim == 64) VX_GO(__nv_bfloat16, 64, 64, 8, 4);
    if (g->qk_dim == 128) VX_GO(__nv_bfloat16, 128, 128, 8, 4);
  }
#undef VX_GO
  return static_fail(VX_ERR_UNSUPPORTED, "qk_dim %d not supported", g->qk_dim);
}

}  // extern "C"
