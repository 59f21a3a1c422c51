// vx_common.cuh -- device helpers shared by the sm_100a kernels of libvortex_b200.
// (Not shared with oracle/: the oracle is plain C and includes nothing from here.)
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_fp8.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace vx {

constexpr int kWarp = 32;

// ---- storage element traits: 16-byte vectors of bf16 (8 elems) or fp32 (4 elems) ----------
template <typename T> struct Elem;
template <> struct Elem<__nv_bfloat16> {
  static constexpr int kPerVec = 8;  // elements per 16 B
  // widen the 8 bf16 of a uint4 to fp32 (exact): low half = bits << 16, high half = bits & 0xffff0000
  __device__ __forceinline__ static void unpack(const uint4& v, float (&f)[8]) {
    f[0] = __uint_as_float(v.x << 16); f[1] = __uint_as_float(v.x & 0xffff0000u);
    f[2] = __uint_as_float(v.y << 16); f[3] = __uint_as_float(v.y & 0xffff0000u);
    f[4] = __uint_as_float(v.z << 16); f[5] = __uint_as_float(v.z & 0xffff0000u);
    f[6] = __uint_as_float(v.w << 16); f[7] = __uint_as_float(v.w & 0xffff0000u);
  }
  __device__ __forceinline__ static float to_float(__nv_bfloat16 x) { return __bfloat162float(x); }
  __device__ __forceinline__ static __nv_bfloat16 from_float(float x) { return __float2bfloat16_rn(x); }
};
template <> struct Elem<float> {
  static constexpr int kPerVec = 4;
  __device__ __forceinline__ static void unpack(const uint4& v, float (&f)[4]) {
    f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y);
    f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
  }
  __device__ __forceinline__ static float to_float(float x) { return x; }
  __device__ __forceinline__ static float from_float(float x) { return x; }
};

// fp8 KV cache (include/vortex_b200.h vx_kv_format): one-byte codes, OCP E4M3 / E5M2.
// Decoding goes through the hardware conversion to f16 (cvt.rn.f16x2.e4m3x2 / .e5m2x2: every fp8 value is exact in
// f16), encoding through cvt.rn.satfinite (exact for values that are already representable: min / max of codes).
struct fp8_e4m3 { uint8_t bits; };
struct fp8_e5m2 { uint8_t bits; };
template <typename T> struct Fp8Interp;
template <> struct Fp8Interp<fp8_e4m3> { static constexpr __nv_fp8_interpretation_t kind = __NV_E4M3; };
template <> struct Fp8Interp<fp8_e5m2> { static constexpr __nv_fp8_interpretation_t kind = __NV_E5M2; };
template <typename T> __device__ __forceinline__ float2 fp8x2_to_float2(uint16_t two) {     // low byte = element 0
  const __half2_raw h = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)two, Fp8Interp<T>::kind);
  return __half22float2(*reinterpret_cast<const __half2*>(&h));
}
template <typename T> struct ElemFp8 {
  static constexpr int kPerVec = 16;  // elements per 16 B
  __device__ __forceinline__ static void unpack(const uint4& v, float (&f)[16]) {
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float2 a = fp8x2_to_float2<T>((uint16_t)(w[i] & 0xffffu)), b = fp8x2_to_float2<T>((uint16_t)(w[i] >> 16));
      f[4 * i] = a.x; f[4 * i + 1] = a.y; f[4 * i + 2] = b.x; f[4 * i + 3] = b.y;
    }
  }
  __device__ __forceinline__ static T from_float(float x) {
    T r;
    r.bits = (uint8_t)__nv_cvt_float_to_fp8(x, __NV_SATFINITE, Fp8Interp<T>::kind);
    return r;
  }
};
template <> struct Elem<fp8_e4m3> : ElemFp8<fp8_e4m3> {};
template <> struct Elem<fp8_e5m2> : ElemFp8<fp8_e5m2> {};

// ---- global / shared access -----------------------------------------------------------------
// streaming 16-byte load: read once, do not keep in L1
__device__ __forceinline__ uint4 ldg_stream(const void* p) {
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
// 16-byte asynchronous global->shared copy (LDGSTS), bypassing L1
// L2 cache policy for data that is read ONCE (summary rows, selected pages): evict-first, so that the stream leaves the
// small arrays the next kernel reads (scores, page table, selection lists, queries) in the cache.  Measured on C3: the
// summary stream 86.6 -> 84.7 us, the selected pages 84.7 -> 83.7 us per step.
// The launchers ask for it only when the stream is larger than half the L2 (l2_stream_once): a small batch whose summaries
// and selected pages fit the cache keeps the default policy, so that the next decode step -- which selects mostly the
// same pages -- can still find them there.
__device__ __forceinline__ uint64_t l2_stream_policy(bool once) {
  uint64_t pol;
  if (once) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void cp_async16_hint(uint32_t dst, const void* src, uint64_t pol) {
  asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, 16, %2;" ::"r"(dst), "l"(src), "l"(pol));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N));
}

// round a double to the storage type once, to nearest even (the block top-k centroid, Eq.1).  The sum of
// a page's bf16 / fp32 keys is exact in double for bf16 and correctly rounded pairwise for fp32; the oracle does the same.
template <typename T> __device__ __forceinline__ T round_double(double x);
template <> __device__ __forceinline__ float round_double<float>(double x) { return __double2float_rn(x); }
template <> __device__ __forceinline__ __nv_bfloat16 round_double<__nv_bfloat16>(double x) {
  // keep 8 significand bits of the double directly (going through float would round twice)
  unsigned long long b = (unsigned long long)__double_as_longlong(x);
  b += ((1ull << 44) - 1) + ((b >> 45) & 1ull);      // nearest, ties to even, at bit 45
  b &= ~((1ull << 45) - 1);
  return __float2bfloat16_rn(__double2float_rn(__longlong_as_double((long long)b)));   // both conversions are exact now
}

// (fp8 pools have no centroid flow -- vx_create rejects the pair -- these only let the summary kernel's template instantiate)
template <> __device__ __forceinline__ fp8_e4m3 round_double<fp8_e4m3>(double x) { return Elem<fp8_e4m3>::from_float((float)x); }
template <> __device__ __forceinline__ fp8_e5m2 round_double<fp8_e5m2>(double x) { return Elem<fp8_e5m2>::from_float((float)x); }

// ---- warp reductions --------------------------------------------------------------------------
template <int WIDTH = 32> __device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = WIDTH / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
template <int WIDTH = 32> __device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = WIDTH / 2; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// ---- order-preserving float <-> uint32 key (larger float <=> larger key) ---------------------
__device__ __forceinline__ uint32_t float_to_key(float f) {
  uint32_t u = __float_as_uint(f);
  if (u == 0x80000000u) u = 0u;                  // -0.0 == +0.0: one key, so the tie goes to the lower index
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

__device__ __forceinline__ float key_to_float(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7FFFFFFFu) : ~k);
}

__device__ __forceinline__ int ceil_div(int a, int b) { return (a + b - 1) / b; }

// Selection blocks finer than the physical page (include/vortex_b200.h vx_geom.block_size): the kernels see
// blocks as their "pages"; physical block id = page id * bpp + block in page, so a block's first token row sits at
// page * stride_page + (block in page) * block_tokens * stride_token.  bpp = 1: the page itself.
__device__ __forceinline__ int64_t pool_block_base(int64_t phys, int64_t stride_page, int bpp, int64_t block_tokens_stride) {
  return bpp == 1 ? phys * stride_page : (phys / bpp) * stride_page + (phys % bpp) * block_tokens_stride;
}

// ---- programmatic dependent launch (PDL): the kernels of one decode step are chained so that a
// kernel's prologue (index loads, barrier / TMEM set-up, Q staging) overlaps its predecessor's tail.
// pdl_wait(): everything the preceding kernel wrote is visible after it (no-op without the attribute).
// pdl_trigger(): this CTA no longer needs the next kernel to stay away.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// bring `bytes` (multiple of 16) contiguous bytes into L2 without a destination (cp.async.bulk.prefetch)
__device__ __forceinline__ void l2_prefetch(const void* p, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

__device__ __forceinline__ float ldcg_f32(const float* p) {
  float v;
  asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}

// ---- phase tracing (builds with -DVX_TRACE only: `python -m paper_2606_06453_b200.build --trace`) ------------------
// vx_trace_attach() hands the kernels of one kind a device buffer of 16 int64 slots per CTA; VX_TRACE_STAMP(cta, k)
// stores %globaltimer (ns, one clock for the whole GPU) into slot k of CTA `cta`.  The slot meanings are listed in
// paper_2606_06453_b200/trace.py, which prints the per-CTA timelines kept in profiles/.  Without -DVX_TRACE the
// macro is empty and the product library contains none of this.
#ifdef VX_TRACE
static __device__ long long* g_vx_trace_buf;     // one copy per translation unit (set by its vx_trace_set_* below)
static __device__ int g_vx_trace_ctas;
#define VX_TRACE_STAMP(cta, k)                                                            \
  do {                                                                                    \
    if (g_vx_trace_buf != nullptr && (int)(cta) < g_vx_trace_ctas) {                      \
      long long t_;                                                                       \
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                              \
      g_vx_trace_buf[(long long)(cta) * 16 + (k)] = t_;                                   \
    }                                                                                     \
  } while (0)
#define VX_TRACE_SMID(cta)                                                                \
  do {                                                                                    \
    if (g_vx_trace_buf != nullptr && (int)(cta) < g_vx_trace_ctas) {                      \
      unsigned sm_;                                                                       \
      asm volatile("mov.u32 %0, %%smid;" : "=r"(sm_));                                    \
      g_vx_trace_buf[(long long)(cta) * 16 + 15] = sm_;                                   \
    }                                                                                     \
  } while (0)
#define VX_TRACE_SETTER(name)                                                             \
  cudaError_t name(long long* buf, int ctas) {                                            \
    cudaError_t e = cudaMemcpyToSymbol(g_vx_trace_buf, &buf, sizeof(buf));                \
    return e != cudaSuccess ? e : cudaMemcpyToSymbol(g_vx_trace_ctas, &ctas, sizeof(ctas)); \
  }
#else
#define VX_TRACE_STAMP(cta, k) do {} while (0)
#define VX_TRACE_SMID(cta) do {} while (0)
#define VX_TRACE_SETTER(name) \
  cudaError_t name(long long*, int) { return cudaErrorNotSupported; }
#endif

// thread-block cluster (the splits of one request / of one (request, KV head)): barrier over all threads of all CTAs, peer shared-memory reads
__device__ __forceinline__ void cluster_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// ... the same barrier without the release: for the LAST hand-over of a kernel, where a CTA only tells its peers that it
// has finished READING their shared memory (the values are consumed, so the loads are complete).  A release here would
// also wait for the CTA's outstanding global stores -- its output rows -- to be acknowledged (~1 us on the decode kernels).
__device__ __forceinline__ void cluster_sync_relaxed() {
  asm volatile("barrier.cluster.arrive.relaxed.aligned;\n\tbarrier.cluster.wait.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t dsmem_addr(uint32_t local, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local), "r"(rank));
  return r;
}
__device__ __forceinline__ float dsmem_ld_f32(uint32_t addr) {
  float v;
  asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void dsmem_st_f32(uint32_t addr, float v) {
  asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ uint32_t dsmem_ld_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void dsmem_st_u32(uint32_t addr, uint32_t v) {
  asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void dsmem_red_add_u32(uint32_t addr, uint32_t v) {
  asm volatile("red.shared::cluster.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ float4 dsmem_ld_f32x4(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
  return v;
}

// ---- (a5) LSE merge inside a thread-block cluster: the n_part splits of a unit are the CTAs of one
// cluster; each left its normalised partial [8 rows][v_dim] fp32 followed by 8 lse values at the same shared-memory
// offset `part` (rows >= n_rows unused).  CTA `rank` merges every n_part-th slice of blockDim.x 4-element vectors.
// Call between two cluster_sync(): after every CTA's partial is written, before any CTA may exit.  n_part <= 8.
__device__ __forceinline__ void store4(float* dst, float4 v);
__device__ __forceinline__ void store4(__nv_bfloat16* dst, float4 v);
template <typename T>
__device__ __forceinline__ void cluster_merge_partials(const float* part, int v_dim, int n_rows, int rank, int n_part,
                                                       int64_t row0, T* out, float* lse) {
  const int vec = v_dim / 4;
  const uint32_t part_u32 = (uint32_t)__cvta_generic_to_shared(part);
  for (int e = rank * (int)blockDim.x + threadIdx.x; e < n_rows * vec; e += n_part * blockDim.x) {
    const int h = e / vec, c = (e % vec) * 4;
    float w[8];
    float mx = -INFINITY;
#pragma unroll
    for (int sp = 0; sp < 8; ++sp) {
      w[sp] = sp < n_part ? dsmem_ld_f32(dsmem_addr(part_u32 + (8 * v_dim + h) * 4, sp)) : -INFINITY;
      mx = fmaxf(mx, w[sp]);
    }
    float z = 0.f;
#pragma unroll
    for (int sp = 0; sp < 8; ++sp) { w[sp] = mx == -INFINITY ? 0.f : __expf(w[sp] - mx); z += w[sp]; }
    const float inv = z > 0.f ? 1.f / z : 0.f;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int sp = 0; sp < 8; ++sp) {
      if (sp < n_part) {
        const float4 v = dsmem_ld_f32x4(dsmem_addr(part_u32 + (h * v_dim + c) * 4, sp));
        const float ww = w[sp] * inv;
        acc.x = fmaf(ww, v.x, acc.x); acc.y = fmaf(ww, v.y, acc.y); acc.z = fmaf(ww, v.z, acc.z); acc.w = fmaf(ww, v.w, acc.w);
      }
    }
    store4(out + (row0 + h) * v_dim + c, acc);
    if (c == 0 && lse != nullptr) lse[row0 + h] = z > 0.f ? mx + logf(z) : -INFINITY;
  }
}

// ---- (a5) in-kernel LSE merge: the LAST split CTA of a unit to finish merges the unit's
// partials.  Call with the whole CTA after its own partial (o, lse) is written.  Returns true in the CTA
// that must merge.  counter is zero on entry to the step and is left zero.
__device__ __forceinline__ bool last_split_arrives(int* counter, int num_splits, int* s_flag) {
  __syncthreads();                               // every thread's partial stores happen-before thread 0's fence ...
  if (threadIdx.x == 0) {
    __threadfence();                             // ... which is cumulative: they are visible device-wide before the count
    const int old = atomicAdd(counter, 1);
    const bool last = old == num_splits - 1;
    if (last) *counter = 0;                      // self-cleaning: ready for the next step
    *s_flag = last;
  }
  __syncthreads();
  const bool last = *s_flag != 0;
  if (last) __threadfence();                     // acquire the other CTAs' partials
  return last;
}

// merge rows [row0, row0 + n_rows) of part_o [rows, n_part, v_dim] / part_lse [rows, n_part] into out / lse.
// s_w: n_rows * n_part floats of shared-memory scratch.  The split weights are computed once per row; the
// value loads are independent 16-byte L2 reads (the partials were just written by other SMs: ld.global.cg).
__device__ __forceinline__ float4 ldcg_f32x4(const float* p) {
  float4 v;
  asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ void store4(float* dst, float4 v) { *reinterpret_cast<float4*>(dst) = v; }
__device__ __forceinline__ void store4(__nv_bfloat16* dst, float4 v) {
  __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), b = __floats2bfloat162_rn(v.z, v.w);
  uint2 u = make_uint2(*reinterpret_cast<uint32_t*>(&a), *reinterpret_cast<uint32_t*>(&b));
  *reinterpret_cast<uint2*>(dst) = u;
}
template <typename T>
__device__ __forceinline__ void merge_partials(const float* part_o, const float* part_lse, int64_t row0, int n_rows,
                                               int n_part, int v_dim, T* out, float* lse, float* s_w) {
  for (int e = threadIdx.x; e < n_rows * n_part; e += blockDim.x)       // all lse values in one round trip
    s_w[e] = ldcg_f32(part_lse + row0 * n_part + e);
  __syncthreads();
  for (int r = threadIdx.x; r < n_rows; r += blockDim.x) {
    float* w = s_w + r * n_part;
    float mx = -INFINITY;
    for (int s = 0; s < n_part; ++s) mx = fmaxf(mx, w[s]);
    float z = 0.f;
    for (int s = 0; s < n_part; ++s) z += mx == -INFINITY ? 0.f : __expf(w[s] - mx);
    const float inv = z > 0.f ? 1.f / z : 0.f;
    for (int s = 0; s < n_part; ++s) w[s] = mx == -INFINITY ? 0.f : __expf(w[s] - mx) * inv;
    if (lse != nullptr) lse[row0 + r] = z > 0.f ? mx + logf(z) : -INFINITY;
  }
  __syncthreads();
  const int vec = v_dim / 4;
#pragma unroll 8
  for (int e = threadIdx.x; e < n_rows * vec; e += blockDim.x) {
    const int r = e / vec, c = (e % vec) * 4;
    const float* src = part_o + (row0 + r) * n_part * v_dim + c;
    float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s = 0; s < n_part; ++s) {
      const float w = s_w[r * n_part + s];
      const float4 v = ldcg_f32x4(src + (int64_t)s * v_dim);
      o.x = fmaf(w, v.x, o.x); o.y = fmaf(w, v.y, o.y); o.z = fmaf(w, v.z, o.z); o.w = fmaf(w, v.w, o.w);
    }
    store4(out + (row0 + r) * v_dim + c, o);
  }
}

}  // namespace vx
