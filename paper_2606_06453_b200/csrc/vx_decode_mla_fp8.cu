// vx_decode_mla_fp8.cu -- (a4)+(a5) for the absorbed-MLA latent cache stored as fp8 codes ("inherits their
// precision support, such as fp8 KV cache"; :525 fp8_e4m3 / fp8_e5m2, readings G25-G27).
//
// Two launches: (1) the SELECTED latent pages of every request are widened into a bf16 staging pool in the workspace --
// every fp8 code is exactly a bf16 value, so nothing is rounded; (2) the tensor-core latent decode kernel
// (vx_decode_mla.cu: tcgen05 + TMA + TMEM) runs on that pool through a rewritten selection list, with the pool's
// per-tensor scales folded where the definition puts them: logits = sm_scale * k_scale * (q . code), out = v_scale * sum p * code.
// Against the CUDA-core kernel of vx_decode_generic.cu, which was the only fp8 path for this geometry, this reads the fp8
// pages once (36.9 KB a page) and pays a bf16 write + read of the same pages (2 x 73.7 KB) -- ~8x faster on C4, still
// 3x the bytes of a kernel that converts inside its pipeline.
#include "vx_common.cuh"
#include "vx_internal.h"
#include "vx_mla.cuh"

namespace vx {

template <typename TKV> __device__ __forceinline__ void fp8x4_to_bf16x4(uint32_t four, uint32_t& lo, uint32_t& hi);
template <> __device__ __forceinline__ void fp8x4_to_bf16x4<fp8_e4m3>(uint32_t four, uint32_t& lo, uint32_t& hi) {
  uint32_t h0, h1;
  asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %2;\n\tcvt.rn.f16x2.e4m3x2 %0, l;\n\tcvt.rn.f16x2.e4m3x2 %1, h;\n\t}"
      : "=r"(h0), "=r"(h1) : "r"(four));
  const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&h0)), b = __half22float2(*reinterpret_cast<const __half2*>(&h1));
  const __nv_bfloat162 x = __floats2bfloat162_rn(a.x, a.y), y = __floats2bfloat162_rn(b.x, b.y);   // exact: 4 significant bits
  lo = *reinterpret_cast<const uint32_t*>(&x);
  hi = *reinterpret_cast<const uint32_t*>(&y);
}
template <> __device__ __forceinline__ void fp8x4_to_bf16x4<fp8_e5m2>(uint32_t four, uint32_t& lo, uint32_t& hi) {
  uint32_t h0, h1;
  asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %2;\n\tcvt.rn.f16x2.e5m2x2 %0, l;\n\tcvt.rn.f16x2.e5m2x2 %1, h;\n\t}"
      : "=r"(h0), "=r"(h1) : "r"(four));
  const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&h0)), b = __half22float2(*reinterpret_cast<const __half2*>(&h1));
  const __nv_bfloat162 x = __floats2bfloat162_rn(a.x, a.y), y = __floats2bfloat162_rn(b.x, b.y);   // exact: 3 significant bits
  lo = *reinterpret_cast<const uint32_t*>(&x);
  hi = *reinterpret_cast<const uint32_t*>(&y);
}

// grid (max_budget, batch): CTA (r, i) widens the r-th selected page of request i into staging page i * max_budget + r.
// Tokens past the request's end are written as zeros (their probabilities are zero; a stale code there could be a NaN).
template <typename TKV>
__global__ void __launch_bounds__(256)
stage_latent_fp8_kernel(const uint8_t* __restrict__ kpool, int64_t stride_page, int64_t stride_token,
                        const int32_t* __restrict__ seq_lens, const int32_t* __restrict__ sel_phys,
                        const int32_t* __restrict__ sel_logical, const int32_t* __restrict__ sel_count, int max_budget,
                        __nv_bfloat16* __restrict__ stage, int32_t* __restrict__ stage_sel) {
  using namespace mla;
  constexpr int CH = D / 16;                    // 16-code chunks per token row: 36
  const int r = blockIdx.x, i = blockIdx.y;
  const int n_tok = seq_lens[i];
  pdl_wait();                                   // the selection lists come from the preceding kernel of the step
  const int cnt = sel_count[i];
  const int slot = i * max_budget + r;
  if (threadIdx.x == 0) stage_sel[slot] = r < cnt ? slot : -1;
  if (r >= cnt) return;
  const int phys = sel_phys[slot], lg = sel_logical[slot];
  const int valid = min(PAGE, n_tok - lg * PAGE);
  const uint8_t* src = kpool + (int64_t)phys * stride_page;
  __nv_bfloat16* dst = stage + (int64_t)slot * PAGE * D;
  for (int x0 = threadIdx.x; x0 < PAGE * CH; x0 += 3 * 256) {          // three independent 16-byte loads in flight
    uint4 v[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const int x = x0 + k * 256, t = x / CH, c = x % CH;
      v[k] = (x < PAGE * CH && t < valid) ? *reinterpret_cast<const uint4*>(src + (int64_t)t * stride_token + c * 16) : make_uint4(0, 0, 0, 0);
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const int x = x0 + k * 256;
      if (x < PAGE * CH) {
        uint4 a, b;
        fp8x4_to_bf16x4<TKV>(v[k].x, a.x, a.y);
        fp8x4_to_bf16x4<TKV>(v[k].y, a.z, a.w);
        fp8x4_to_bf16x4<TKV>(v[k].z, b.x, b.y);
        fp8x4_to_bf16x4<TKV>(v[k].w, b.z, b.w);
        uint4* o = reinterpret_cast<uint4*>(dst + (int64_t)(x / CH) * D + (x % CH) * 16);
        o[0] = a;
        o[1] = b;
      }
    }
  }
}

bool mla_fp8_staged_supported(const vx_geom& g) {
  return g.kv_shared && kv_is_fp8(g) && g.dtype == VX_DT_BF16 && g.num_kv_heads == 1 && g.qk_dim == mla::D && g.v_dim == mla::DV &&
         g.page_size == mla::PAGE && (g.block_size == 0 || g.block_size == g.page_size) && g.num_q_heads <= mla::NH;
}

size_t mla_fp8_stage_elems(const vx_geom& g, int max_batch, int max_budget) {
  return mla_fp8_staged_supported(g) ? (size_t)max_batch * (size_t)max_budget * mla::PAGE * mla::D : 0;
}

cudaError_t launch_decode_mla_fp8_staged(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                         const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                         int32_t max_budget, void* out, float* lse, cudaStream_t s, const DecodeOpts& opt) {
  if (max_budget > c->max_budget || pt.batch > c->max_batch) return cudaErrorInvalidValue;   // (the staging pool's size)
  dim3 grid(max_budget, pt.batch);
  auto kernel = c->g.kv_format == VX_KV_FP8_E4M3 ? stage_latent_fp8_kernel<fp8_e4m3> : stage_latent_fp8_kernel<fp8_e5m2>;
  cudaError_t e = launch_kernel(kernel, grid, dim3(256), 0, s, opt.pdl, static_cast<const uint8_t*>(pool.k), pool.stride_page,
                                pool.stride_token, pt.seq_lens, sel_phys, sel_logical, sel_count, max_budget,
                                static_cast<__nv_bfloat16*>(c->ws.mla_stage), c->ws.mla_stage_sel);
  c->launches += 1;
  if (e != cudaSuccess) return e;
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  vx_kv_pool staged{};
  staged.k = c->ws.mla_stage;
  staged.v = nullptr;
  staged.stride_page = (int64_t)mla::PAGE * mla::D;
  staged.stride_token = mla::D;
  staged.stride_head = 0;
  staged.num_pool_pages = (int64_t)pt.batch * max_budget;
  staged.k_scale = staged.v_scale = 1.f;
  DecodeOpts o2;
  o2.pdl = true;                                // waits for the staging kernel
  o2.budget = opt.budget;
  o2.scale_mul = pool.k_scale;
  o2.out_scale = pool.v_scale;
  return launch_decode_mla_tc(c, q, staged, pt, c->ws.mla_stage_sel, sel_logical, sel_count, max_budget, out, lse, s, o2);
}

}  // namespace vx
