// vx_decode_gqa_fp8.cu -- (a4)+(a5) sparse paged decode for GQA over an fp8 KV cache (page 16, d = dv = 128, group <= 8,
// bf16 queries and outputs).  PAPER.md:92 Eq.4 over the selected pages (:200), split + LSE merge (:75); fp8 KV cache :200,
// :520, :525 (a code c stands for scale * decode(c), G25-G26).
//
// The structure of vx_decode_gqa.cu (every warp streams its own pages through a private cp.async ring, the skinny
// contractions S^T = K Q^T and O^T += V^T P^T as m16n8k16 MMAs with the group's heads on N = 8) with one-byte elements:
//   * a (page, head) chunk is 2 KB for K and 2 KB for V -- half the HBM bytes, which is the point of the format;
//   * the tiles stay fp8 in shared memory and are widened in registers: ldmatrix (b16 units = PAIRS of codes) hands a
//     thread four consecutive channels of a token; the hardware conversion cvt.rn.f16x2.{e4m3,e5m2}x2 makes the f16
//     fragments (every fp8 value is exact in f16), so the MMAs are f16 x f16 -> fp32.  The contraction index of
//     S^T (channels) and the row index of O^T (channels) are permuted to fit what ldmatrix delivers -- the same
//     permutation on the Q fragments / on the epilogue's addressing, so nothing is shuffled;
//   * Q is converted bf16 -> f16 once (exact in the f16 normal range; a power-of-two pre-scale, folded back into the
//     softmax scale, keeps |q| below 2^15 whatever the queries are);  P is rounded to f16 (11 bits) for the second MMA;
//   * k_scale rides in the softmax scale, v_scale in the final normalisation.
#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

namespace gq8 {
constexpr int WARPS = 4, STAGES = 4, PAGE = 16, D = 128;
constexpr int ROWB = D;                       // bytes per token row
constexpr int PAGEB = PAGE * ROWB;            // 2 KB: one K (or V) chunk of a (page, head)
constexpr int KS = D / 16;                    // k-steps of QK^T = m-tiles of PV
constexpr int CP_ITERS = PAGE * (ROWB / 16) / kWarp;      // 16-byte copies per lane per chunk: 4
constexpr int SMEM = WARPS * STAGES * 2 * PAGEB;          // 64 KB
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
}  // namespace gq8

__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_trans(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ uint32_t movm_trans(uint32_t x) {
  uint32_t y;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(y) : "r"(x));
  return y;
}
// D(16x8, fp32) += A(16x16, f16 row) * B(16x8, f16 col)
__device__ __forceinline__ void mma_f16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_f16x2(float lo, float hi) {
  const __half2 v = __floats2half2_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&v);
}
// four fp8 codes (one 32-bit word) -> two f16x2 words: lo = codes 0, 1; hi = codes 2, 3.  One F2FP.UNPACK_B each (the
// library intrinsic's __half2_raw return value cost two extra PRMT per conversion here).
template <typename TKV> __device__ __forceinline__ void fp8x4_to_f16(uint32_t four, uint32_t& lo, uint32_t& hi);
template <> __device__ __forceinline__ void fp8x4_to_f16<fp8_e4m3>(uint32_t four, uint32_t& lo, uint32_t& hi) {
  asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %2;\n\tcvt.rn.f16x2.e4m3x2 %0, l;\n\tcvt.rn.f16x2.e4m3x2 %1, h;\n\t}"
      : "=r"(lo), "=r"(hi) : "r"(four));
}
template <> __device__ __forceinline__ void fp8x4_to_f16<fp8_e5m2>(uint32_t four, uint32_t& lo, uint32_t& hi) {
  asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %2;\n\tcvt.rn.f16x2.e5m2x2 %0, l;\n\tcvt.rn.f16x2.e5m2x2 %1, h;\n\t}"
      : "=r"(lo), "=r"(hi) : "r"(four));
}
__device__ __forceinline__ void cp16_zfill(uint32_t dst, const void* src, bool valid, uint64_t pol) {   // (evict-first: vx_common.cuh)
  asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2, %3;" ::"r"(dst), "l"(src), "r"(valid ? 16 : 0), "l"(pol));
}

template <typename TKV, bool CL>
__global__ void __launch_bounds__(gq8::WARPS * kWarp)
decode_gqa_fp8_kernel(const __nv_bfloat16* __restrict__ q, const uint8_t* __restrict__ kpool, const uint8_t* __restrict__ vpool,
                      int64_t stride_page, int64_t stride_token, int64_t stride_head, int num_q_heads, int num_kv_heads,
                      float scale_log2, float v_scale, const int32_t* __restrict__ seq_lens,
                      const int32_t* __restrict__ sel_phys, const int32_t* __restrict__ sel_logical,
                      const int32_t* __restrict__ sel_count, int max_budget, int num_splits, float* __restrict__ part_o,
                      float* __restrict__ part_lse, int* __restrict__ unit_counter, __nv_bfloat16* __restrict__ out,
                      float* __restrict__ lse_out, const int32_t* __restrict__ budget_opt, int bpp,
                      uint8_t* __restrict__ summary_upd, int stream_once) {
  using namespace gq8;
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ float s_m[WARPS][8], s_l[WARPS][8];
  __shared__ float s_hinv[8], s_hlse[8];           // per head of the group: v_scale / denominator and LSE of this CTA's pages
  __shared__ int s_valid[WARPS][STAGES];         // valid tokens of the page staged in each slot (bit 8: the request's newest page)
  __shared__ int s_phys[WARPS][STAGES];          // its physical id
  __shared__ int s_last;

  const int split = blockIdx.x, kvh = blockIdx.y, i = blockIdx.z;
  const int warp = threadIdx.x / kWarp, lane = threadIdx.x % kWarp;
  const int grp = num_q_heads / num_kv_heads;
  const int n_tok = seq_lens[i];
  const int newest_page = (n_tok - 1) / PAGE;
  const int cnt_known = budget_opt ? max(0, min(min(budget_opt[i], max_budget), newest_page + 1)) : -1;

  // Q^T as the B operand, f16.  Thread (head h = lane / 4, j = lane % 4) holds for k-step ks the channels 16 ks + 4 j .. + 3:
  // k-slots (2j, 2j+1) <- channels 4j, 4j+1;  k-slots (2j+8, 2j+9) <- channels 4j+2, 4j+3  (what ldmatrix hands the A side)
  uint32_t qb[KS][2];
  {
    const int h = lane / 4, j = lane % 4;
    const __nv_bfloat16* qrow = q + ((int64_t)i * num_q_heads + kvh * grp + h) * D;
    float qf[KS][4];
    float qmax = 0.f;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      uint2 raw = make_uint2(0u, 0u);
      if (h < grp) raw = *reinterpret_cast<const uint2*>(qrow + ks * 16 + 4 * j);
      qf[ks][0] = __uint_as_float(raw.x << 16); qf[ks][1] = __uint_as_float(raw.x & 0xffff0000u);
      qf[ks][2] = __uint_as_float(raw.y << 16); qf[ks][3] = __uint_as_float(raw.y & 0xffff0000u);
#pragma unroll
      for (int e = 0; e < 4; ++e) qmax = fmaxf(qmax, fabsf(qf[ks][e]));
    }
    qmax = warp_max(qmax);
    const int e2 = qmax > 16384.f ? ilogbf(qmax) - 13 : 0;        // |q| 2^-e2 < 2^14: inside the f16 range
    const float down = exp2f((float)-e2);
    scale_log2 *= exp2f((float)e2);
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      qb[ks][0] = pack_f16x2(qf[ks][0] * down, qf[ks][1] * down);
      qb[ks][1] = pack_f16x2(qf[ks][2] * down, qf[ks][3] * down);
    }
  }
  pdl_wait();                                   // the selection lists come from the preceding kernel of the step

  const int cnt = cnt_known >= 0 ? cnt_known : sel_count[i * num_kv_heads + kvh];
  const int per_split = (cnt + num_splits - 1) / num_splits;
  const int r_begin = min(split * per_split, cnt), r_end = min(r_begin + per_split, cnt);
  const int32_t* phys_list = sel_phys + ((int64_t)i * num_kv_heads + kvh) * max_budget;
  const int32_t* log_list = sel_logical + ((int64_t)i * num_kv_heads + kvh) * max_budget;
  const int my_pages = r_end - r_begin > warp ? (r_end - r_begin - warp + WARPS - 1) / WARPS : 0;   // r_begin + warp, + WARPS, ..

  uint8_t* ring = smem + (size_t)warp * STAGES * 2 * PAGEB;
  const uint32_t ring_u32 = smem_u32(ring);
  int id_phys = 0, id_valid = 0;                // lane l: this warp's (base + l)-th page
  auto fetch_ids = [&](int base) {
    const int p = base + lane;
    if (p < my_pages) {
      const int r = r_begin + warp + p * WARPS;
      id_phys = phys_list[r];
      const int lg = log_list[r];
      id_valid = min(PAGE, n_tok - lg * PAGE) | (lg == newest_page ? 256 : 0);
    }
  };
  const uint64_t pol = l2_stream_policy(stream_once != 0);
  auto issue = [&](int p) {                     // all lanes: copy page p of this warp into slot p % STAGES
    const int phys = __shfl_sync(0xffffffffu, id_phys, p & 31);
    const int venc = __shfl_sync(0xffffffffu, id_valid, p & 31);
    const int nv = venc & 255;
    const int64_t base = pool_block_base(phys, stride_page, bpp, PAGE * stride_token) + (int64_t)kvh * stride_head;
    const uint32_t dst = ring_u32 + (uint32_t)(p % STAGES) * 2 * PAGEB;
    if (lane == 0) { s_valid[warp][p % STAGES] = venc; s_phys[warp][p % STAGES] = phys; }
#pragma unroll
    for (int it = 0; it < CP_ITERS; ++it) {
      const int x = it * kWarp + lane;
      const int t = x / 8, c = x % 8;           // token row, 16-byte chunk (16 channels)
      const uint32_t off = t * ROWB + ((c ^ (t & 7)) * 16);
      const int64_t src = base + (int64_t)t * stride_token + c * 16;
      cp16_zfill(dst + off, kpool + src, t < nv, pol);
      cp16_zfill(dst + PAGEB + off, vpool + src, t < nv, pol);
    }
  };

  float o[KS][4];
#pragma unroll
  for (int mt = 0; mt < KS; ++mt) { o[mt][0] = o[mt][1] = o[mt][2] = o[mt][3] = 0.f; }
  float m_a = -INFINITY, m_b = -INFINITY, l_a = 0.f, l_b = 0.f;   // heads 2 * (lane % 4), + 1

  fetch_ids(0);
#pragma unroll
  for (int p = 0; p < STAGES - 1; ++p) {
    if (p < my_pages) issue(p);
    cp_async_commit();
  }
  const int tr = lane & 15, hi = lane >> 4;     // ldmatrix row address: token row, and which of the two 16-channel chunks
  for (int p = 0; p < my_pages; ++p) {
    cp_async_wait<STAGES - 2>();                // page p has landed (this lane's copies)
    __syncwarp();                               // ... and every lane's; all lanes are done with page p - 1
    const int valid_enc = s_valid[warp][p % STAGES];
    const int valid = valid_enc & 255;
    const int phys_p = s_phys[warp][p % STAGES];
    {
      const int nxt = p + STAGES - 1;           // refill the slot page p - 1 used
      if ((nxt & 31) == 0 && nxt < my_pages) fetch_ids(nxt);
      if (nxt < my_pages) issue(nxt);
      cp_async_commit();
    }
    const uint32_t kst = ring_u32 + (uint32_t)(p % STAGES) * 2 * PAGEB, vst = kst + PAGEB;

    if (summary_upd != nullptr && (valid_enc & 256)) {
      // (a1) this is the request's newest page: rebuild its min / max summary CODES from the staged keys (
      // exact: the envelope of representable values is representable).  Lane owns 4 consecutive channels of the row.
      const int c = lane >> 2, o16 = (lane & 3) * 4;
      const uint8_t* kt = ring + (size_t)(p % STAGES) * 2 * PAGEB;
      uint32_t w0, w1;
      fp8x4_to_f16<TKV>(*reinterpret_cast<const uint32_t*>(kt + (c * 16) + o16), w0, w1);      // token 0 (c ^ 0 = c)
      __half2 lo0 = *reinterpret_cast<__half2*>(&w0), lo1 = *reinterpret_cast<__half2*>(&w1), hi0 = lo0, hi1 = lo1;
      for (int t = 1; t < valid; ++t) {
        fp8x4_to_f16<TKV>(*reinterpret_cast<const uint32_t*>(kt + t * ROWB + ((c ^ (t & 7)) * 16) + o16), w0, w1);
        const __half2 a = *reinterpret_cast<__half2*>(&w0), b = *reinterpret_cast<__half2*>(&w1);
        lo0 = __hmin2(lo0, a); lo1 = __hmin2(lo1, b);
        hi0 = __hmax2(hi0, a); hi1 = __hmax2(hi1, b);
      }
      auto pack4 = [](__half2 x, __half2 y) -> uint32_t {                   // four f16 that are fp8 values -> their codes
        const __nv_fp8x2_storage_t p0 = __nv_cvt_halfraw2_to_fp8x2(*reinterpret_cast<__half2_raw*>(&x), __NV_SATFINITE, Fp8Interp<TKV>::kind);
        const __nv_fp8x2_storage_t p1 = __nv_cvt_halfraw2_to_fp8x2(*reinterpret_cast<__half2_raw*>(&y), __NV_SATFINITE, Fp8Interp<TKV>::kind);
        return (uint32_t)p0 | ((uint32_t)p1 << 16);
      };
      uint8_t* dst = summary_upd + (((int64_t)phys_p * num_kv_heads + kvh) * 2) * D + lane * 4;
      *reinterpret_cast<uint32_t*>(dst) = pack4(lo0, lo1);
      *reinterpret_cast<uint32_t*>(dst + D) = pack4(hi0, hi1);
    }

    // S^T[16 tokens x 8 heads] = K[16 x D] . Q^T : one ldmatrix.x4 = two k-steps (tokens 0-7 / 8-15 x chunks 2 kk, 2 kk + 1)
    float s[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int kk = 0; kk < KS / 2; ++kk) {
      uint32_t r[4];
      const int c = 2 * kk + hi;
      ldsm_x4(r, kst + tr * ROWB + ((c ^ (tr & 7)) * 16));
      // r[0]: token lane/4, r[1]: token lane/4 + 8 (chunk 2 kk);  r[2], r[3]: the same tokens, chunk 2 kk + 1
      uint32_t a0, a1, a2, a3;
      fp8x4_to_f16<TKV>(r[0], a0, a2);
      fp8x4_to_f16<TKV>(r[1], a1, a3);
      mma_f16(s, a0, a1, a2, a3, qb[2 * kk][0], qb[2 * kk][1]);
      fp8x4_to_f16<TKV>(r[2], a0, a2);
      fp8x4_to_f16<TKV>(r[3], a1, a3);
      mma_f16(s, a0, a1, a2, a3, qb[2 * kk + 1][0], qb[2 * kk + 1][1]);
    }
    // online softmax, base 2.  s[0], s[1]: token lane/4, heads a, b;  s[2], s[3]: token lane/4 + 8
    const int t0 = lane / 4;
    const float sa0 = t0 < valid ? s[0] * scale_log2 : -INFINITY, sb0 = t0 < valid ? s[1] * scale_log2 : -INFINITY;
    const float sa1 = t0 + 8 < valid ? s[2] * scale_log2 : -INFINITY, sb1 = t0 + 8 < valid ? s[3] * scale_log2 : -INFINITY;
    float mx_a = fmaxf(sa0, sa1), mx_b = fmaxf(sb0, sb1);
#pragma unroll
    for (int off = 4; off < 32; off <<= 1) {
      mx_a = fmaxf(mx_a, __shfl_xor_sync(0xffffffffu, mx_a, off));
      mx_b = fmaxf(mx_b, __shfl_xor_sync(0xffffffffu, mx_b, off));
    }
    const float mn_a = fmaxf(m_a, mx_a), mn_b = fmaxf(m_b, mx_b);   // finite: token 0 of a page is always valid
    const float al_a = exp2f(m_a - mn_a), al_b = exp2f(m_b - mn_b);
    const float pa0 = exp2f(sa0 - mn_a), pb0 = exp2f(sb0 - mn_b), pa1 = exp2f(sa1 - mn_a), pb1 = exp2f(sb1 - mn_b);
    l_a = l_a * al_a + pa0 + pa1;
    l_b = l_b * al_b + pb0 + pb1;
    m_a = mn_a; m_b = mn_b;
    // P^T as the B operand of the second MMA: transpose the 8x8 (token, head) tiles across the warp
    const uint32_t pb_lo = movm_trans(pack_f16x2(pa0, pb0));
    const uint32_t pb_hi = movm_trans(pack_f16x2(pa1, pb1));

    // O^T[D x 8 heads] = O^T * alpha + V^T[D x 16 tokens] . P.  ldmatrix.trans hands a thread (tokens 2j, 2j+1) x (channels
    // 2g, 2g+1) of a 16-channel chunk as bytes [t0c0, t0c1, t1c0, t1c1]; one byte permute makes the token pairs of channel
    // 2g (row slot g of the m-tile) and of channel 2g+1 (row slot g + 8).
#pragma unroll
    for (int mm = 0; mm < KS / 2; ++mm) {
      uint32_t r[4];
      const int c = 2 * mm + hi;
      ldsm_x4_trans(r, vst + tr * ROWB + ((c ^ (tr & 7)) * 16));
#pragma unroll
      for (int u = 0; u < 2; ++u) {             // m-tile mt = 2 mm + u: r[2u] = tokens 0-7, r[2u+1] = tokens 8-15
        const int mt = 2 * mm + u;
        const uint32_t x0 = __byte_perm(r[2 * u], 0u, 0x3120), x1 = __byte_perm(r[2 * u + 1], 0u, 0x3120);
        o[mt][0] *= al_a; o[mt][1] *= al_b; o[mt][2] *= al_a; o[mt][3] *= al_b;
        uint32_t a0, a1, a2, a3;
        fp8x4_to_f16<TKV>(x0, a0, a1);
        fp8x4_to_f16<TKV>(x1, a2, a3);
        mma_f16(o[mt], a0, a1, a2, a3, pb_lo, pb_hi);
      }
    }
  }
  cp_async_wait<0>();
  pdl_trigger();

  // per-warp denominators: sum the lane partials of each head column
#pragma unroll
  for (int off = 4; off < 32; off <<= 1) {
    l_a += __shfl_xor_sync(0xffffffffu, l_a, off);
    l_b += __shfl_xor_sync(0xffffffffu, l_b, off);
  }
  if (lane < 4) {
    s_m[warp][2 * lane] = m_a; s_m[warp][2 * lane + 1] = m_b;
    s_l[warp][2 * lane] = l_a; s_l[warp][2 * lane + 1] = l_b;
  }
  __syncthreads();                              // every warp is done with its ring: reuse it for the merge
  const int ha = 2 * (lane % 4);
  float mb_a = -INFINITY, mb_b = -INFINITY;
#pragma unroll
  for (int w = 0; w < WARPS; ++w) { mb_a = fmaxf(mb_a, s_m[w][ha]); mb_b = fmaxf(mb_b, s_m[w][ha + 1]); }
  const float f_a = m_a == -INFINITY ? 0.f : exp2f(m_a - mb_a), f_b = m_b == -INFINITY ? 0.f : exp2f(m_b - mb_b);
  float* so = reinterpret_cast<float*>(ring);   // [D][8 heads] fp32 = 4 KB = one stage
  // cluster merge: this CTA's normalised partial [8 heads][D] + 8 lse, behind warp 0's `so` (nobody else's)
  [[maybe_unused]] float* cl_part = reinterpret_cast<float*>(smem + 2 * PAGEB);
#pragma unroll
  for (int mt = 0; mt < KS; ++mt) {             // row slot g <-> channel 16 mt + 2 g, row slot g + 8 <-> channel 16 mt + 2 g + 1
    const int d0 = mt * 16 + 2 * (lane / 4);
    *reinterpret_cast<float2*>(so + d0 * 8 + ha) = make_float2(o[mt][0] * f_a, o[mt][1] * f_b);
    *reinterpret_cast<float2*>(so + (d0 + 1) * 8 + ha) = make_float2(o[mt][2] * f_a, o[mt][3] * f_b);
  }
  if (threadIdx.x < 8) {                        // per head, once: the CTA's reference, v_scale / denominator and LSE
    const int h = threadIdx.x;
    float mb = -INFINITY;
#pragma unroll
    for (int w = 0; w < WARPS; ++w) mb = fmaxf(mb, s_m[w][h]);
    float lsum = 0.f;
#pragma unroll
    for (int w = 0; w < WARPS; ++w) lsum += s_m[w][h] == -INFINITY ? 0.f : s_l[w][h] * exp2f(s_m[w][h] - mb);
    s_hinv[h] = lsum > 0.f ? v_scale / lsum : 0.f;
    s_hlse[h] = lsum > 0.f ? (mb + log2f(lsum)) * kLn2 : -INFINITY;
  }
  __syncthreads();
  // four heads of one channel per thread: one 16-byte read per warp partial
  for (int e = threadIdx.x; e < ((grp + 3) / 4) * D; e += WARPS * kWarp) {
    const int d = e % D, h0 = 4 * (e / D);
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int w = 0; w < WARPS; ++w) {
      const float4 v = *reinterpret_cast<const float4*>(smem + (size_t)w * STAGES * 2 * PAGEB + (d * 8 + h0) * 4);
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    const float a4[4] = {acc.x, acc.y, acc.z, acc.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int h = h0 + k;
      if (h < grp) {
        const float val = a4[k] * s_hinv[h];
        const int64_t head_row = (int64_t)i * num_q_heads + kvh * grp + h;
        if (num_splits == 1) {
          out[head_row * D + d] = __float2bfloat16_rn(val);
          if (d == 0 && lse_out != nullptr) lse_out[head_row] = s_hlse[h];
        } else if constexpr (CL) {
          cl_part[h * D + d] = val;
          if (d == 0) cl_part[8 * D + h] = s_hlse[h];
        } else {
          part_o[(head_row * num_splits + split) * D + d] = val;
          if (d == 0) part_lse[head_row * num_splits + split] = s_hlse[h];
        }
      }
    }
  }
  if constexpr (CL) {                           // (a5) the splits are one cluster: merge over distributed shared memory
    cluster_sync();
    cluster_merge_partials(cl_part, D, grp, split, num_splits, (int64_t)i * num_q_heads + kvh * grp, out, lse_out);
    cluster_sync_relaxed();                       // no CTA leaves while a peer still reads its partial
  } else if (num_splits > 1) {                  // (a5) the last split of this (request, KV head) merges by LSE
    if (last_split_arrives(unit_counter + i * num_kv_heads + kvh, num_splits, &s_last))
      merge_partials<__nv_bfloat16>(part_o, part_lse, (int64_t)i * num_q_heads + kvh * grp, grp, num_splits, D, out, lse_out,
                                     reinterpret_cast<float*>(smem));
  }
}

bool gqa_fp8_fast_supported(const vx_geom& g) {
  const int grp = g.num_kv_heads > 0 ? g.num_q_heads / g.num_kv_heads : 0;
  return kv_is_fp8(g) && g.dtype == VX_DT_BF16 && !g.kv_shared && g.page_size == gq8::PAGE && g.qk_dim == gq8::D &&
         g.v_dim == gq8::D && grp >= 1 && grp <= 8;
}

static int decode_gqa_fp8_splits(const vx_ctx* c, int n_req, int max_budget) {
  const int units = n_req * c->g.num_kv_heads;
  const int per_sm = 227 * 1024 / (gq8::SMEM + 1024);
  const int slots = c->num_sms * (per_sm > 0 ? per_sm : 1);
  int splits = 1, best_cost = 1 << 30;
  for (int sp = 1; sp <= kMaxSplits && sp <= max_budget; ++sp) {
    const int waves = (units * sp + slots - 1) / slots;
    // a wave costs its pages per warp plus ~30 page times that stream nothing (measured on C2 / C3: launch, Q and id
    // loads, first-page latency, in-CTA and cross-split merge ~ 15 us against 0.5 us per page and warp)
    const int cost = waves * (((max_budget + sp - 1) / sp + gq8::WARPS - 1) / gq8::WARPS + 30);
    if (cost < best_cost) { best_cost = cost; splits = sp; }
  }
  return splits;
}

template <typename TKV>
static cudaError_t launch_gqa_fp8_t(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                    const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                    int32_t max_budget, void* out, float* lse, cudaStream_t s, bool pdl, const int32_t* budget,
                                    void* summary_upd) {
  const vx_geom& g = c->g;
  if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(decode_gqa_fp8_kernel<TKV, false>), c->device, gq8::SMEM)) return e;
  if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(decode_gqa_fp8_kernel<TKV, true>), c->device, gq8::SMEM)) return e;
  const int splits = decode_gqa_fp8_splits(c, pt.batch, max_budget);
  dim3 grid(splits, g.num_kv_heads, pt.batch);
  const bool cl = splits == 2 || splits == 4 || splits == 8;
  cudaError_t e = launch_kernel_cluster(cl ? decode_gqa_fp8_kernel<TKV, true> : decode_gqa_fp8_kernel<TKV, false>, grid,
      dim3(gq8::WARPS * kWarp), (size_t)gq8::SMEM, s, pdl, cl ? splits : 1,
      static_cast<const __nv_bfloat16*>(q), static_cast<const uint8_t*>(pool.k), static_cast<const uint8_t*>(pool.v),
      pool.stride_page, pool.stride_token, pool.stride_head, g.num_q_heads, g.num_kv_heads,
      g.sm_scale * pool.k_scale * gq8::kLog2e, pool.v_scale, pt.seq_lens, sel_phys, sel_logical, sel_count, max_budget, splits,
      c->ws.part_o, c->ws.part_lse, c->ws.unit_counter, static_cast<__nv_bfloat16*>(out), lse, budget, c->bpp, static_cast<uint8_t*>(summary_upd),
      l2_stream_once(c, (int64_t)pt.batch * g.num_kv_heads * max_budget * 2 * gq8::PAGEB) ? 1 : 0);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_decode_gqa_fp8(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                  const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                  int32_t max_budget, void* out, float* lse, cudaStream_t s, bool pdl, const int32_t* budget,
                                  void* summary_upd) {
  return c->g.kv_format == VX_KV_FP8_E4M3
             ? launch_gqa_fp8_t<fp8_e4m3>(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s, pdl, budget, summary_upd)
             : launch_gqa_fp8_t<fp8_e5m2>(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s, pdl, budget, summary_upd);
}

}  // namespace vx
