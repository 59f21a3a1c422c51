// vx_decode_gqa.cu -- (a4) sparse paged decode for bf16 GQA (page 16, d = dv in {64, 128}, group <= 8).
// PAPER.md:92 Eq.4 over the tokens of the selected pages, reached through the sparse block table (:200);
// split along pages with an LSE merge (:75).
//
// HBM-bound gather: per selected (page, KV head) one contiguous 16 x d K chunk and one V chunk
// (4 KB each at d = 128).  Every warp streams its own pages through a private 3-stage cp.async
// ring in shared memory (16-byte LDGSTS, XOR-swizzled so ldmatrix is bank-conflict free), so no
// block-wide barrier sits in the loop and 2 pages (16 KB) per warp are always in flight.
// The contractions are skinny: S^T[16 tokens x 8 heads] = K Q^T and O^T[d x 8 heads] = V^T P^T.
// They run as m16n8k16 bf16 MMAs with fp32 accumulation (tokens / channels on M, the query heads
// of the group on N = 8), which keeps the instruction stream ~8x below the CUDA-core formulation
// and the kernel on the bandwidth roofline; the softmax (exp2, running max / sum) is fp32 in
// registers, P is rounded to bf16 for the second MMA.
// The splits of a (request, KV head) merge in-kernel: the last split CTA to arrive (a self-resetting
// atomic counter) merges the partials by LSE.  In the fused step the warp that stages the request's
// newest page also rebuilds that page's summary (min / max, or the block top-k centroid) from shared
// memory (a1): the newest page is a forced local page, so no separate launch is needed.
#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

constexpr int kGqaWarps = 4;
constexpr int kGqaStages = 3;
constexpr int kGqaPage = 16;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

__device__ __forceinline__ void ldmatrix_x4(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t x) {
  uint32_t y;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(y) : "r"(x));
  return y;
}
// D(16x8, fp32) += A(16x16, bf16 row) * B(16x8, bf16 col)
__device__ __forceinline__ void mma_bf16(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}
// 16-byte async copy that writes zeros when !valid (src-size 0)
// (with an L2 cache policy: the selected pages are read once -- evict-first, so that they leave the small hot arrays alone)
__device__ __forceinline__ void cp_async16_zfill(uint32_t dst, const void* src, bool valid, uint64_t pol) {
  asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2, %3;" ::"r"(dst), "l"(src), "r"(valid ? 16 : 0), "l"(pol));
}

template <int D, bool CL>
__global__ void __launch_bounds__(kGqaWarps * kWarp)
decode_gqa_mma_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ kpool,
                      const __nv_bfloat16* __restrict__ vpool, int64_t stride_page, int64_t stride_token,
                      int64_t stride_head, int num_q_heads, int num_kv_heads, float scale_log2,
                      const int32_t* __restrict__ seq_lens, const int32_t* __restrict__ sel_phys,
                      const int32_t* __restrict__ sel_logical, const int32_t* __restrict__ sel_count,
                      int max_budget, int num_splits, float* __restrict__ part_o, float* __restrict__ part_lse,
                      int* __restrict__ unit_counter, __nv_bfloat16* __restrict__ summary_upd, int summary_kind,
                      __nv_bfloat16* __restrict__ out, float* __restrict__ lse_out, int req0,
                      const int32_t* __restrict__ budget_opt, int bpp, int stream_once) {
  constexpr int ROWB = D * 2;                 // bytes per token row
  constexpr int CH = ROWB / 16;               // 16-byte chunks per row
  constexpr int PAGEB = kGqaPage * ROWB;      // bytes of one K (or V) page chunk
  constexpr int KS = D / 16;                  // k-steps of QK^T = m-tiles of PV
  constexpr int CP_ITERS = kGqaPage * CH / kWarp;
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ float s_m[kGqaWarps][8], s_l[kGqaWarps][8];
  __shared__ float s_hinv[8], s_hlse[8];           // per head of the group: 1 / denominator and LSE of this CTA's pages
  __shared__ int s_valid[kGqaWarps][kGqaStages];   // valid tokens of the page staged in each slot (bit 8: newest page)
  __shared__ int s_phys[kGqaWarps][kGqaStages];    // its physical id
  __shared__ int s_last;

  const int split = blockIdx.x, kvh = blockIdx.y, i = blockIdx.z + req0;
  const int warp = threadIdx.x / kWarp, lane = threadIdx.x % kWarp;
  [[maybe_unused]] const int cta = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
  if (threadIdx.x == 0) { VX_TRACE_STAMP(cta, 0); VX_TRACE_SMID(cta); }
  const int grp = num_q_heads / num_kv_heads;
  const int n_tok = seq_lens[i];
  const int newest_page = (n_tok - 1) / kGqaPage;
  const int cnt_known = budget_opt ? max(0, min(min(budget_opt[i], max_budget), newest_page + 1)) : -1;

  // Q^T as the B operand: qb[ks] = Q[head lane/4][16*ks + 2*(lane%4) + {0,1}], [.. + 8 ..]
  uint32_t qb[KS][2];
  {
    const int h = lane / 4;
    const __nv_bfloat16* qrow = q + ((int64_t)i * num_q_heads + kvh * grp + h) * D;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      const int c = ks * 16 + 2 * (lane % 4);
      qb[ks][0] = h < grp ? *reinterpret_cast<const uint32_t*>(qrow + c) : 0u;
      qb[ks][1] = h < grp ? *reinterpret_cast<const uint32_t*>(qrow + c + 8) : 0u;
    }
  }
  if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 1);
  pdl_wait();                                   // the selection lists come from the preceding kernel of the step
  if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 2);

  const int cnt = cnt_known >= 0 ? cnt_known : sel_count[i * num_kv_heads + kvh];
  const int per_split = (cnt + num_splits - 1) / num_splits;
  const int r_begin = min(split * per_split, cnt), r_end = min(r_begin + per_split, cnt);
  const int32_t* phys_list = sel_phys + ((int64_t)i * num_kv_heads + kvh) * max_budget;
  const int32_t* log_list = sel_logical + ((int64_t)i * num_kv_heads + kvh) * max_budget;
  // this warp's pages: r_begin + warp, + kGqaWarps, ...
  const int my_pages = r_end - r_begin > warp ? (r_end - r_begin - warp + kGqaWarps - 1) / kGqaWarps : 0;

  uint8_t* ring = smem + (size_t)warp * kGqaStages * 2 * PAGEB;
  const uint32_t ring_u32 = smem_u32(ring);

  const uint64_t pol = l2_stream_policy(stream_once != 0);
  int id_phys = 0, id_valid = 0;                // lane j: this warp's (base + j)-th page
  auto fetch_ids = [&](int base) {
    const int p = base + lane;
    if (p < my_pages) {
      const int r = r_begin + warp + p * kGqaWarps;
      id_phys = phys_list[r];
      const int lg = log_list[r];
      id_valid = min(kGqaPage, n_tok - lg * kGqaPage) | (lg == newest_page ? 256 : 0);
    }
  };
  auto issue = [&](int p) {                     // all lanes: copy page p of this warp into slot p % stages
    const int phys = __shfl_sync(0xffffffffu, id_phys, p & 31);
    const int valid = __shfl_sync(0xffffffffu, id_valid, p & 31);
    const int64_t base = pool_block_base(phys, stride_page, bpp, kGqaPage * stride_token) + (int64_t)kvh * stride_head;
    const uint32_t dst = ring_u32 + (uint32_t)(p % kGqaStages) * 2 * PAGEB;
    if (lane == 0) { s_valid[warp][p % kGqaStages] = valid; s_phys[warp][p % kGqaStages] = phys; }
    const int nv = valid & 255;
#pragma unroll
    for (int it = 0; it < CP_ITERS; ++it) {
      const int x = it * kWarp + lane;
      const int t = x / CH, c = x % CH;
      const uint32_t off = t * ROWB + ((c ^ (t & 7)) * 16);
      const int64_t src = base + (int64_t)t * stride_token + c * 8;
      cp_async16_zfill(dst + off, kpool + src, t < nv, pol);
      cp_async16_zfill(dst + PAGEB + off, vpool + src, t < nv, pol);
    }
  };

  float o[KS][4];
#pragma unroll
  for (int mt = 0; mt < KS; ++mt) { o[mt][0] = o[mt][1] = o[mt][2] = o[mt][3] = 0.f; }
  float m_a = -INFINITY, m_b = -INFINITY, l_a = 0.f, l_b = 0.f;   // heads 2*(lane%4), +1

  fetch_ids(0);
#pragma unroll
  for (int p = 0; p < kGqaStages - 1; ++p) {
    if (p < my_pages) issue(p);
    cp_async_commit();
  }
  if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 3);

  for (int p = 0; p < my_pages; ++p) {
    cp_async_wait<kGqaStages - 2>();            // page p has landed (this lane's copies)
    __syncwarp();
    if (threadIdx.x == 0 && p == 0) VX_TRACE_STAMP(cta, 4);
    if (threadIdx.x == 0 && p == my_pages - 1) VX_TRACE_STAMP(cta, 5);                               // ... and every lane's; also: all lanes are done with page p-1
    const int valid_enc = s_valid[warp][p % kGqaStages];
    const int valid = valid_enc & 255;
    const int phys_p = s_phys[warp][p % kGqaStages];
    {
      const int nxt = p + kGqaStages - 1;       // refill the slot page p-1 used
      if ((nxt & 31) == 0 && nxt < my_pages) fetch_ids(nxt);   // ids of pages nxt .. nxt+31 (p's were read above)
      if (nxt < my_pages) issue(nxt);
      cp_async_commit();
    }
    const uint32_t kst = ring_u32 + (uint32_t)(p % kGqaStages) * 2 * PAGEB, vst = kst + PAGEB;

    if (summary_upd != nullptr && (valid_enc & 256)) {
      // (a1) this is the request's newest page: rebuild its min / max summary from the staged keys
      // (exact in bf16).  Lane owns W consecutive 32-bit words (2 channels each) of the row.
      constexpr int W = ROWB / 128;
      const int byte0 = lane * W * 4, c = byte0 / 16, o16 = byte0 % 16;
      if (summary_kind == VX_SUMMARY_CENTROID) {   // block top-k: exact mean of the valid keys, one rounding (Eq.1)
        double sum[2 * W];
#pragma unroll
        for (int w = 0; w < 2 * W; ++w) sum[w] = 0.0;
        for (int t = 0; t < valid; ++t) {
#pragma unroll
          for (int w = 0; w < W; ++w) {
            const uint32_t x = *reinterpret_cast<const uint32_t*>(ring + (size_t)(p % kGqaStages) * 2 * PAGEB + t * ROWB +
                                                                  ((c ^ (t & 7)) * 16) + o16 + w * 4);
            sum[2 * w] += (double)__uint_as_float(x << 16);
            sum[2 * w + 1] += (double)__uint_as_float(x & 0xffff0000u);
          }
        }
        __nv_bfloat16* dstc = summary_upd + ((int64_t)phys_p * num_kv_heads + kvh) * D + lane * W * 2;
#pragma unroll
        for (int w = 0; w < 2 * W; ++w) dstc[w] = round_double<__nv_bfloat16>(sum[w] / (double)valid);
      } else {
      __nv_bfloat162 lo[W], hi[W];
#pragma unroll
      for (int w = 0; w < W; ++w) {
        const uint32_t x = *reinterpret_cast<const uint32_t*>(ring + (size_t)(p % kGqaStages) * 2 * PAGEB + o16 + w * 4 + (c * 16));
        lo[w] = hi[w] = *reinterpret_cast<const __nv_bfloat162*>(&x);       // token 0 (c ^ 0 = c)
      }
      for (int t = 1; t < valid; ++t) {
#pragma unroll
        for (int w = 0; w < W; ++w) {
          const uint32_t x = *reinterpret_cast<const uint32_t*>(ring + (size_t)(p % kGqaStages) * 2 * PAGEB + t * ROWB +
                                                                ((c ^ (t & 7)) * 16) + o16 + w * 4);
          const __nv_bfloat162 v = *reinterpret_cast<const __nv_bfloat162*>(&x);
          lo[w] = __hmin2(lo[w], v);
          hi[w] = __hmax2(hi[w], v);
        }
      }
      __nv_bfloat16* dst = summary_upd + (((int64_t)phys_p * num_kv_heads + kvh) * 2) * D + lane * W * 2;
#pragma unroll
      for (int w = 0; w < W; ++w) {
        *reinterpret_cast<__nv_bfloat162*>(dst + 2 * w) = lo[w];
        *reinterpret_cast<__nv_bfloat162*>(dst + D + 2 * w) = hi[w];
      }
      }
    }

    // S^T[16 tokens x 8 heads] = K[16 x D] . Q^T
    float s[4] = {0.f, 0.f, 0.f, 0.f};
    {
      const int j = lane / 8, r = lane % 8;
      const int t = (j & 1) * 8 + r;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        uint32_t a[4];
        const int c = 2 * ks + (j >> 1);
        ldmatrix_x4(a, kst + t * ROWB + ((c ^ (t & 7)) * 16));
        mma_bf16(s, a, qb[ks][0], qb[ks][1]);
      }
    }
    // online softmax, base 2.  s[0],s[1]: token lane/4, heads a,b;  s[2],s[3]: token lane/4 + 8
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
    const uint32_t pb_lo = movmatrix_trans(pack_bf16x2(pa0, pb0));
    const uint32_t pb_hi = movmatrix_trans(pack_bf16x2(pa1, pb1));

    // O^T[D x 8 heads] = O^T * alpha + V^T[D x 16 tokens] . P
    {
      const int j = lane / 8, r = lane % 8;
      const int t = (j >> 1) * 8 + r;
#pragma unroll
      for (int mt = 0; mt < KS; ++mt) {
        uint32_t a[4];
        const int c = 2 * mt + (j & 1);
        ldmatrix_x4_trans(a, vst + t * ROWB + ((c ^ (t & 7)) * 16));
        o[mt][0] *= al_a; o[mt][1] *= al_b; o[mt][2] *= al_a; o[mt][3] *= al_b;
        mma_bf16(o[mt], a, pb_lo, pb_hi);
      }
    }
  }
  cp_async_wait<0>();
  pdl_trigger();
  if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 6);

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
  if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 7);
  const int ha = 2 * (lane % 4);
  float mb_a = -INFINITY, mb_b = -INFINITY;
#pragma unroll
  for (int w = 0; w < kGqaWarps; ++w) { mb_a = fmaxf(mb_a, s_m[w][ha]); mb_b = fmaxf(mb_b, s_m[w][ha + 1]); }
  const float f_a = m_a == -INFINITY ? 0.f : exp2f(m_a - mb_a), f_b = m_b == -INFINITY ? 0.f : exp2f(m_b - mb_b);
  float* so = reinterpret_cast<float*>(ring);   // [D][8 heads] fp32 = D * 32 bytes <= one stage
  // cluster merge: this CTA's normalised partial [8 heads][D] + 8 lse, in warp 0's second stage (nobody's `so`)
  [[maybe_unused]] float* cl_part = reinterpret_cast<float*>(smem + 2 * PAGEB);
#pragma unroll
  for (int mt = 0; mt < KS; ++mt) {
    const int d0 = mt * 16 + lane / 4;
    *reinterpret_cast<float2*>(so + d0 * 8 + ha) = make_float2(o[mt][0] * f_a, o[mt][1] * f_b);
    *reinterpret_cast<float2*>(so + (d0 + 8) * 8 + ha) = make_float2(o[mt][2] * f_a, o[mt][3] * f_b);
  }
  if (threadIdx.x < 8) {                        // per head, once: the CTA's reference, 1 / denominator and LSE
    const int h = threadIdx.x;
    float mb = -INFINITY;
#pragma unroll
    for (int w = 0; w < kGqaWarps; ++w) mb = fmaxf(mb, s_m[w][h]);
    float lsum = 0.f;
#pragma unroll
    for (int w = 0; w < kGqaWarps; ++w) lsum += s_m[w][h] == -INFINITY ? 0.f : s_l[w][h] * exp2f(s_m[w][h] - mb);
    s_hinv[h] = lsum > 0.f ? 1.f / lsum : 0.f;
    s_hlse[h] = lsum > 0.f ? (mb + log2f(lsum)) * kLn2 : -INFINITY;
  }
  __syncthreads();
  // four heads of one channel per thread: one 16-byte read per warp partial
  for (int e = threadIdx.x; e < ((grp + 3) / 4) * D; e += kGqaWarps * kWarp) {
    const int d = e % D, h0 = 4 * (e / D);
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int w = 0; w < kGqaWarps; ++w) {
      const float4 v = *reinterpret_cast<const float4*>(smem + (size_t)w * kGqaStages * 2 * PAGEB + (d * 8 + h0) * 4);
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
        } else if constexpr (CL) {              // this split's partial stays in shared memory for the cluster merge
          cl_part[h * D + d] = val;
          if (d == 0) cl_part[8 * D + h] = s_hlse[h];
        } else {
          part_o[(head_row * num_splits + split) * D + d] = val;
          if (d == 0) part_lse[head_row * num_splits + split] = s_hlse[h];
        }
      }
    }
  }
  if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 8);
  if constexpr (CL) {
    // (a5) the splits of this (request, KV head) are the CTAs of one thread-block cluster: every CTA merges a slice of
    // the group's output rows out of its peers' shared memory; no partials in HBM, no counter, no fence
    cluster_sync();
    if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 9);
    cluster_merge_partials(cl_part, D, grp, split, num_splits, (int64_t)i * num_q_heads + kvh * grp, out, lse_out);
    if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 10);
    cluster_sync_relaxed();                       // no CTA leaves while a peer still reads its partial
  } else if (num_splits > 1) {                  // (a5) the last split of this (request, KV head) merges by LSE
    if (last_split_arrives(unit_counter + i * num_kv_heads + kvh, num_splits, &s_last)) {
      if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 9);
      merge_partials<__nv_bfloat16>(part_o, part_lse, (int64_t)i * num_q_heads + kvh * grp, grp, num_splits, D, out, lse_out,
                                     reinterpret_cast<float*>(smem));
      if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 10);
    }
  }
  if (threadIdx.x == 0) VX_TRACE_STAMP(cta, 11);
}

VX_TRACE_SETTER(vx_trace_set_decode_gqa)

bool gqa_mma_supported(const vx_geom& g) {
  const int grp = g.num_q_heads / g.num_kv_heads;
  return g.dtype == VX_DT_BF16 && g.kv_format == VX_KV_SAME && !g.kv_shared && g.page_size == kGqaPage && g.qk_dim == g.v_dim &&
         (g.qk_dim == 128 || g.qk_dim == 64) && grp <= 8;
}

template <int D>
static cudaError_t launch_gqa_mma_t(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                    const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                    int32_t max_budget, void* out, float* lse, cudaStream_t s, const DecodeOpts& opt) {
  const vx_geom& g = c->g;
  constexpr int smem = kGqaWarps * kGqaStages * 2 * kGqaPage * D * 2;
  if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(decode_gqa_mma_kernel<D, false>), c->device, smem)) return e;
  if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(decode_gqa_mma_kernel<D, true>), c->device, smem)) return e;
  // splits: whole waves of equal CTAs.  cost(sp) = waves x (pages per warp + ~3 pages of pipeline fill)
  const int n_req = opt.rr.count < 0 ? pt.batch : opt.rr.count;
  const int splits = decode_gqa_splits(c, n_req, max_budget);
  dim3 grid(splits, g.num_kv_heads, n_req);
  // 2, 4 or 8 splits: one thread-block cluster per (request, KV head), merged over distributed shared memory
  const bool cl = splits == 2 || splits == 4 || splits == 8;
  cudaError_t e = launch_kernel_cluster(cl ? decode_gqa_mma_kernel<D, true> : decode_gqa_mma_kernel<D, false>, grid,
      dim3(kGqaWarps * kWarp), (size_t)smem, s, opt.pdl, cl ? splits : 1,
      static_cast<const __nv_bfloat16*>(q), static_cast<const __nv_bfloat16*>(pool.k),
      static_cast<const __nv_bfloat16*>(pool.v), pool.stride_page, pool.stride_token, pool.stride_head,
      g.num_q_heads, g.num_kv_heads, g.sm_scale * kLog2e, pt.seq_lens, sel_phys, sel_logical, sel_count, max_budget,
      splits, c->ws.part_o, c->ws.part_lse, c->ws.unit_counter, static_cast<__nv_bfloat16*>(opt.summary_upd), g.summary_kind,
      static_cast<__nv_bfloat16*>(out), lse, opt.rr.begin, opt.budget, c->bpp,
      l2_stream_once(c, (int64_t)n_req * g.num_kv_heads * max_budget * 2 * kGqaPage * D * 2) ? 1 : 0);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

int decode_gqa_splits(const vx_ctx* c, int n_req, int max_budget) {
  const int units = n_req * c->g.num_kv_heads;
  const int cta_smem = kGqaWarps * kGqaStages * 2 * kGqaPage * c->g.qk_dim * 2 + 1024;   // ring + static / reserved
  const int slots = c->num_sms * (227 * 1024 / cta_smem > 0 ? 227 * 1024 / cta_smem : 1);    // resident CTAs
  int splits = 1, best_cost = 1 << 30;
  for (int sp = 1; sp <= kMaxSplits && sp <= max_budget; ++sp) {
    const int waves = (units * sp + slots - 1) / slots;
    const int cost = waves * (((max_budget + sp - 1) / sp + kGqaWarps - 1) / kGqaWarps + 3);
    if (cost < best_cost) { best_cost = cost; splits = sp; }
  }
  return splits;
}

bool decode_folds_summary(const vx_ctx* c) { return (gqa_mma_supported(c->g) || mla_tc_supported(c->g) || gqa_fp8_fast_supported(c->g)); }

cudaError_t launch_decode_gqa_mma(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                  const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                  int32_t max_budget, void* out, float* lse, cudaStream_t s, const DecodeOpts& opt) {
  if (c->g.qk_dim == 128)
    return launch_gqa_mma_t<128>(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s, opt);
  return launch_gqa_mma_t<64>(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s, opt);
}

}  // namespace vx
