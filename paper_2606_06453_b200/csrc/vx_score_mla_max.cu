// vx_score_mla_max.cu -- (a2) VX_AGG_MAX page scores for the MLA group: S[j] = max_h u[h, j],
// u[h, j] = sum_c max(q[h,c] * M[j,c], q[h,c] * m[j,c])   (PAPER.md:552 per-head envelope score; :556, :600, :628
// the max_h aggregation of the Quest-family flows).
//
// With 32 query heads sharing one latent head the per-head form costs 32 x the SUM form's arithmetic: too much for
// the CUDA cores at the summary stream's rate, so this is the one scoring path that is a dense contraction.  Since
// M >= m, max(q M, q m) = q+ M + q- m with q+ = max(q, 0), q- = min(q, 0) (both exact in bf16), hence
//     U[h, j] = [q-[h, :] | q+[h, :]] . [m[j, :] | M[j, :]]  =  A[h, 0:1152] . B[j, 0:1152],
// a [Hq x 1152] x [1152 x pages] GEMM whose B rows are the summary pool's rows as they lie in HBM.  It runs on the
// tensor cores with mma.sync m16n8k16 (bf16 in, fp32 accumulate): 74 flop per summary byte, ~0.5 PFLOP/s at the full
// HBM rate -- a memory-bound use of them, which is why the warp-level instruction (no TMEM / TMA staging) is enough.
//
// One CTA serves one request: it splits the request's queries by sign into A in shared memory (rows padded to
// 2,368 B so that a quarter-warp's 16-byte fragment loads cover all 32 banks once), then each warp takes 16-page
// chunks: per 32-wide k block a thread loads one 16-byte piece of each of its 2 page rows straight from global
// memory (8 rows x 64 contiguous bytes per warp instruction) and the A fragments for both 16-head tiles from shared
// memory.  The k order inside a block is permuted -- thread t owns elements 8t..8t+7 and feeds 8t..8t+3 to one
// mma and 8t+4..8t+7 to the next -- identically for A and B, which a dot product does not notice; it turns every
// fragment load into one 128-bit access.  The head maximum is taken over the accumulator rows in registers and by
// three shuffles; scores leave as fp32.  The page rows go global -> registers through a 6-deep register pipeline
// (loads of k blocks kb+1 .. kb+5 in flight under block kb's mma).
#include <cuda_bf16.h>

#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

namespace {
constexpr int kD = 576;                         // latent width (512 + 64 RoPE), "full fused-latent"
constexpr int kK = 2 * kD;                      // contraction length: [min | max] halves of a summary row
constexpr int kKBlocks = kK / 32;               // 36 blocks of 32
constexpr int kARowBytes = kK * 2 + 64;         // 2,368: consecutive rows start 64 B apart modulo 128
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / kWarp;
constexpr int kNT = 2;                          // n tiles of 8 pages per warp item
constexpr int kDepth = 6;                       // k blocks in the register pipeline (bytes in flight set the rate)
constexpr int kChunk = 8 * kNT;                 // pages per warp item

__device__ __forceinline__ uint4 ldg_stream_v4(const void* p) {
  uint4 v;
  asm("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                               uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
               "{%0, %1, %2, %3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
}  // namespace

template <int MT>                               // 16-head tiles: Hq = 16 * MT
__global__ void __launch_bounds__(kThreads, 2)
score_mla_max_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ summary,
                     const int32_t* __restrict__ page_indptr, const int32_t* __restrict__ page_indices,
                     float* __restrict__ scores, int req0) {
  extern __shared__ __align__(128) uint8_t s_a[];               // A[16 * MT][kARowBytes]
  constexpr int HQ = 16 * MT;
  const int i = blockIdx.y + req0;
  const int tid = threadIdx.x, lane = tid % kWarp, warp = tid / kWarp;
  const int g = lane >> 2, t = lane & 3;
  pdl_trigger();                                // the selection kernel may queue up behind us
  const int row0 = page_indptr[i], n_pages = page_indptr[i + 1] - row0;
  if (blockIdx.x * kWarps * kChunk >= n_pages) return;          // a short request needs fewer CTAs than the grid has

  // ---- A = [q- | q+] of this request's heads -------------------------------------------------------------------
  const __nv_bfloat16* qi = q + (int64_t)i * HQ * kD;
  // (8 elements per thread and step, all loads of a thread independent: the 36 KB of queries come from L2 once)
  constexpr int kVecs = HQ * kD / 8;
#pragma unroll
  for (int v0 = 0; v0 < kVecs; v0 += kThreads) {
    const int v = v0 + tid;
    if (v < kVecs) {
      const int h = v / (kD / 8), c = (v - h * (kD / 8)) * 8;
      const uint4 x = *reinterpret_cast<const uint4*>(qi + (size_t)v * 8);
      const uint32_t w[4] = {x.x, x.y, x.z, x.w};
      uint32_t neg[4], pos[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {             // bf16 pairs: the sign bit decides (-0.0 goes to q-, which adds 0 either way)
        const uint32_t m = ((w[e] & 0x00008000u) ? 0x0000FFFFu : 0u) | ((w[e] & 0x80000000u) ? 0xFFFF0000u : 0u);
        neg[e] = w[e] & m;
        pos[e] = w[e] & ~m;
      }
      uint8_t* row = s_a + (size_t)h * kARowBytes;
      *reinterpret_cast<uint4*>(row + c * 2) = make_uint4(neg[0], neg[1], neg[2], neg[3]);              // pairs with m
      *reinterpret_cast<uint4*>(row + (kD + c) * 2) = make_uint4(pos[0], pos[1], pos[2], pos[3]);       // pairs with M
    }
  }
  __syncthreads();

  const int n_chunks = (n_pages + kChunk - 1) / kChunk;
  for (int chunk = blockIdx.x * kWarps + warp; chunk < n_chunks; chunk += gridDim.x * kWarps) {
    const int j0 = chunk * kChunk;
    const uint8_t* brow[kNT];                   // my page row of each n tile (clamped: the tail repeats a valid page)
#pragma unroll
    for (int nt = 0; nt < kNT; ++nt) {
      const int j = min(j0 + nt * 8 + g, n_pages - 1);
      brow[nt] = reinterpret_cast<const uint8_t*>(summary + (int64_t)page_indices[row0 + j] * kK) + t * 16;
    }
    float acc[MT][kNT][4];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int nt = 0; nt < kNT; ++nt)
#pragma unroll
        for (int e = 0; e < 4; ++e) acc[mt][nt][e] = 0.f;
    const uint8_t* arow = s_a + (size_t)g * kARowBytes + t * 16;
    // register pipeline, kDepth k blocks deep: the loads of blocks kb + 1 .. kb + kDepth - 1 are in flight under block kb's mma
    uint4 b[kDepth][kNT];
    auto load_b = [&](uint4 (&dst)[kNT], int kb) {
      const int off = min(kb, kKBlocks - 1) * 64;               // (past the end: a harmless repeat of the last block)
#pragma unroll
      for (int nt = 0; nt < kNT; ++nt) dst[nt] = ldg_stream_v4(brow[nt] + off);
    };
    auto compute = [&](const uint4 (&bb)[kNT], int kb) {
#pragma unroll
      for (int mt = 0; mt < MT; ++mt) {
        const uint4 lo = *reinterpret_cast<const uint4*>(arow + (size_t)(mt * 16) * kARowBytes + kb * 64);      // head 16 mt + g
        const uint4 hi = *reinterpret_cast<const uint4*>(arow + (size_t)(mt * 16 + 8) * kARowBytes + kb * 64);  // head 16 mt + g + 8
#pragma unroll
        for (int nt = 0; nt < kNT; ++nt) {
          mma_bf16_16816(acc[mt][nt], lo.x, hi.x, lo.y, hi.y, bb[nt].x, bb[nt].y);
          mma_bf16_16816(acc[mt][nt], lo.z, hi.z, lo.w, hi.w, bb[nt].z, bb[nt].w);
        }
      }
    };
    static_assert(kKBlocks % kDepth == 0, "pipeline depth");
#pragma unroll
    for (int st = 0; st < kDepth - 1; ++st) load_b(b[st], st);
#pragma unroll 1
    for (int kb = 0; kb < kKBlocks; kb += kDepth) {
#pragma unroll
      for (int st = 0; st < kDepth; ++st) {
        load_b(b[(st + kDepth - 1) % kDepth], kb + st + kDepth - 1);
        compute(b[st], kb + st);
      }
    }
    // ---- max over the heads: accumulator rows g, g + 8 of every tile, then the 8 lanes that share t -----------
#pragma unroll
    for (int nt = 0; nt < kNT; ++nt) {
      float m0 = fmaxf(acc[0][nt][0], acc[0][nt][2]), m1 = fmaxf(acc[0][nt][1], acc[0][nt][3]);   // pages 2t, 2t + 1
#pragma unroll
      for (int mt = 1; mt < MT; ++mt) {
        m0 = fmaxf(m0, fmaxf(acc[mt][nt][0], acc[mt][nt][2]));
        m1 = fmaxf(m1, fmaxf(acc[mt][nt][1], acc[mt][nt][3]));
      }
#pragma unroll
      for (int o = 4; o < kWarp; o <<= 1) {
        m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, o));
        m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, o));
      }
      if (g == 0) {
        const int j = j0 + nt * 8 + 2 * t;
        if (j < n_pages) scores[row0 + j] = m0;
        if (j + 1 < n_pages) scores[row0 + j + 1] = m1;
      }
    }
  }
}

bool score_mla_max_supported(const vx_geom& g) {
  return g.kv_shared && g.num_kv_heads == 1 && g.agg == VX_AGG_MAX && g.summary_kind == VX_SUMMARY_ENVELOPE &&
         g.dtype == VX_DT_BF16 && g.qk_dim == kD && (g.num_q_heads == 16 || g.num_q_heads == 32);
}

template <int MT>
static cudaError_t launch_mt(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt, float* scores,
                             cudaStream_t s, const ReqRange& rr) {
  constexpr int smem = 16 * MT * kARowBytes;
  if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(score_mla_max_kernel<MT>), c->device, smem)) return e;
  const int n_req = rr.count < 0 ? pt.batch : rr.count;
  // CTAs per request: enough warps for the longest request's chunks, capped at ~2 resident CTAs per SM over the batch
  // (one chunk per warp whatever the batch -- 512 CTAs on C4 -- measured 35.0 us against 32.5: every CTA rebuilds A);
  // CTAs beyond a shorter request's chunks leave at once
  const int chunks = (pt.max_pages_per_req + kChunk - 1) / kChunk;
  int per_req = (chunks + kWarps - 1) / kWarps;
  const int cap = (2 * c->num_sms + n_req - 1) / n_req;
  if (per_req > cap) per_req = cap;
  if (per_req < 1) per_req = 1;
  score_mla_max_kernel<MT><<<dim3(per_req, n_req), kThreads, smem, s>>>(
      static_cast<const __nv_bfloat16*>(q), static_cast<const __nv_bfloat16*>(summary), pt.page_indptr, pt.page_indices,
      scores, rr.begin);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_score_mla_max(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt, float* scores,
                                 cudaStream_t s, const ReqRange& rr) {
  return c->g.num_q_heads == 32 ? launch_mt<2>(c, q, summary, pt, scores, s, rr)
                                : launch_mt<1>(c, q, summary, pt, scores, s, rr);
}

}  // namespace vx
