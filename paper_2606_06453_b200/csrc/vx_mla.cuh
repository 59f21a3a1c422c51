// vx_mla.cuh -- what the two MLA kernels share: the geometry / shared-memory layout constants, the tcgen05 / TMA / mbarrier
// wrappers, and the two split merges (global partials + last arriver; thread-block cluster over distributed shared memory).
//   vx_decode_mla.cu   (a4)+(a5): sparse paged decode over a given block table (vx_sparse_paged_decode)
//   vx_step_mla.cu     (a2)->(a3)->(a4)->(a5) of a request in one kernel on the cluster that owns it (vx_sparse_decode_step)
#pragma once
#include <cuda.h>

#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

namespace mla {
constexpr int D = 576, DV = 512, PAGE = 64, NH = 32;      // geometry this kernel is built for
constexpr int THREADS = 256;                              // fused step: TMA producer, QK issuer, 4 epilogue warps (one = softmax), PV issuer, one spare
                                                          // (8 warps: its selection wants a divisor of 2,048 bins, its summary stream 7 warps)
constexpr int THREADS_DECODE = 224;                       // the separate decode call: the 7 warps of the loop (an idle eighth warp measured +2.5 us on C4)
constexpr int PV_WARP = 6;
constexpr int PAGE_BYTES = PAGE * D * 2;                  // 73728
constexpr int SOFTMAX_THREADS = 128;
constexpr int SOFTMAX_WARP = 4;                           // warp % 4 == 0: TMEM lanes 0..31
constexpr int CHUNKS = D * 2 / 16;                        // 72 16-byte chunks per token row
constexpr int ATOMS = CHUNKS / 8;                         // 9 swizzle atoms (64 channels each)
constexpr int K_ATOM_BYTES = PAGE * 128;                  // 8192: 64 rows x 128 B
constexpr int PAIR_BYTES = 2 * K_ATOM_BYTES;              // 16384: 128 value channels
constexpr int P_BYTES = NH * 128;                         // 4096: [32 heads][64 tokens] bf16
constexpr int N_PAIR = 12, N_ROPE = 3;                    // ring slots: 3 pages
constexpr int PAIRS_PER_PAGE = DV / 128;                  // 4
constexpr int OFF_P = 0;
constexpr int OFF_PAIR = OFF_P + 2 * P_BYTES;             // 8192
constexpr int OFF_ROPE = OFF_PAIR + N_PAIR * PAIR_BYTES;  // 204800
constexpr int SMEM_BYTES = OFF_ROPE + N_ROPE * K_ATOM_BYTES;   // 229376 of dynamic shared memory, declared 1024-byte aligned (fused step)
constexpr int SMEM_BYTES_DECODE = SMEM_BYTES + 1024;          // the separate decode call aligns by hand inside its allocation
// The fused step's front end (score + select) lives in the same shared memory before the first page arrives:
//   [OFF_P, +4608)                          the query vector [Qm | Qp] fp32 (the P buffers are free until the loop)
//   [OFF_PAIR + (k * F_WARPS + w) * F_STAGE_BYTES, ..)  slot k of stream warp w's private ring of summary stages (F_PG rows
//                                           each); the area of the LAST slot group first holds the staged Q rows
//   [SMEM_BYTES - 8 p_cap, SMEM_BYTES)      fp32 scores (later the keys) and physical page ids of the request's pages
constexpr int F_PG = 4;                                   // summary rows per stage
constexpr int F_WARPS = THREADS / kWarp - 1;              // stream warps 1..7, each its own producer and consumer
constexpr int F_SLOTS_MAX = 3;                            // stages per warp: 7 x 3 x 9 KB = 193 KB in flight
constexpr int F_MAX_ROW_BYTES = 2 * D * 2;                // envelope row [min | max]: 2,304 B (centroid: 1,152 B)
constexpr int F_STAGE_BYTES = F_PG * F_MAX_ROW_BYTES;     // 9216
constexpr int F_Q_PITCH = D * 2 + 16;                     // Q staging row pitch (bank spread)
constexpr int OFF_F_QVEC = OFF_P;
constexpr int F_MAX_PAGES = 8192;                         // pages per request: leaves 2 slots per warp beside scores + ids
constexpr int F_MAX_LIST = 64;                            // selected pages per CTA (its split's share of the block table)
static_assert((SMEM_BYTES - 8 * F_MAX_PAGES - OFF_PAIR) / (F_WARPS * F_STAGE_BYTES) >= 2 && F_WARPS * F_STAGE_BYTES >= NH * F_Q_PITCH,
              "fused front-end layout: at least 2 slots per stream warp, the staged Q rows fit one slot group");
constexpr int TMEM_COLS = 512;
constexpr int TM_Q = 0;                                   // Q[head = lane][576 bf16] as 288 32-bit columns (A operand of S)
constexpr int TM_S = 320;                                 // S[head][64 tokens]
constexpr int TM_O = 384;                                 // O^T block mb: [384 + 32mb, +32)
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kRescaleThreshold = 8.f;                  // log2 units

// instruction descriptors (kind::f16): D fp32, A/B bf16
constexpr uint32_t IDESC_QK = (1u << 4) | (1u << 7) | (1u << 10) | ((64u >> 3) << 17) | ((128u >> 4) << 24);   // M128 N64
constexpr uint32_t IDESC_PV = (1u << 4) | (1u << 7) | (1u << 10) | (1u << 15) | ((NH >> 3) << 17) | ((128u >> 4) << 24);

// shared-memory matrix descriptor, 128-byte swizzle, Blackwell version bit
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
         ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | (1ull << 46) | (2ull << 61);
}
__device__ __forceinline__ void umma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, bool accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"((uint32_t)accumulate));
}
// same with the A operand in tensor memory (32-bit columns, two bf16 along K per column)
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, bool accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"((uint32_t)accumulate));
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
      ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_async_proxy() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// 32 consecutive TMEM columns of this thread's lane -> registers / back
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const float (&v)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
      "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
      ::"r"(taddr), "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])),
        "r"(__float_as_uint(v[3])), "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])),
        "r"(__float_as_uint(v[7])), "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])),
        "r"(__float_as_uint(v[11])), "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])),
        "r"(__float_as_uint(v[15])), "r"(__float_as_uint(v[16])), "r"(__float_as_uint(v[17])), "r"(__float_as_uint(v[18])),
        "r"(__float_as_uint(v[19])), "r"(__float_as_uint(v[20])), "r"(__float_as_uint(v[21])), "r"(__float_as_uint(v[22])),
        "r"(__float_as_uint(v[23])), "r"(__float_as_uint(v[24])), "r"(__float_as_uint(v[25])), "r"(__float_as_uint(v[26])),
        "r"(__float_as_uint(v[27])), "r"(__float_as_uint(v[28])), "r"(__float_as_uint(v[29])), "r"(__float_as_uint(v[30])),
        "r"(__float_as_uint(v[31]))
      : "memory");
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// one [64 channels x 64 tokens] box of page `page` -> 8 KB of 128-byte-swizzled shared memory
__device__ __forceinline__ void tma_box(uint32_t dst, const CUtensorMap* map, int channel0, int page, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst), "l"(map), "r"(channel0), "r"(0), "r"(page), "r"(bar) : "memory");
}
// one lane of a converged warp; ptxas then feeds tcgen05 / TMA operands straight from that lane (no per-lane loop)
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {   // non-blocking
  uint32_t ok;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ void softmax_barrier() { asm volatile("bar.sync 1, %0;" ::"n"(SOFTMAX_THREADS) : "memory"); }

// barrier indices
constexpr int B_PAGE_FULL = 0, B_PAIR_EMPTY = N_ROPE, B_ROPE_EMPTY = B_PAIR_EMPTY + N_PAIR,
              B_S_FULL = B_ROPE_EMPTY + N_ROPE, B_S_EMPTY = B_S_FULL + 1, B_P_FULL = B_S_EMPTY + 1,
              B_PV_DONE = B_P_FULL + 2, B_DECIDE = B_PV_DONE + 2, B_ACK = B_DECIDE + 2, N_BARS = B_ACK + 2;
}  // namespace mla

// (a5) LSE merge of the splits of request i, run by the last split CTA to arrive.
// Partials are [request][split][channel][head] fp32; the merged tile is transposed through shared memory so that
// the bf16 output rows [head][channel] are written with coalesced 16-byte stores.
__device__ __forceinline__ void merge_splits(const float* part_o, const float* part_lse, int i, int num_q_heads,
                                             int n_part, __nv_bfloat16* out, float* lse, uint8_t* scratch) {
  using namespace mla;
  constexpr int PITCH = DV * 2 + 16;                    // bf16 row pitch of the staged tile (bank spread)
  float* s_w = reinterpret_cast<float*>(scratch);       // [n_part][NH] split weights
  uint8_t* tile = scratch + kMaxSplits * NH * 4;
  const int64_t row0 = (int64_t)i * num_q_heads;
  for (int e = threadIdx.x; e < num_q_heads * n_part; e += blockDim.x)      // all lse values in one round trip
    s_w[(e % n_part) * NH + e / n_part] = ldcg_f32(part_lse + row0 * n_part + e);
  __syncthreads();
  if (threadIdx.x < NH) {
    const int j = threadIdx.x;
    if (j < num_q_heads) {
      float mx = -INFINITY;
      for (int s = 0; s < n_part; ++s) mx = fmaxf(mx, s_w[s * NH + j]);
      float z = 0.f;
      for (int s = 0; s < n_part; ++s) z += mx == -INFINITY ? 0.f : __expf(s_w[s * NH + j] - mx);
      const float inv = z > 0.f ? 1.f / z : 0.f;
      for (int s = 0; s < n_part; ++s) s_w[s * NH + j] = mx == -INFINITY ? 0.f : __expf(s_w[s * NH + j] - mx) * inv;
      if (lse != nullptr) lse[row0 + j] = z > 0.f ? mx + logf(z) : -INFINITY;
    } else {
      for (int s = 0; s < n_part; ++s) s_w[s * NH + j] = 0.f;
    }
  }
  __syncthreads();
  const float* src0 = part_o + (int64_t)i * n_part * DV * NH;
  constexpr int N_E = DV * (NH / 4), UNR = 8;           // e -> (channel d, heads j4 .. j4+3); UNR x n_part loads in flight
  auto put = [&](int e, float4 o) {
    const int d = e / (NH / 4), j4 = (e % (NH / 4)) * 4;
    *reinterpret_cast<__nv_bfloat16*>(tile + (j4 + 0) * PITCH + d * 2) = __float2bfloat16_rn(o.x);
    *reinterpret_cast<__nv_bfloat16*>(tile + (j4 + 1) * PITCH + d * 2) = __float2bfloat16_rn(o.y);
    *reinterpret_cast<__nv_bfloat16*>(tile + (j4 + 2) * PITCH + d * 2) = __float2bfloat16_rn(o.z);
    *reinterpret_cast<__nv_bfloat16*>(tile + (j4 + 3) * PITCH + d * 2) = __float2bfloat16_rn(o.w);
  };
  for (int e0 = threadIdx.x; e0 < N_E; e0 += UNR * blockDim.x) {
    float4 acc[UNR];
#pragma unroll
    for (int k = 0; k < UNR; ++k) acc[k] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s0 = 0; s0 < n_part; s0 += 2) {            // two splits at a time: 2 * UNR independent 16-byte L2 reads
      const bool two = s0 + 1 < n_part;
      float4 va[UNR], vb[UNR];
#pragma unroll
      for (int k = 0; k < UNR; ++k) {
        const int e = e0 + k * blockDim.x;
        const bool ok = e < N_E;
        va[k] = ok ? ldcg_f32x4(src0 + (int64_t)s0 * DV * NH + e * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
        vb[k] = ok && two ? ldcg_f32x4(src0 + (int64_t)(s0 + 1) * DV * NH + e * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int k = 0; k < UNR; ++k) {
        const int j4 = ((e0 + k * blockDim.x) % (NH / 4)) * 4;
        const float4 wa = *reinterpret_cast<const float4*>(s_w + s0 * NH + j4);
        const float4 wb = two ? *reinterpret_cast<const float4*>(s_w + (s0 + 1) * NH + j4) : make_float4(0.f, 0.f, 0.f, 0.f);
        acc[k].x += wa.x * va[k].x + wb.x * vb[k].x;
        acc[k].y += wa.y * va[k].y + wb.y * vb[k].y;
        acc[k].z += wa.z * va[k].z + wb.z * vb[k].z;
        acc[k].w += wa.w * va[k].w + wb.w * vb[k].w;
      }
    }
#pragma unroll
    for (int k = 0; k < UNR; ++k)
      if (e0 + k * blockDim.x < N_E) put(e0 + k * blockDim.x, acc[k]);
  }
  __syncthreads();
  for (int e = threadIdx.x; e < num_q_heads * (DV / 8); e += blockDim.x) {   // 16 bytes per thread, rows contiguous
    const int j = e / (DV / 8), c = e % (DV / 8);
    *reinterpret_cast<uint4*>(out + (row0 + j) * DV + c * 8) = *reinterpret_cast<const uint4*>(tile + j * PITCH + c * 16);
  }
}

// (a5) LSE merge inside a thread-block cluster: the splits of a request are the CTAs of one cluster (rank = split).
// Every CTA leaves its normalised partial O [channel][head] fp32 (64 KB, 16-byte columns XOR-swizzled by channel) and
// pushes its per-head LSE into every peer; after a cluster barrier each CTA merges DV / n_part channels, reading
// its peers' tiles through distributed shared memory, and writes that slice of the output rows.  No global
// round trip, no arrival counter: the global-memory merge took 7 us of a 44 us kernel (profiles/r1e_trace.md).
constexpr int kMaxClusterSplits = 8;
__device__ __forceinline__ uint32_t stage_off(int d, int j4) { return (uint32_t)(d * 128 + ((j4 ^ (d & 7)) << 4)); }
// s_lse_all[r][j]: split r's LSE of head j, pushed by its CTA into every CTA of the cluster before the barrier.
// The code that runs once is kept small and rolled: after an L2 flush every first-touched instruction line is a
// memory round trip that all CTAs wait for in lockstep (profiles/r1e_trace.md).
template <int NT>
__device__ __forceinline__ void merge_cluster(uint8_t* stage, const float (*s_lse_all)[mla::NH], float (*s_w)[mla::NH], int i,
                                              int num_q_heads, int n_part, int rank, __nv_bfloat16* out, float* lse) {
  using namespace mla;
  const int64_t row0 = (int64_t)i * num_q_heads;
  const uint32_t stage_s = smem_u32(stage);
  if (threadIdx.x < NH) {
    const int j = threadIdx.x;
    float mx = -INFINITY;
#pragma unroll 1
    for (int r = 0; r < n_part; ++r) mx = fmaxf(mx, s_lse_all[r][j]);
    float z = 0.f;
#pragma unroll 1
    for (int r = 0; r < n_part; ++r) z += mx == -INFINITY ? 0.f : __expf(s_lse_all[r][j] - mx);
    const float inv = z > 0.f ? 1.f / z : 0.f;
#pragma unroll 1
    for (int r = 0; r < n_part; ++r) s_w[r][j] = mx == -INFINITY ? 0.f : __expf(s_lse_all[r][j] - mx) * inv;
    if (rank == 0 && lse != nullptr && j < num_q_heads) lse[row0 + j] = z > 0.f ? mx + logf(z) : -INFINITY;
  }
  __syncthreads();
  const int DS = DV / n_part, d0 = rank * DS;            // my channel slice
  const int pitch = DS * 2 + 16;                         // bf16 row pitch of the transposed tile (bank spread)
  uint8_t* tile = stage + NH * DV * 4;
  constexpr int UNR = 5;
  const int n_e = DS * (NH / 4);                         // e -> (channel d0 + e / 8, heads 4 (e % 8) ..)
  const int j4 = threadIdx.x % (NH / 4);                 // (NT is a multiple of 8: the same heads for all my items)
#pragma unroll 1
  for (int e0 = threadIdx.x; e0 < n_e; e0 += UNR * NT) {
    float4 acc[UNR];
    {                                                    // my own partial: plain shared-memory reads
      const float4 w = *reinterpret_cast<const float4*>(&s_w[rank][j4 * 4]);
#pragma unroll
      for (int k = 0; k < UNR; ++k) {
        const int e = e0 + k * NT;
        const float4 v = e < n_e ? *reinterpret_cast<const float4*>(stage + stage_off(d0 + e / (NH / 4), j4)) : make_float4(0.f, 0.f, 0.f, 0.f);
        acc[k] = make_float4(w.x * v.x, w.y * v.y, w.z * v.z, w.w * v.w);
      }
    }
#pragma unroll 1
    for (int rr = 1; rr < n_part; ++rr) {                // the peers' partials: distributed shared memory, UNR loads in flight
      const int r = (rank + rr) % n_part;
      const uint32_t peer = dsmem_addr(stage_s, r);
      const float4 w = *reinterpret_cast<const float4*>(&s_w[r][j4 * 4]);
      float4 v[UNR];
#pragma unroll
      for (int k = 0; k < UNR; ++k) {
        const int e = e0 + k * NT;
        v[k] = e < n_e ? dsmem_ld_f32x4(peer + stage_off(d0 + e / (NH / 4), j4)) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int k = 0; k < UNR; ++k) {
        acc[k].x += w.x * v[k].x; acc[k].y += w.y * v[k].y; acc[k].z += w.z * v[k].z; acc[k].w += w.w * v[k].w;
      }
    }
#pragma unroll
    for (int k = 0; k < UNR; ++k) {
      const int e = e0 + k * NT;
      if (e < n_e) {
        uint8_t* t = tile + (j4 * 4) * pitch + (e / (NH / 4)) * 2;
        *reinterpret_cast<__nv_bfloat16*>(t) = __float2bfloat16_rn(acc[k].x);
        *reinterpret_cast<__nv_bfloat16*>(t + pitch) = __float2bfloat16_rn(acc[k].y);
        *reinterpret_cast<__nv_bfloat16*>(t + 2 * pitch) = __float2bfloat16_rn(acc[k].z);
        *reinterpret_cast<__nv_bfloat16*>(t + 3 * pitch) = __float2bfloat16_rn(acc[k].w);
      }
    }
  }
  __syncthreads();
#pragma unroll 1
  for (int e = threadIdx.x; e < num_q_heads * (DS / 8); e += NT) {      // 16 bytes per thread, row slices contiguous
    const int j = e / (DS / 8), c = e % (DS / 8);
    *reinterpret_cast<uint4*>(out + (row0 + j) * DV + d0 + c * 8) = *reinterpret_cast<const uint4*>(tile + j * pitch + c * 16);
  }
}

// tensor map over the latent pool: dims (channel, token in page, page), box = 64 channels x 64 tokens, 128-byte swizzle (vx_decode_mla.cu)
cudaError_t make_latent_map(CUtensorMap* map, const vx_kv_pool& pool);

}  // namespace vx
