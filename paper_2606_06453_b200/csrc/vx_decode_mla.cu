// vx_decode_mla.cu -- (a4) sparse paged decode for the MLA absorbed-latent geometry on tcgen05.
// PAPER.md:92 Eq.4 over the selected pages (:200); :202 / :262 cuda_mla role (one latent KV head of
// width 576 = 512 latent + 64 RoPE shared by all query heads, V = first 512 latent channels, G8).
//
// Per 64-token page the work is two dense contractions, ~60 flop per HBM byte:
//     S^T[64 tokens x 32 heads]  = K[64 x 576] . Q^T          36 x tcgen05.mma  M=64  N=32 K=16
//     O^T[512 x 32 heads]       += V^T[512 x 64] . P^T   4 x 4 x tcgen05.mma  M=128 N=32 K=16
// with tokens / channels on the MMA M axis and the 32 heads on N, so no tile is padded.  The page
// (73,728 B, read once for K and V) is staged by 16-byte cp.async into the 128-byte-swizzled
// shared-memory layout both MMAs consume: K-major for K in S^T, MN-major (transposed) for V^T.
// S^T and O^T live in TMEM; the softmax threads (one per token row) read S^T with tcgen05.ld,
// reduce the per-head maxima across lanes, write P (bf16) back to shared memory as the B operand.
// O^T is rescaled in TMEM only when a head's running maximum grows by more than 2^8 (lazy
// rescaling); the denominators are per-thread partial sums reduced once at the end.
// Two page stages: page p+1 is in flight while page p is computed.
#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

namespace mla {
constexpr int D = 576, DV = 512, PAGE = 64, NH = 32;      // geometry this kernel is built for
constexpr int THREADS = 128;
constexpr int CHUNKS = D * 2 / 16;                        // 72 16-byte chunks per token row
constexpr int ATOMS = CHUNKS / 8;                         // 9 swizzle atoms (64 channels each)
constexpr int K_ATOM_BYTES = PAGE * 128;                  // 8192: 64 rows x 128 B
constexpr int Q_ATOM_BYTES = NH * 128;                    // 4096
constexpr int STAGE_BYTES = ATOMS * K_ATOM_BYTES;         // 73728
constexpr int Q_BYTES = ATOMS * Q_ATOM_BYTES;             // 36864
constexpr int P_BYTES = NH * 128;                         // 4096: [32 heads][64 tokens] bf16
constexpr int SMEM_BYTES = 2 * STAGE_BYTES + Q_BYTES + P_BYTES + 1024;   // + alignment slack
constexpr int TMEM_COLS = 256;                            // S^T: cols [0,32); O^T block mb: cols [32+32mb, ..)
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kRescaleThreshold = 8.f;                  // log2 units

// instruction descriptors (kind::f16): D fp32, A/B bf16
constexpr uint32_t IDESC_QK = (1u << 4) | (1u << 7) | (1u << 10) | ((NH >> 3) << 17) | ((64u >> 4) << 24);
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

// max over the 32 lanes of v[j] for every j; lane L returns the result for j == L
// (transposed butterfly: 16 + 8 + 4 + 2 + 1 shuffles instead of 32 x 5)
__device__ __forceinline__ float lanes_max_transposed(const float (&v)[32], int lane) {
  float a[16], b[8], c[4], d[2];
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    const bool up = lane & 16;
    const float r = __shfl_xor_sync(0xffffffffu, up ? v[j] : v[j + 16], 16);
    a[j] = fmaxf(up ? v[j + 16] : v[j], r);
  }
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const bool up = lane & 8;
    const float r = __shfl_xor_sync(0xffffffffu, up ? a[j] : a[j + 8], 8);
    b[j] = fmaxf(up ? a[j + 8] : a[j], r);
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const bool up = lane & 4;
    const float r = __shfl_xor_sync(0xffffffffu, up ? b[j] : b[j + 4], 4);
    c[j] = fmaxf(up ? b[j + 4] : b[j], r);
  }
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const bool up = lane & 2;
    const float r = __shfl_xor_sync(0xffffffffu, up ? c[j] : c[j + 2], 2);
    d[j] = fmaxf(up ? c[j + 2] : c[j], r);
  }
  const bool up = lane & 1;
  const float r = __shfl_xor_sync(0xffffffffu, up ? d[0] : d[1], 1);
  return fmaxf(up ? d[1] : d[0], r);
}
// same with a sum
__device__ __forceinline__ float lanes_sum_transposed(const float (&v)[32], int lane) {
  float a[16], b[8], c[4], d[2];
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    const bool up = lane & 16;
    a[j] = (up ? v[j + 16] : v[j]) + __shfl_xor_sync(0xffffffffu, up ? v[j] : v[j + 16], 16);
  }
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const bool up = lane & 8;
    b[j] = (up ? a[j + 8] : a[j]) + __shfl_xor_sync(0xffffffffu, up ? a[j] : a[j + 8], 8);
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const bool up = lane & 4;
    c[j] = (up ? b[j + 4] : b[j]) + __shfl_xor_sync(0xffffffffu, up ? b[j] : b[j + 4], 4);
  }
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const bool up = lane & 2;
    d[j] = (up ? c[j + 2] : c[j]) + __shfl_xor_sync(0xffffffffu, up ? c[j] : c[j + 2], 2);
  }
  const bool up = lane & 1;
  return (up ? d[1] : d[0]) + __shfl_xor_sync(0xffffffffu, up ? d[0] : d[1], 1);
}
}  // namespace mla

__global__ void __launch_bounds__(mla::THREADS, 1)
decode_mla_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ kpool, int64_t stride_page,
                  int64_t stride_token, int num_q_heads, float scale_log2, const int32_t* __restrict__ seq_lens,
                  const int32_t* __restrict__ sel_phys, const int32_t* __restrict__ sel_logical,
                  const int32_t* __restrict__ sel_count, int max_budget, int num_splits,
                  float* __restrict__ part_o, float* __restrict__ part_lse, __nv_bfloat16* __restrict__ out,
                  float* __restrict__ lse_out) {
  using namespace mla;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t s_bar[2];           // [0]: S^T ready, [1]: O^T accumulated
  __shared__ uint32_t s_tmem;
  __shared__ float s_wred[4][NH], s_mref[NH], s_fac[NH];
  __shared__ int s_flag;

  const int split = blockIdx.x, i = blockIdx.z;
  const int tid = threadIdx.x, warp = tid / kWarp, lane = tid % kWarp;
  const int n_tok = seq_lens[i];
  const int cnt = sel_count[i];
  const int per_split = (cnt + num_splits - 1) / num_splits;
  const int r_begin = min(split * per_split, cnt), r_end = min(r_begin + per_split, cnt);
  const int n_pages = r_end - r_begin;
  const int32_t* phys_list = sel_phys + (int64_t)i * max_budget + r_begin;
  const int32_t* log_list = sel_logical + (int64_t)i * max_budget + r_begin;
  const int dim_of_thread = warp * 32 + lane;          // O^T row (within a 128-channel block) this thread reads

  if (n_pages == 0) {                                  // empty split: contributes nothing to the merge
    for (int e = tid; e < num_q_heads * DV; e += THREADS) {
      const int h = e / DV, d = e % DV;
      const int64_t row = (int64_t)i * num_q_heads + h;
      if (num_splits == 1) out[row * DV + d] = __float2bfloat16_rn(0.f);
      else part_o[(row * num_splits + split) * DV + d] = 0.f;
    }
    if (tid < num_q_heads) {
      const int64_t row = (int64_t)i * num_q_heads + tid;
      if (num_splits == 1) { if (lse_out) lse_out[row] = -INFINITY; }
      else part_lse[row * num_splits + split] = -INFINITY;
    }
    return;
  }

  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;        // swizzle atoms need 1024-byte alignment
  uint8_t* sm = smem_raw + (base - raw);
  const uint32_t q_base = base + 2 * STAGE_BYTES, p_base = q_base + Q_BYTES;
  const uint32_t bar_s = smem_u32(&s_bar[0]), bar_o = smem_u32(&s_bar[1]);

  auto issue_page = [&](int p) {                       // all threads: page p -> stage p & 1 (zero-fill invalid rows)
    const int64_t phys = phys_list[p];
    const int valid = min(PAGE, n_tok - log_list[p] * PAGE);
    const __nv_bfloat16* src = kpool + phys * stride_page;
    const uint32_t dst = base + (uint32_t)(p & 1) * STAGE_BYTES;
#pragma unroll 4
    for (int x = tid; x < PAGE * CHUNKS; x += THREADS) {
      const int r = x / CHUNKS, c = x % CHUNKS;
      const uint32_t off = (c >> 3) * K_ATOM_BYTES + (r >> 3) * 1024 + (r & 7) * 128 + (((c & 7) ^ (r & 7)) << 4);
      const int n = r < valid ? 16 : 0;
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst + off),
                   "l"(src + (int64_t)r * stride_token + c * 8), "r"(n));
    }
  };

  // ---- prologue: TMEM, barriers, Q tile, first page ------------------------------------------
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 0) {
    mbar_init(bar_s, 1);
    mbar_init(bar_o, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  issue_page(0);
  cp_async_commit();
  for (int x = tid; x < NH * CHUNKS; x += THREADS) {   // Q[32 x 576] -> K-major swizzled B operand (zero rows past Hq)
    const int h = x / CHUNKS, c = x % CHUNKS;
    uint4 v = make_uint4(0, 0, 0, 0);
    if (h < num_q_heads) v = *reinterpret_cast<const uint4*>(q + ((int64_t)i * num_q_heads + h) * D + c * 8);
    const uint32_t off = (c >> 3) * Q_ATOM_BYTES + (h >> 3) * 1024 + (h & 7) * 128 + (((c & 7) ^ (h & 7)) << 4);
    *reinterpret_cast<uint4*>(sm + 2 * STAGE_BYTES + off) = v;
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = s_tmem;
  const uint32_t t_lane = tmem + ((uint32_t)(warp * 32) << 16);

  float l_thr[NH];
#pragma unroll
  for (int j = 0; j < NH; ++j) l_thr[j] = 0.f;

  for (int p = 0; p < n_pages; ++p) {
    const uint32_t stage = base + (uint32_t)(p & 1) * STAGE_BYTES;
    if (p > 0) mbar_wait(bar_o, (p - 1) & 1);          // PV of page p-1 done: P and the other stage are free
    if (p + 1 < n_pages) issue_page(p + 1);
    cp_async_commit();
    cp_async_wait<1>();                                // page p has landed (this thread's copies)
    fence_async_proxy();                               // make cp.async / st.shared data visible to the MMA proxy
    __syncthreads();
    if (tid == 0) {
      tc_fence_after();
#pragma unroll 4
      for (int ks = 0; ks < D / 16; ++ks) {
        const uint32_t a = stage + (ks >> 2) * K_ATOM_BYTES + (ks & 3) * 32;
        const uint32_t b = q_base + (ks >> 2) * Q_ATOM_BYTES + (ks & 3) * 32;
        umma(tmem, smem_desc(a, 16, 1024), smem_desc(b, 16, 1024), IDESC_QK, ks > 0);
      }
      umma_commit(bar_s);
    }
    const int valid = min(PAGE, n_tok - log_list[p] * PAGE);
    const int row = warp * 16 + lane;                  // M = 64: token row r sits in TMEM lane (r % 16) + 32 * (r / 16)
    const bool live = lane < 16 && row < valid;
    mbar_wait(bar_s, p & 1);
    tc_fence_after();
    float s[NH];
    tmem_ld32(t_lane, s);
#pragma unroll
    for (int j = 0; j < NH; ++j) s[j] = live ? s[j] * scale_log2 : -INFINITY;
    s_wred[warp][lane] = lanes_max_transposed(s, lane);
    __syncthreads();
    if (warp == 0) {                                   // lane = head: tile maximum, lazy running reference
      const float tmax = fmaxf(fmaxf(s_wred[0][lane], s_wred[1][lane]), fmaxf(s_wred[2][lane], s_wred[3][lane]));
      bool grow = false;
      if (p == 0) {
        s_mref[lane] = tmax;
      } else {
        const float old = s_mref[lane];
        grow = tmax > old + kRescaleThreshold;
        s_fac[lane] = grow ? exp2f(old - tmax) : 1.f;
        if (grow) s_mref[lane] = tmax;
      }
      const bool any = __any_sync(0xffffffffu, grow);
      if (lane == 0) s_flag = any;
    }
    __syncthreads();
    if (p > 0 && s_flag) {                             // rare: rescale O^T in TMEM and the partial denominators
#pragma unroll 1
      for (int mb = 0; mb < DV / 128; ++mb) {
        float o[NH];
        tmem_ld32(t_lane + 32 + 32 * mb, o);
#pragma unroll
        for (int j = 0; j < NH; ++j) o[j] *= s_fac[j];
        tmem_st32(t_lane + 32 + 32 * mb, o);
      }
#pragma unroll
      for (int j = 0; j < NH; ++j) l_thr[j] *= s_fac[j];
    }
    if (lane < 16) {                                   // P[head][token] bf16, K-major swizzled B operand
      uint8_t* pdst = sm + 2 * STAGE_BYTES + Q_BYTES + (row & 7) * 2;
      const int tc = row >> 3;
#pragma unroll
      for (int j = 0; j < NH; ++j) {
        const float pj = exp2f(s[j] - s_mref[j]);
        l_thr[j] += pj;
        *reinterpret_cast<__nv_bfloat16*>(pdst + (j >> 3) * 1024 + (j & 7) * 128 + ((tc ^ (j & 7)) << 4)) =
            __float2bfloat16_rn(pj);
      }
    }
    fence_async_proxy();
    tc_fence_before();
    __syncthreads();
    if (tid == 0) {
      tc_fence_after();
#pragma unroll
      for (int ks = 0; ks < PAGE / 16; ++ks)
#pragma unroll
        for (int mb = 0; mb < DV / 128; ++mb)
          umma(tmem + 32 + 32 * mb, smem_desc(stage + 2 * mb * K_ATOM_BYTES + ks * 2048, K_ATOM_BYTES, 1024),
               smem_desc(p_base + ks * 32, 16, 1024), IDESC_PV, p > 0 || ks > 0);
      umma_commit(bar_o);
    }
  }
  cp_async_wait<0>();
  mbar_wait(bar_o, (n_pages - 1) & 1);
  tc_fence_after();

  // ---- epilogue: denominators, normalise, write the partial (or final) result -------------------
  s_wred[warp][lane] = lanes_sum_transposed(l_thr, lane);
  __syncthreads();
  if (warp == 0) s_fac[lane] = s_wred[0][lane] + s_wred[1][lane] + s_wred[2][lane] + s_wred[3][lane];
  __syncthreads();
#pragma unroll 1
  for (int mb = 0; mb < DV / 128; ++mb) {
    float o[NH];
    tmem_ld32(t_lane + 32 + 32 * mb, o);
    const int d = mb * 128 + dim_of_thread;
#pragma unroll
    for (int j = 0; j < NH; ++j) {
      if (j < num_q_heads) {
        const float val = o[j] / s_fac[j];
        const int64_t row = (int64_t)i * num_q_heads + j;
        if (num_splits == 1) out[row * DV + d] = __float2bfloat16_rn(val);
        else part_o[(row * num_splits + split) * DV + d] = val;
      }
    }
  }
  if (tid < num_q_heads) {
    const float lse = (s_mref[tid] + log2f(s_fac[tid])) * kLn2;
    const int64_t row = (int64_t)i * num_q_heads + tid;
    if (num_splits == 1) { if (lse_out) lse_out[row] = lse; }
    else part_lse[row * num_splits + split] = lse;
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
}

bool mla_tc_supported(const vx_geom& g) {
  return g.kv_shared && g.dtype == VX_DT_BF16 && g.num_kv_heads == 1 && g.qk_dim == mla::D && g.v_dim == mla::DV &&
         g.page_size == mla::PAGE && g.num_q_heads <= mla::NH;
}

cudaError_t launch_decode_mla_tc(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                 const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                 int32_t max_budget, void* out, float* lse, cudaStream_t s, const DecodeOpts& opt) {
  const vx_geom& g = c->g;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(decode_mla_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, mla::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  // one CTA per SM (190 KB of shared memory): pick the split count that minimises
  // waves x pages-per-CTA (+1 page of prologue per wave)
  int best = 1, best_cost = 1 << 30;
  for (int sp = 1; sp <= kMaxSplits && sp <= max_budget; ++sp) {
    const int waves = (pt.batch * sp + c->num_sms - 1) / c->num_sms;
    const int cost = waves * ((max_budget + sp - 1) / sp + 1);
    if (cost < best_cost) { best_cost = cost; best = sp; }
  }
  dim3 grid(best, 1, pt.batch);
  decode_mla_kernel<<<grid, mla::THREADS, mla::SMEM_BYTES, s>>>(
      static_cast<const __nv_bfloat16*>(q), static_cast<const __nv_bfloat16*>(pool.k), pool.stride_page,
      pool.stride_token, g.num_q_heads, g.sm_scale * mla::kLog2e, pt.seq_lens, sel_phys, sel_logical, sel_count,
      max_budget, best, c->ws.part_o, c->ws.part_lse, static_cast<__nv_bfloat16*>(out), lse);
  c->launches += 1;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess || best == 1) return e;
  return launch_combine(c, pt.batch, best, out, lse, s);
}

}  // namespace vx
