// vx_decode_mla.cu -- (a4)+(a5)(+a1) sparse paged decode for the MLA absorbed-latent geometry on tcgen05.
// PAPER.md:92 Eq.4 over the selected pages (:200); :202 / :262 cuda_mla role (one latent KV head of
// width 576 = 512 latent + 64 RoPE shared by all query heads, V = first 512 latent channels, G8).
//
// Per 64-token page the work is two dense contractions, ~60 flop per HBM byte:
//     S[32 heads x 64 tokens]  = Q[32 x 576] . K^T           36 x tcgen05.mma  M=128 N=64 K=16, A = Q in TMEM
//     O^T[512 x 32 heads]     += V^T[512 x 64] . P^T     4 x 4 x tcgen05.mma  M=128 N=32 K=16
// S keeps the heads on the MMA M axis (TMEM lanes 32..127 of the A operand are don't-care: every D row depends
// on its own A row only), and Q -- constant for the whole CTA -- is the A operand held in TENSOR MEMORY
// (288 columns, written once with tcgen05.st).  Measured on B200 (clock64 traces): with a K-major A tile in
// shared memory an MMA of this shape retires every ~107 cycles (the 128-row A fetch dominates the skinny
// N = 64 math), which made the tensor pipe, not HBM, the bound.  With heads on TMEM lanes a softmax thread owns
// one head: running max, sum and the P row are thread-local, no cross-lane or cross-warp reduction in the loop.
//
// Warp-specialised, one CTA per SM:
//   warp 0      TMA producer.  The latent page (73,728 B, read once for K and V) arrives as nine
//               [64 tokens x 64 channels] boxes (cp.async.bulk.tensor, 128-byte swizzle) -- exactly the
//               shared-memory layout both MMAs consume (K-major B operand of S, MN-major A operand of O^T).
//               The ring is managed per BOX PAIR (16 KB = 128 value channels): 12 pair slots + 3 RoPE slots
//               = 3 pages, each slot released by the tcgen05.commit of the last MMA that reads it.
//   warp 1      QK issuer (one elected lane): once S is free and page p has landed (ONE full barrier per page), the
//               36 MMAs of S(p) go out back to back.  warp 6, the PV issuer, sends the 16 MMAs of O^T += V(p)^T P(p)^T
//               the moment P(p) is written, and its commits free the page's slots.  Both wait on their mbarriers in a
//               fixed order with blocking waits: one warp polling several barriers (~150 cycles per test_wait) was
//               the kernel's bound.  S (64 columns), Q (288) and O^T (128 columns, 512 x 32 fp32) live in TMEM.
//   warp 4      softmax (TMEM lanes 0..31 = heads): tcgen05.ld S, thread-local max / exp2 / sum, P row (bf16,
//               128 B) to shared memory as the B operand of PV, double-buffered.  O^T is rescaled lazily (only
//               when a head's running max grows by more than 2^8): the softmax warp publishes the factors,
//               warps 2, 3, 5 rescale the TMEM lanes it cannot reach.
//   warps 2..5  epilogue: O^T / l -> partial or final output.
// Splits of a request merge in-kernel (the last split to arrive merges by LSE).  In the
// fused step the CTA holding the request's newest page also rebuilds that page's summary (min / max, or the
// block top-k centroid) from the staged tile (a1; the newest page is a forced local page).
// (The fused step of this geometry -- score, select, decode and merge of a request in one kernel -- is vx_step_mla.cu; the
//  kernel below is kept textually apart from it: its inner loops are sensitive to how ptxas schedules the code around them,
//  a shared template measured 3 us slower on C4.)
#include "vx_mla.cuh"

namespace vx {

__global__ void __launch_bounds__(mla::THREADS_DECODE, 1)
decode_mla_kernel(const __grid_constant__ CUtensorMap kmap, const __nv_bfloat16* __restrict__ q, int num_q_heads,
                  float scale_log2, const int32_t* __restrict__ seq_lens, const int32_t* __restrict__ sel_phys,
                  const int32_t* __restrict__ sel_logical, const int32_t* __restrict__ sel_count, int max_budget,
                  int num_splits, float* __restrict__ part_o, float* __restrict__ part_lse,
                  int* __restrict__ unit_counter, __nv_bfloat16* __restrict__ summary_upd, int summary_kind,
                  __nv_bfloat16* __restrict__ out, float* __restrict__ lse_out, int req0,
                  const int32_t* __restrict__ budget_opt, int cluster_merge, float out_scale) {
  using namespace mla;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t s_bar[N_BARS];
  __shared__ uint32_t s_tmem;
  __shared__ float s_fac[2][NH];                       // lazy-rescale factors of page p (buffer p & 1)
  __shared__ int s_flag[2];                            // ... and whether any head needs them
  __shared__ float s_l[NH], s_m[NH], s_inv[NH];        // final denominators / references
  __shared__ int s_last;
  __shared__ float s_lse_all[kMaxClusterSplits][NH];   // cluster merge: every split's per-head LSE (pushed by its CTA)

  const int split = blockIdx.x, i = blockIdx.z + req0;
  const int tid = threadIdx.x, warp = tid / kWarp, lane = tid % kWarp;
  [[maybe_unused]] const int cta = blockIdx.z * gridDim.x + blockIdx.x;
  if (tid == 0) { VX_TRACE_STAMP(cta, 0); VX_TRACE_SMID(cta); }
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;        // swizzle atoms need 1024-byte alignment
  uint8_t* sm = smem_raw + (base - raw);
  const uint32_t bar0 = smem_u32(&s_bar[0]);
  auto bar = [&](int idx) -> uint32_t { return bar0 + 8u * (uint32_t)idx; };
  const int n_tok = seq_lens[i];
  const int newest_page = (n_tok - 1) / PAGE;
  const int cnt_known = budget_opt ? max(0, min(min(budget_opt[i], max_budget), newest_page + 1)) : -1;

  // ---- prologue (overlaps the preceding kernel under PDL): barriers, TMEM, Q tile ---------------------
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 0) {
    for (int s = 0; s < N_PAIR; ++s) mbar_init(bar(B_PAIR_EMPTY + s), 1);
    for (int s = 0; s < N_ROPE; ++s) { mbar_init(bar(B_PAGE_FULL + s), 1); mbar_init(bar(B_ROPE_EMPTY + s), 1); }
    mbar_init(bar(B_S_FULL), 1);
    mbar_init(bar(B_S_EMPTY), 1);
    for (int b = 0; b < 2; ++b) {
      mbar_init(bar(B_P_FULL + b), 1);
      mbar_init(bar(B_PV_DONE + b), 1);
      mbar_init(bar(B_DECIDE + b), 1);
      mbar_init(bar(B_ACK + b), 3);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&kmap) : "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (tid == 0) VX_TRACE_STAMP(cta, 1);
  const uint32_t tmem = s_tmem;
  // Q[32 x 576] -> TMEM lanes 0..31 (heads), 288 columns (zero rows past Hq): coalesced through the (still
  // idle) ring, row pitch padded to 1168 B so that the per-head reads are bank-conflict free
  constexpr int Q_PITCH = D * 2 + 16;
  if (warp >= 2 && warp <= 5) {
    constexpr int Q_IT = NH * CHUNKS / SOFTMAX_THREADS;          // 18 independent 16-byte loads per thread
    static_assert(NH * CHUNKS % SOFTMAX_THREADS == 0, "Q staging");
    uint4 qv[Q_IT];
#pragma unroll
    for (int k = 0; k < Q_IT; ++k) {
      const int x = tid - 64 + k * SOFTMAX_THREADS, h = x / CHUNKS, c = x % CHUNKS;
      qv[k] = h < num_q_heads ? *reinterpret_cast<const uint4*>(q + ((int64_t)i * num_q_heads + h) * D + c * 8)
                              : make_uint4(0, 0, 0, 0);
    }
#pragma unroll
    for (int k = 0; k < Q_IT; ++k) {
      const int x = tid - 64 + k * SOFTMAX_THREADS, h = x / CHUNKS, c = x % CHUNKS;
      *reinterpret_cast<uint4*>(sm + OFF_PAIR + h * Q_PITCH + c * 16) = qv[k];
    }
    softmax_barrier();
    if (warp == SOFTMAX_WARP) {
      const uint4* qrow = reinterpret_cast<const uint4*>(sm + OFF_PAIR + lane * Q_PITCH);
#pragma unroll 1
      for (int c = 0; c < D / 64; ++c) {               // 64 channels = 32 columns at a time
        float w[32];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          const uint4 v = qrow[c * 8 + e];
          w[4 * e + 0] = __uint_as_float(v.x); w[4 * e + 1] = __uint_as_float(v.y);
          w[4 * e + 2] = __uint_as_float(v.z); w[4 * e + 3] = __uint_as_float(v.w);
        }
        tmem_st32(tmem + TM_Q + 32 * c, w);
      }
      tc_fence_before();
    }
  }
  __syncthreads();
  tc_fence_after();
  if (tid == 0) VX_TRACE_STAMP(cta, 2);
  pdl_wait();
  if (tid == 0) VX_TRACE_STAMP(cta, 3);                                          // the selection lists come from the preceding kernel of the step

  const int cnt = cnt_known >= 0 ? cnt_known : sel_count[i];
  const int per_split = (cnt + num_splits - 1) / num_splits;
  const int r_begin = min(split * per_split, cnt), r_end = min(r_begin + per_split, cnt);
  const int n_pages = r_end - r_begin;
  const int32_t* phys_list = sel_phys + (int64_t)i * max_budget + r_begin;
  const int32_t* log_list = sel_logical + (int64_t)i * max_budget + r_begin;
  const uint32_t p_base = base + OFF_P;

  if (n_pages == 0 && cluster_merge) {                 // empty split: a zero tile with weight zero
    for (int e = tid; e < NH * DV / 4; e += THREADS_DECODE) reinterpret_cast<float4*>(sm + OFF_PAIR)[e] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid < NH)
      for (int r = 0; r < num_splits; ++r) dsmem_st_f32(dsmem_addr(smem_u32(&s_lse_all[split][tid]), r), -INFINITY);
  } else if (n_pages == 0) {                           // empty split: contributes nothing to the merge
    for (int e = tid; e < NH * DV; e += THREADS_DECODE) {       // partial layout: [request][split][channel][head]
      const int h = e / DV, d = e % DV;
      if (num_splits > 1) part_o[(((int64_t)i * num_splits + split) * DV + d) * NH + h] = 0.f;
      else if (h < num_q_heads) out[((int64_t)i * num_q_heads + h) * DV + d] = __float2bfloat16_rn(0.f);
    }
    if (tid < num_q_heads) {
      const int64_t row = (int64_t)i * num_q_heads + tid;
      if (num_splits == 1) { if (lse_out) lse_out[row] = -INFINITY; }
      else part_lse[row * num_splits + split] = -INFINITY;
    }
  } else if (warp == 0) {
    // ===== TMA producer: page p -> ring page p % 3 (4 pair slots + 1 RoPE slot), one full barrier per page =====
    static_assert(N_PAIR == N_ROPE * PAIRS_PER_PAGE, "the ring is a whole number of pages");
    int my_phys = 0;
    for (int p = 0; p < n_pages; ++p) {
      if ((p & 31) == 0) my_phys = p + lane < n_pages ? phys_list[p + lane] : 0;
      const int phys = __shfl_sync(0xffffffffu, my_phys, p & 31);
      if (elect_one()) {
        const int rs = p % N_ROPE, u = p / N_ROPE;
        const uint32_t full = bar(B_PAGE_FULL + rs);
        if (u >= 1) mbar_wait(bar(B_ROPE_EMPTY + rs), (u - 1) & 1);      // QK(p-3) done (it also observed the last phase)
        mbar_expect_tx(full, PAGE_BYTES);
        tma_box(base + OFF_ROPE + rs * K_ATOM_BYTES, &kmap, DV, phys, full);
#pragma unroll
        for (int j = 0; j < PAIRS_PER_PAGE; ++j) {
          const int ps = rs * PAIRS_PER_PAGE + j;
          if (u >= 1) mbar_wait(bar(B_PAIR_EMPTY + ps), (u - 1) & 1);    // PV(p-3) has read this pair
          const uint32_t dst = base + OFF_PAIR + ps * PAIR_BYTES;
          tma_box(dst, &kmap, 128 * j, phys, full);
          tma_box(dst + K_ATOM_BYTES, &kmap, 128 * j + 64, phys, full);
        }
        if (p == 0) VX_TRACE_STAMP(cta, 4);
      }
      __syncwarp();
    }
  } else if (warp == 1) {
    // ===== QK issuer: S(p) = Q . K(p)^T, 36 MMAs back to back once the page has landed and S is free ==========
    // (barrier waits are blocking and in a fixed order -- polling several mbarriers cost ~150 cycles per test and
    //  made the issue loop, not the tensor pipe, the bound)
    for (int p = 0; p < n_pages; ++p) {
      const int rs = p % N_ROPE;
      if (p >= 1) mbar_wait(bar(B_S_EMPTY), (p - 1) & 1);                // softmax has read S(p-1)
      mbar_wait(bar(B_PAGE_FULL + rs), (p / N_ROPE) & 1);
      tc_fence_after();
      if (elect_one()) {
        if (p == 0) VX_TRACE_STAMP(cta, 5);
        if (p == n_pages - 1) VX_TRACE_STAMP(cta, 6);
#pragma unroll
        for (int j = 0; j < PAIRS_PER_PAGE; ++j)
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) {
            const uint32_t kb = base + OFF_PAIR + (rs * PAIRS_PER_PAGE + j) * PAIR_BYTES + (ks >> 2) * K_ATOM_BYTES + (ks & 3) * 32;
            umma_ts(tmem + TM_S, tmem + TM_Q + 64 * j + 8 * ks, smem_desc(kb, 16, 1024), IDESC_QK, j > 0 || ks > 0);
          }
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)                                   // RoPE channels 512 + 16 ks: Q columns 256 + 8 ks
          umma_ts(tmem + TM_S, tmem + TM_Q + 256 + 8 * ks, smem_desc(base + OFF_ROPE + rs * K_ATOM_BYTES + ks * 32, 16, 1024),
                  IDESC_QK, true);
        umma_commit(bar(B_ROPE_EMPTY + rs));
        umma_commit(bar(B_S_FULL));
      }
      __syncwarp();
    }
  } else if (warp == PV_WARP) {
    // ===== PV issuer: O^T += V(p)^T . P(p)^T the moment P(p) is written; frees the page's pair slots ============
    for (int p = 0; p < n_pages; ++p) {
      const int b = p & 1, rs = p % N_ROPE;
      mbar_wait(bar(B_P_FULL + b), (p >> 1) & 1);                        // P(p) written, O^T rescaled if it had to be
      tc_fence_after();
      if (elect_one()) {
#pragma unroll
        for (int ks = 0; ks < PAGE / 16; ++ks)                           // ks-major: consecutive MMAs go to different O^T blocks
#pragma unroll
          for (int mb = 0; mb < PAIRS_PER_PAGE; ++mb)
            umma(tmem + TM_O + 32 * mb,
                 smem_desc(base + OFF_PAIR + (rs * PAIRS_PER_PAGE + mb) * PAIR_BYTES + ks * 2048, K_ATOM_BYTES, 1024),
                 smem_desc(p_base + b * P_BYTES + ks * 32, 16, 1024), IDESC_PV, p > 0 || ks > 0);
#pragma unroll
        for (int mb = 0; mb < PAIRS_PER_PAGE; ++mb) umma_commit(bar(B_PAIR_EMPTY + rs * PAIRS_PER_PAGE + mb));
        umma_commit(bar(B_PV_DONE + b));
        if (p == n_pages - 1) VX_TRACE_STAMP(cta, 7);
      }
      __syncwarp();
    }
    pdl_trigger();
  } else {
    // ===== warps 2..5: softmax (warp 4) + rescale helpers, then the epilogue ==============================
    const int sp = warp & 3;                             // TMEM sub-partition this warp may access
    const uint32_t t_lane = tmem + ((uint32_t)(sp * 32) << 16);
    const int pl = n_pages - 1;
    if (warp == SOFTMAX_WARP) {
      // thread = head `lane` (TMEM lane); columns = the 64 tokens of the page
      float m_ref = 0.f, l_sum = 0.f;
      int lg = log_list[0];
      for (int p = 0; p < n_pages; ++p) {
        const int b = p & 1;
        const int valid = min(PAGE, n_tok - lg * PAGE);
        if (p + 1 < n_pages) lg = log_list[p + 1];       // prefetch for the next page
        mbar_wait(bar(B_S_FULL), p & 1);
        tc_fence_after();
        float s[PAGE];
        tmem_ld32(t_lane + TM_S, *reinterpret_cast<float(*)[32]>(&s[0]));
        tmem_ld32(t_lane + TM_S + 32, *reinterpret_cast<float(*)[32]>(&s[32]));
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(B_S_EMPTY));      // S may be overwritten by QK(p+1)
        float tmax = -INFINITY;
#pragma unroll
        for (int t = 0; t < PAGE; ++t) {
          s[t] = t < valid ? s[t] * scale_log2 : -INFINITY;
          tmax = fmaxf(tmax, s[t]);
        }
        // lazy running reference: it moves only on a growth > 2^8 (token 0 of a page is always valid: tmax finite)
        const bool grow = p > 0 && tmax > m_ref + kRescaleThreshold;
        const float fac = grow ? exp2f(m_ref - tmax) : 1.f;
        if (p == 0 || grow) m_ref = tmax;
        l_sum *= fac;
        const bool grow_any = __any_sync(0xffffffffu, grow);
        // publish the decision to the helper warps (they acknowledged page p-2 before its buffer is reused)
        if (p >= 2) mbar_wait(bar(B_ACK + b), ((p >> 1) - 1) & 1);
        s_fac[b][lane] = fac;
        if (lane == 0) s_flag[b] = grow_any;
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(B_DECIDE + b));
        if (p >= 2) mbar_wait(bar(B_PV_DONE + b), ((p >> 1) - 1) & 1);   // PV(p-2) done: P buffer b is free
        if (grow_any) {                                  // rare: rescale O^T in TMEM (my 32 lanes; helpers do theirs)
          mbar_wait(bar(B_PV_DONE + ((p - 1) & 1)), ((p - 1) >> 1) & 1); // PV(p-1) done: O^T is stable
          tc_fence_after();
#pragma unroll 1
          for (int mb = 0; mb < PAIRS_PER_PAGE; ++mb) {
            float o[NH];
            tmem_ld32(t_lane + TM_O + 32 * mb, o);
#pragma unroll
            for (int j = 0; j < NH; ++j) o[j] *= s_fac[b][j];
            tmem_st32(t_lane + TM_O + 32 * mb, o);
          }
          tc_fence_before();
          mbar_wait(bar(B_ACK + b), (p >> 1) & 1);        // the helpers have rescaled their lanes
        }
        if (valid < PAGE) {                              // partial page: zero the stale value rows (0 x garbage must be 0)
          const int n_rows = PAGE - valid;
          for (int xx = lane; xx < n_rows * 64; xx += kWarp) {
            const int r = valid + xx / 64, a = (xx % 64) >> 3, c = xx & 7;
            const int ps = (p * PAIRS_PER_PAGE + (a >> 1)) % N_PAIR;
            *reinterpret_cast<uint4*>(sm + OFF_PAIR + ps * PAIR_BYTES + (a & 1) * K_ATOM_BYTES + (r >> 3) * 1024 +
                                      (r & 7) * 128 + c * 16) = make_uint4(0, 0, 0, 0);
          }
        }
        // P[head = lane][token] bf16: one 128-byte row of the K-major swizzled B operand
        uint8_t* prow = sm + OFF_P + b * P_BYTES + (lane >> 3) * 1024 + (lane & 7) * 128;
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          uint32_t w[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float p0 = ex2_approx(s[8 * c + 2 * e] - m_ref), p1 = ex2_approx(s[8 * c + 2 * e + 1] - m_ref);
            l_sum += p0 + p1;
            __nv_bfloat162 v = __floats2bfloat162_rn(p0, p1);
            w[e] = *reinterpret_cast<uint32_t*>(&v);
          }
          *reinterpret_cast<uint4*>(prow + ((c ^ (lane & 7)) << 4)) = make_uint4(w[0], w[1], w[2], w[3]);
        }
        fence_async_proxy();                             // P / zeroed rows visible to the MMA proxy
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(B_P_FULL + b));
      }
      s_l[lane] = l_sum;
      s_m[lane] = m_ref;
      s_inv[lane] = out_scale / l_sum;              // (out_scale: 1, or an fp8 pool's v_scale)
    } else {
      // helper warps: follow the softmax warp's decisions; rescale their TMEM lanes of O^T when asked (rare)
      for (int p = 0; p < n_pages; ++p) {
        const int b = p & 1;
        mbar_wait(bar(B_DECIDE + b), (p >> 1) & 1);
        if (s_flag[b]) {
          mbar_wait(bar(B_PV_DONE + ((p - 1) & 1)), ((p - 1) >> 1) & 1);
          tc_fence_after();
#pragma unroll 1
          for (int mb = 0; mb < PAIRS_PER_PAGE; ++mb) {
            float o[NH];
            tmem_ld32(t_lane + TM_O + 32 * mb, o);
#pragma unroll
            for (int j = 0; j < NH; ++j) o[j] *= s_fac[b][j];
            tmem_st32(t_lane + TM_O + 32 * mb, o);
          }
          tc_fence_before();
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(B_ACK + b));
      }
      // (a1) the request's newest page is this CTA's last page: rebuild its min / max summary from the staged
      // tile (exact in bf16).  One helper thread per 16-byte channel chunk over the valid tokens.
      const int hidx = (warp == 5 ? 2 : warp - 2) * kWarp + lane;      // 0..95
      const int lg_last = log_list[pl];
      if (summary_upd != nullptr && lg_last == newest_page && hidx < CHUNKS) {
        mbar_wait(bar(B_S_FULL), pl & 1);                              // QK(last) done: every box of the page has landed
        const int valid = min(PAGE, n_tok - lg_last * PAGE);
        const int cc = hidx, a = cc >> 3;
        const uint8_t* atom = a < 8 ? sm + OFF_PAIR + ((pl * PAIRS_PER_PAGE + (a >> 1)) % N_PAIR) * PAIR_BYTES + (a & 1) * K_ATOM_BYTES
                                    : sm + OFF_ROPE + (pl % N_ROPE) * K_ATOM_BYTES;
        if (summary_kind == VX_SUMMARY_CENTROID) {       // block top-k: exact mean of the valid latents, one rounding
          double sum[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) sum[e] = 0.0;
          for (int r = 0; r < valid; ++r) {
            const uint4 v4 = *reinterpret_cast<const uint4*>(atom + (r >> 3) * 1024 + (r & 7) * 128 + (((cc & 7) ^ (r & 7)) << 4));
            float f[8];
            Elem<__nv_bfloat16>::unpack(v4, f);
#pragma unroll
            for (int e = 0; e < 8; ++e) sum[e] += (double)f[e];
          }
          alignas(16) __nv_bfloat16 o8[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) o8[e] = round_double<__nv_bfloat16>(sum[e] / (double)valid);
          *reinterpret_cast<uint4*>(summary_upd + (int64_t)phys_list[pl] * D + cc * 8) = *reinterpret_cast<const uint4*>(o8);
        } else {
        uint4 lo4 = *reinterpret_cast<const uint4*>(atom + ((cc & 7) << 4)), hi4 = lo4;     // token 0
        __nv_bfloat162* lo = reinterpret_cast<__nv_bfloat162*>(&lo4);
        __nv_bfloat162* hi = reinterpret_cast<__nv_bfloat162*>(&hi4);
        for (int r = 1; r < valid; ++r) {
          const uint4 v4 = *reinterpret_cast<const uint4*>(atom + (r >> 3) * 1024 + (r & 7) * 128 + (((cc & 7) ^ (r & 7)) << 4));
          const __nv_bfloat162* v = reinterpret_cast<const __nv_bfloat162*>(&v4);
#pragma unroll
          for (int e = 0; e < 4; ++e) { lo[e] = __hmin2(lo[e], v[e]); hi[e] = __hmax2(hi[e], v[e]); }
        }
        __nv_bfloat16* dst = summary_upd + (int64_t)phys_list[pl] * 2 * D + cc * 8;
        *reinterpret_cast<uint4*>(dst) = lo4;
        *reinterpret_cast<uint4*>(dst + D) = hi4;
        }
      }
    }
    // ---- epilogue (warps 2..5): O^T / l -> partial or final output ----------------------------------------
    softmax_barrier();                                   // s_l / s_m published
    mbar_wait(bar(B_PV_DONE + (pl & 1)), (pl >> 1) & 1); // the last PV has landed in TMEM
    tc_fence_after();
#pragma unroll 1
    for (int mb = 0; mb < PAIRS_PER_PAGE; ++mb) {
      float o[NH];
      tmem_ld32(t_lane + TM_O + 32 * mb, o);
      const int d = mb * 128 + sp * 32 + lane;
      if (cluster_merge) {                               // partial stays in shared memory (the ring is drained)
        uint8_t* stage = sm + OFF_PAIR;
#pragma unroll
        for (int j4 = 0; j4 < NH / 4; ++j4)
          *reinterpret_cast<float4*>(stage + stage_off(d, j4)) =
              make_float4(o[4 * j4] * s_inv[4 * j4], o[4 * j4 + 1] * s_inv[4 * j4 + 1], o[4 * j4 + 2] * s_inv[4 * j4 + 2],
                          o[4 * j4 + 3] * s_inv[4 * j4 + 3]);
      } else if (num_splits > 1) {                       // partial [request][split][channel][head]: 128 contiguous bytes per thread
        float4* dst = reinterpret_cast<float4*>(part_o + (((int64_t)i * num_splits + split) * DV + d) * NH);
#pragma unroll
        for (int j4 = 0; j4 < NH / 4; ++j4)
          dst[j4] = make_float4(o[4 * j4] * s_inv[4 * j4], o[4 * j4 + 1] * s_inv[4 * j4 + 1],
                                o[4 * j4 + 2] * s_inv[4 * j4 + 2], o[4 * j4 + 3] * s_inv[4 * j4 + 3]);
      } else {
#pragma unroll
        for (int j = 0; j < NH; ++j)
          if (j < num_q_heads) out[((int64_t)i * num_q_heads + j) * DV + d] = __float2bfloat16_rn(o[j] * s_inv[j]);
      }
    }
    if (warp == SOFTMAX_WARP && cluster_merge) {
      const float my_lse = lane < num_q_heads ? (s_m[lane] + log2f(s_l[lane])) * kLn2 : -INFINITY;
#pragma unroll 1
      for (int r = 0; r < num_splits; ++r) dsmem_st_f32(dsmem_addr(smem_u32(&s_lse_all[split][lane]), r), my_lse);
    } else if (warp == SOFTMAX_WARP && lane < num_q_heads) {
      const float lse = (s_m[lane] + log2f(s_l[lane])) * kLn2;
      const int64_t orow = (int64_t)i * num_q_heads + lane;
      if (num_splits == 1) { if (lse_out) lse_out[orow] = lse; }
      else part_lse[orow * num_splits + split] = lse;
    }
  }

  // ---- (a5) the last split of the request to arrive merges the partials; release TMEM -------------------
  if (tid == 64) VX_TRACE_STAMP(cta, 8);                // epilogue stored
  tc_fence_before();
  if (cluster_merge) {
    cluster_sync();                                      // every split's tile and LSE are in place
    if (tid == 0) VX_TRACE_STAMP(cta, 9);
    merge_cluster<THREADS_DECODE>(sm + OFF_PAIR, s_lse_all, reinterpret_cast<float (*)[NH]>(sm + OFF_PAIR + 96 * 1024), i, num_q_heads, num_splits, split,
                  out, lse_out);
    if (tid == 0) VX_TRACE_STAMP(cta, 10);
    cluster_sync_relaxed();                              // my tile stays until every peer has read it
  } else if (num_splits > 1) {
    if (last_split_arrives(unit_counter + i, num_splits, &s_last))
      merge_splits(part_o, part_lse, i, num_q_heads, num_splits, out, lse_out, sm + OFF_PAIR);
  }
  __syncthreads();
  if (tid == 0) VX_TRACE_STAMP(cta, 11);
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
}

VX_TRACE_SETTER(vx_trace_set_decode_mla)

bool mla_tc_supported(const vx_geom& g) {
  return g.kv_shared && g.dtype == VX_DT_BF16 && g.kv_format == VX_KV_SAME && g.num_kv_heads == 1 && g.qk_dim == mla::D && g.v_dim == mla::DV &&
         g.page_size == mla::PAGE && g.num_q_heads <= mla::NH;
}

// tensor map over the latent pool: dims (channel, token in page, page), box = 64 channels x 64 tokens, 128-byte swizzle
cudaError_t make_latent_map(CUtensorMap* map, const vx_kv_pool& pool) {
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn encode = nullptr;
  if (!encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return e;
    if (qres != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
    encode = reinterpret_cast<encode_fn>(fn);
  }
  if (pool.num_pool_pages <= 0) return cudaErrorInvalidValue;
  const cuuint64_t dims[3] = {(cuuint64_t)mla::D, (cuuint64_t)mla::PAGE, (cuuint64_t)pool.num_pool_pages};
  const cuuint64_t strides[2] = {(cuuint64_t)pool.stride_token * 2, (cuuint64_t)pool.stride_page * 2};
  const cuuint32_t box[3] = {64, (cuuint32_t)mla::PAGE, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = encode(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(pool.k), dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

int decode_mla_splits(const vx_ctx* c, int n_req, int max_budget) {
  int best = 1, best_cost = 1 << 30;
  for (int sp = 1; sp <= kMaxSplits && sp <= max_budget && sp <= c->g.num_q_heads; ++sp) {   // partial buffer: splits <= Hq
    const int waves = (n_req * sp + c->num_sms - 1) / c->num_sms;
    const int cost = waves * ((max_budget + sp - 1) / sp + 2);
    if (cost < best_cost) { best_cost = cost; best = sp; }
  }
  return best;
}

cudaError_t launch_decode_mla_tc(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                 const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                 int32_t max_budget, void* out, float* lse, cudaStream_t s, const DecodeOpts& opt) {
  const vx_geom& g = c->g;
  if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(decode_mla_kernel), c->device, mla::SMEM_BYTES_DECODE)) return e;
  CUtensorMap kmap;
  if (cudaError_t e = make_latent_map(&kmap, pool)) return e;
  // one CTA per SM (221 KB of shared memory): whole waves of equal CTAs,
  // cost(sp) = waves x (pages per CTA + ~2 pages of pipeline fill and epilogue)
  const int n_req = opt.rr.count < 0 ? pt.batch : opt.rr.count;
  const int best = decode_mla_splits(c, n_req, max_budget);
  dim3 grid(best, 1, n_req);
  // splits of 2, 4 or 8: the splits of a request form a thread-block cluster and merge through shared memory
  const int cluster = (best == 2 || best == 4 || best == 8) ? best : 1;
  cudaError_t e = launch_kernel_cluster(decode_mla_kernel, grid, dim3(mla::THREADS_DECODE), (size_t)mla::SMEM_BYTES_DECODE, s, opt.pdl, cluster, kmap,
                                static_cast<const __nv_bfloat16*>(q), g.num_q_heads, g.sm_scale * opt.scale_mul * mla::kLog2e, pt.seq_lens,
                                sel_phys, sel_logical, sel_count, max_budget, best, c->ws.part_o, c->ws.part_lse,
                                c->ws.unit_counter, static_cast<__nv_bfloat16*>(opt.summary_upd), g.summary_kind,
                                static_cast<__nv_bfloat16*>(out), lse, opt.rr.begin, opt.budget, cluster > 1 ? 1 : 0, opt.out_scale);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace vx
