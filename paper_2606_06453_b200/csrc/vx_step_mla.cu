// vx_step_mla.cu -- (a6) the whole decode step of one MLA request in ONE kernel: (a2) page scores -> (a3) top-k pages ->
// (a4) sparse paged decode -> (a5) split merge, with (a1) for the newest page folded in.  PAPER.md:188 (persistent programs
// over the iteration's planned work list), :190 (fusion "to reduce intermediate memory traffic"), :202 / :262 (the role of
// the paper's own cuda_mla backend); the arithmetic of each step is that of vx_score.cu / vx_select.cuh / vx_decode_mla.cu.
//
// The whole decode step of one request in ONE kernel (a2 -> a3 -> a4 -> a5, a1 folded in):
// the cluster that owns the request (its splits) first streams the request's summary rows through the (still idle)
// page ring with bulk copies -- each CTA a contiguous share of the logical pages, scores S = [Qm | Qp] . [m | M]
// (vx_score.cu's collapsed SUM form, same summation order, so the scores are bit-identical to vx_page_score's)
// pushed into every CTA's shared memory -- then every CTA runs the exact selection of vx_select.cuh on the
// request's scores (identical results, no broadcast), writes its split's share of the block table, and goes straight
// into the tcgen05 loop.  Three dependent grids become one: the requests of a batch have different lengths, so while
// one cluster selects (no HBM traffic) the others stream, and the per-kernel ramps and tails are paid once
// (PAPER.md:188 persistent programs over a planned work list, :190 fusion "to reduce intermediate memory traffic").
#include <cuda.h>
#include <cstdlib>
#include "vx_mla.cuh"
#include "vx_select.cuh"

namespace vx {

struct MlaStepArgs {
  const __nv_bfloat16* summary;      // summary pool, rows of row_chunks * 8 elements, addressed by physical page id
  const int32_t* page_indptr;        // [batch + 1]
  const int32_t* page_indices;       // [total_pages]
  const int32_t* budget;             // [batch], pages incl. forced
  int32_t* sel_count;                // [batch] out
  int n_sink, n_local;
  int row_chunks;                    // 16-byte chunks per summary row: 144 envelope [min | max], 72 centroid
  int p_cap;                         // pt.max_pages_per_req rounded up to 32: sizes the score / id arrays in shared memory
};

__device__ __forceinline__ void bulk_row_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// the staged Q rows (row pitch F_Q_PITCH, head = lane) -> TMEM lanes 0..31, 288 columns.  Called by ONE warp with warp % 4 == 0.
// (A plain function on purpose: with this or the loads that feed it wrapped in a capturing lambda the kernel measured 3 us longer.)
__device__ __forceinline__ void staged_q_to_tmem(const uint8_t* rows, uint32_t tmem_q, int lane) {
  using namespace mla;
  const uint4* qrow = reinterpret_cast<const uint4*>(rows + lane * F_Q_PITCH);
#pragma unroll 1
  for (int c = 0; c < D / 64; ++c) {                   // 64 channels = 32 columns at a time
    float w[32];
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      const uint4 v = qrow[c * 8 + e];
      w[4 * e + 0] = __uint_as_float(v.x); w[4 * e + 1] = __uint_as_float(v.y);
      w[4 * e + 2] = __uint_as_float(v.z); w[4 * e + 3] = __uint_as_float(v.w);
    }
    tmem_st32(tmem_q + 32 * c, w);
  }
  tc_fence_before();
}

__global__ void __launch_bounds__(mla::THREADS, 1)
step_mla_kernel(const __grid_constant__ CUtensorMap kmap, const __nv_bfloat16* __restrict__ q, int num_q_heads,
                float scale_log2, const int32_t* __restrict__ seq_lens, int32_t* __restrict__ sel_phys,
                int32_t* __restrict__ sel_logical, int max_budget, int num_splits, __nv_bfloat16* __restrict__ summary_upd,
                int summary_kind, __nv_bfloat16* __restrict__ out, float* __restrict__ lse_out, const MlaStepArgs fa) {
  // grid (num_splits, 1, batch), launched as clusters of num_splits CTAs: cluster = request, rank = split
  using namespace mla;
  constexpr int NT = THREADS;
  const bool cluster_merge = num_splits > 1;
  extern __shared__ __align__(1024) uint8_t smem_raw[];   // swizzle atoms need 1024-byte alignment
  __shared__ __align__(8) uint64_t s_bar[N_BARS];
  __shared__ __align__(8) uint64_t s_fbar[F_SLOTS_MAX * F_WARPS + 1];   // fused front end: the stream warps' stage barriers, staged Q rows consumed
  __shared__ int s_mylist[2][F_MAX_LIST];              // fused step: my split's share of the block table (physical, logical)
  __shared__ uint32_t s_tmem;
  __shared__ float s_fac[2][NH];                       // lazy-rescale factors of page p (buffer p & 1)
  __shared__ int s_flag[2];                            // ... and whether any head needs them
  __shared__ float s_l[NH], s_m[NH], s_inv[NH];        // final denominators / references
  __shared__ float s_lse_all[kMaxClusterSplits][NH];   // cluster merge: every split's per-head LSE (pushed by its CTA)

  const int split = blockIdx.x, i = blockIdx.z;
  const int tid = threadIdx.x, warp = tid / kWarp, lane = tid % kWarp;
  [[maybe_unused]] const int cta = blockIdx.z * gridDim.x + blockIdx.x;
  if (tid == 0) { VX_TRACE_STAMP(cta, 0); VX_TRACE_SMID(cta); }
  const uint32_t base = smem_u32(smem_raw);
  if (base & 1023u) __trap();                          // (the static variables above end below 3 KB; the driver honours the alignment)
  uint8_t* sm = smem_raw;
  const uint32_t bar0 = smem_u32(&s_bar[0]);
  auto bar = [&](int idx) -> uint32_t { return bar0 + 8u * (uint32_t)idx; };
  const uint32_t fbar0 = smem_u32(&s_fbar[0]);
  auto fbar = [&](int idx) -> uint32_t { return fbar0 + 8u * (uint32_t)idx; };
  const int n_tok = seq_lens[i];
  const int newest_page = (n_tok - 1) / PAGE;
  // fused step: this CTA's share [c_begin, c_end) of the request's logical pages in the summary stream; the producer
  // warp's first page ids are requested now, under the barrier / TMEM set-up
  int row0 = 0, k_budget = 0, c_begin = 0, c_end = 0, ids_cur = 0, ids_nxt = 0;
  // stream warp w = warp - 1 takes the groups g = w, w + 7, .. of F_PG pages; lane l of its m-th id block holds the page
  // id of row l % 4 of its (8 m + l / 4)-th group
  auto my_page = [&](int blk, int l) -> int { return c_begin + F_PG * ((warp - 1) + F_WARPS * (8 * blk + (l >> 2))) + (l & 3); };
  // fused step: the Q rows are requested at entry (warps 2..5), ahead of everything that can wait
  constexpr int Q_IT = NH * CHUNKS / SOFTMAX_THREADS;  // 18 independent 16-byte loads per thread
  static_assert(NH * CHUNKS % SOFTMAX_THREADS == 0, "Q staging");
  uint4 qv_early[Q_IT];
  {
    if (warp >= 2 && warp <= 5) {
#pragma unroll
      for (int k = 0; k < Q_IT; ++k) {
        const int x = tid - 64 + k * SOFTMAX_THREADS, h = x / CHUNKS, c = x % CHUNKS;
        qv_early[k] = h < num_q_heads ? *reinterpret_cast<const uint4*>(q + ((int64_t)i * num_q_heads + h) * D + c * 8)
                                      : make_uint4(0, 0, 0, 0);
      }
    }
  }
  {
    row0 = fa.page_indptr[i];
    k_budget = max(0, min(fa.budget[i], max_budget));
    const int P = newest_page + 1;
    c_begin = (int)((int64_t)P * split / num_splits);
    c_end = (int)((int64_t)P * (split + 1) / num_splits);
    if (warp >= 1) {
      ids_cur = my_page(0, lane) < c_end ? fa.page_indices[row0 + my_page(0, lane)] : 0;
      ids_nxt = my_page(1, lane) < c_end ? fa.page_indices[row0 + my_page(1, lane)] : 0;
    }
  }

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
    {
      for (int s = 0; s < F_SLOTS_MAX * F_WARPS; ++s) mbar_init(fbar(s), 1);
      mbar_init(fbar(F_SLOTS_MAX * F_WARPS), 2);       // the query-vector build and the TMEM store have both read the staged Q rows
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&kmap) : "memory");
  }
  tc_fence_before();
  if (num_splits > 1) cluster_sync();             // every CTA of the cluster runs before anyone pushes scores into it
  else __syncthreads();
  tc_fence_after();
  if (tid == 0) VX_TRACE_STAMP(cta, 1);
  const uint32_t tmem = s_tmem;
  // fused front end: where things sit (see the layout note at F_PG)
  const int tail_off = SMEM_BYTES - 8 * fa.p_cap;
  const int nslot = min(F_SLOTS_MAX, (tail_off - OFF_PAIR) / (F_WARPS * F_STAGE_BYTES));   // stages per stream warp
  // Q[32 x 576] -> TMEM lanes 0..31 (heads), 288 columns (zero rows past Hq): coalesced through the (still
  // idle) ring, row pitch padded to 1168 B so that the per-head reads are bank-conflict free
  constexpr int Q_PITCH = F_Q_PITCH;
  const int q_off = OFF_PAIR + (nslot - 1) * F_WARPS * F_STAGE_BYTES;   // the last slot group
  int cnt;
  {
    // ===== (a2) + (a3) of THIS request, on the cluster that will decode it =====================================
    const int P = newest_page + 1;                     // logical pages of the request
    const int n_groups = (c_end - c_begin + F_PG - 1) / F_PG;
    const uint32_t row_bytes = (uint32_t)fa.row_chunks * 16u;
    float* s_qvec = reinterpret_cast<float*>(sm + OFF_F_QVEC);
    float* s_scores = reinterpret_cast<float*>(sm + tail_off);
    int* s_phys = reinterpret_cast<int*>(sm + tail_off + 4 * fa.p_cap);
    constexpr int FB_QFREE = F_SLOTS_MAX * F_WARPS;
    if (warp == 0) {
      // ---- warp 0 (idle while the summaries stream): Q rows, once staged by warps 2..5 -> tensor memory
      asm volatile("bar.sync 3, %0;" ::"n"(SOFTMAX_THREADS + kWarp) : "memory");
      staged_q_to_tmem(sm + q_off, tmem + TM_Q, lane);
      __syncwarp();
      if (lane == 0) mbar_arrive(fbar(FB_QFREE));
    } else {
      // ---- stream warps 1..7: each runs a PRIVATE ring of nslot stages -- it issues its own bulk copies (one per summary
      // row, lanes 4 (m % 8) .. +3 hold the ids of the warp's m-th group), waits on its own barriers and refills a slot
      // as soon as it has consumed it: no producer warp (one warp issuing every copy of the CTA capped the stream at
      // ~45 GB/s per SM, ~500 cycles per stage plus ~50 per copy), no cross-warp hand-over, and a warp meets the phases
      // of its barriers in order.
      const int cw = warp - 1;
      const int n_my = n_groups > cw ? (n_groups - cw + F_WARPS - 1) / F_WARPS : 0;       // my groups
      const int n_first = min(n_my, nslot - 1);        // my ring has nslot slots; the last slot group still holds the staged Q rows
      int blk = 0;                                     // id block of ids_cur (8 groups)
      auto push_ids = [&](int b_, int id) {            // the ids go to every CTA of the cluster (the block table is built from them)
        const int page = my_page(b_, lane);
        if (page < c_end) {
          if (num_splits == 1) s_phys[page] = id;
          else
            for (int r = 0; r < num_splits; ++r) dsmem_st_u32(dsmem_addr(smem_u32(&s_phys[page]), r), (uint32_t)id);
        }
      };
      auto issue = [&](int m) {                        // my m-th group -> slot m % nslot
        const int slot = m % nslot;
        const int first = c_begin + F_PG * (cw + F_WARPS * m), count = min(F_PG, c_end - first);
        const uint32_t fb = fbar(slot * F_WARPS + cw);
        const int id = (m >> 3) == blk ? ids_cur : ids_nxt;
        if (lane == 4 * (m & 7)) mbar_expect_tx(fb, (uint32_t)count * row_bytes);
        __syncwarp();
        if ((lane >> 2) == (m & 7) && (lane & 3) < count)
          bulk_row_g2s(base + OFF_PAIR + (uint32_t)((slot * F_WARPS + cw) * F_PG + (lane & 3)) * F_MAX_ROW_BYTES,
                       reinterpret_cast<const uint8_t*>(fa.summary) + (int64_t)id * row_bytes, row_bytes, fb);
      };
      push_ids(0, ids_cur);
      for (int m = 0; m < n_first; ++m) issue(m);
      if (cw == 0 && lane == 0) VX_TRACE_STAMP(cta, 12);
      if (warp >= 2 && warp <= 5) {
#pragma unroll
      for (int k = 0; k < Q_IT; ++k) {                 // the Q rows requested at entry -> staged (coalesced, padded pitch)
        const int x = tid - 64 + k * SOFTMAX_THREADS, h = x / CHUNKS, c = x % CHUNKS;
        *reinterpret_cast<uint4*>(sm + q_off + h * Q_PITCH + c * 16) = qv_early[k];
      }
      softmax_barrier();
      asm volatile("bar.arrive 3, %0;" ::"n"(SOFTMAX_THREADS + kWarp) : "memory");   // warp 0 may move them into tensor memory
      // ---- the query vector of the collapsed SUM form, in vx_score.cu's summation order (three head groups of
      // ceil(g / 3) heads, each summed head by head, then (p0 + p1) + p2): envelope [Qm | Qp], centroid [Qsum]
      const bool envelope = fa.row_chunks == 2 * CHUNKS;
      for (int c = tid - 64; c < CHUNKS; c += SOFTMAX_THREADS) {
        const int per = (num_q_heads + 2) / 3;
        float tp[8], tm[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) { tp[x] = 0.f; tm[x] = 0.f; }
#pragma unroll 1
        for (int gi = 0; gi < 3; ++gi) {
          float qp[8], qm[8];
#pragma unroll
          for (int x = 0; x < 8; ++x) { qp[x] = 0.f; qm[x] = 0.f; }
          const int h1 = min(gi * per + per, num_q_heads);
          for (int h = gi * per; h < h1; ++h) {
            float f[8];
            Elem<__nv_bfloat16>::unpack(*reinterpret_cast<const uint4*>(sm + q_off + h * Q_PITCH + c * 16), f);
#pragma unroll
            for (int x = 0; x < 8; ++x) {
              if (envelope) { qp[x] += fmaxf(f[x], 0.f); qm[x] += fminf(f[x], 0.f); }
              else qp[x] += f[x];
            }
          }
#pragma unroll
          for (int x = 0; x < 8; ++x) {                // gi = 0: 0 + p0;  1: p0 + p1;  2: (p0 + p1) + p2
            tp[x] = gi == 0 ? qp[x] : tp[x] + qp[x];
            tm[x] = gi == 0 ? qm[x] : tm[x] + qm[x];
          }
        }
#pragma unroll
        for (int x = 0; x < 8; ++x) {
          if (envelope) { s_qvec[c * 8 + x] = tm[x]; s_qvec[D + c * 8 + x] = tp[x]; }
          else s_qvec[c * 8 + x] = tp[x];
        }
      }
      }
      asm volatile("bar.sync 2, %0;" ::"n"(THREADS - kWarp) : "memory");   // warps 1..7: the query vector is complete
      if (tid == 64) mbar_arrive(fbar(FB_QFREE));
      bool q_free = false;                             // the last slot group joins my ring once both readers of the staged Q rows are done
      // ---- consume: the four rows of a stage as independent accumulation chains (the dot product of a row is a 40-deep
      // FMA chain per lane).  Summation order = vx_score.cu's: per lane chunk by chunk, then the xor tree 16, 8, 4, 2, 1
      // (here in its transposed form: the same tree, evaluated only in the lanes that keep the row).
      constexpr int NIT = (2 * CHUNKS + kWarp - 1) / kWarp;     // 5 chunks per lane (envelope), 3 used by centroid rows
      float qreg[NIT][8];
#pragma unroll
      for (int t = 0; t < NIT; ++t) {
        const int c = lane + t * kWarp;
#pragma unroll
        for (int e = 0; e < 8; ++e) qreg[t][e] = c < fa.row_chunks ? s_qvec[c * 8 + e] : 0.f;
      }
      static_assert(F_PG == 4, "a stage is four rows: one transposed butterfly");
      for (int m = 0; m < n_my; ++m) {
        if (!q_free) {                                 // (warp-uniform; blocking only when my next group is the one that waits for it)
          const bool ready = m == n_first || __shfl_sync(0xffffffffu, lane == 0 ? (int)mbar_test(fbar(FB_QFREE), 0) : 0, 0) != 0;
          if (ready) {
            if (m == n_first) mbar_wait(fbar(FB_QFREE), 0);
            q_free = true;
            if (n_first < n_my) issue(n_first);
          }
        }
        const int slot = m % nslot;
        const int first = c_begin + F_PG * (cw + F_WARPS * m), count = min(F_PG, c_end - first);
        if ((m & 7) == 0 && m > 0) {                   // my next block of 32 ids
          ++blk;
          ids_cur = ids_nxt;
          ids_nxt = my_page(blk + 1, lane) < c_end ? fa.page_indices[row0 + my_page(blk + 1, lane)] : 0;
          push_ids(blk, ids_cur);
        }
        mbar_wait(fbar(slot * F_WARPS + cw), (m / nslot) & 1);
        if (m == 0 && cw == 0 && lane == 0) VX_TRACE_STAMP(cta, 13);
        const uint8_t* stage = sm + OFF_PAIR + (size_t)(slot * F_WARPS + cw) * F_STAGE_BYTES + lane * 16;
        uint4 v[4][NIT];
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
#pragma unroll
          for (int t = 0; t < NIT; ++t) {
            const bool ok = kk < count && lane + t * kWarp < fa.row_chunks;
            v[kk][t] = ok ? *reinterpret_cast<const uint4*>(stage + kk * F_MAX_ROW_BYTES + t * kWarp * 16) : make_uint4(0, 0, 0, 0);
          }
        }
        float part[4];
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          float acc = 0.f;
#pragma unroll
          for (int t = 0; t < NIT; ++t) {
            float f[8];
            Elem<__nv_bfloat16>::unpack(v[kk][t], f);
#pragma unroll
            for (int e = 0; e < 8; ++e) acc = fmaf(qreg[t][e], f[e], acc);
          }
          part[kk] = acc;
        }
        // the stage's rows have been used (their loads are complete): refill the slot with my group m + nslot
        fence_async_proxy();
        __syncwarp();
        if (m + nslot < n_my) issue(m + nslot);
        float a2[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const bool up = lane & 16;
          a2[j] = (up ? part[j + 2] : part[j]) + __shfl_xor_sync(0xffffffffu, up ? part[j] : part[j + 2], 16);
        }
        const bool up8 = lane & 8;
        float tot = (up8 ? a2[1] : a2[0]) + __shfl_xor_sync(0xffffffffu, up8 ? a2[0] : a2[1], 8);
        tot += __shfl_xor_sync(0xffffffffu, tot, 4);
        tot += __shfl_xor_sync(0xffffffffu, tot, 2);
        tot += __shfl_xor_sync(0xffffffffu, tot, 1);
        const int r = lane >> 3;                       // lanes [8k, 8k + 8) hold row k
        if (r < count) {                               // the score of logical page first + r goes to every CTA of the cluster
          if (num_splits == 1) { if ((lane & 7) == 0) s_scores[first + r] = tot; }
          else if ((lane & 7) < num_splits) dsmem_st_f32(dsmem_addr(smem_u32(&s_scores[first + r]), lane & 7), tot);
        }
      }
    }
    // ---- every CTA of the cluster has pushed its share: the request's scores and page ids are complete in my shared memory
    if (num_splits > 1) cluster_sync();
    else __syncthreads();
    if (tid == 0) VX_TRACE_STAMP(cta, 14);
    SelectScratch& scratch = *reinterpret_cast<SelectScratch*>(sm + OFF_PAIR);
    static_assert(sizeof(SelectScratch) <= 2 * F_STAGE_BYTES && THREADS == 256, "selection scratch sits in the drained stages 0 and 1");
    cnt = cta_select_pages<THREADS>(scratch, reinterpret_cast<uint32_t*>(s_scores), P, k_budget, fa.n_sink, fa.n_local);
    if (tid == 0) VX_TRACE_STAMP(cta, 2);
    {                                                  // my split's share of the block table: shared memory for the loop below,
      const int per = (cnt + num_splits - 1) / num_splits;     // global for the caller (its arrays or the workspace)
      const int rb = min(split * per, cnt), re = min(rb + per, cnt);
      int32_t* gp = sel_phys + (int64_t)i * max_budget;
      int32_t* gl = sel_logical + (int64_t)i * max_budget;
      for (int r = rb + tid; r < re; r += THREADS) {
        const int j = scratch.hist[r];
        const int phys = s_phys[j];
        s_mylist[0][r - rb] = phys;
        s_mylist[1][r - rb] = j;
        gp[r] = phys;
        gl[r] = j;
      }
      if (split == 0) {
        for (int r = cnt + tid; r < max_budget; r += THREADS) { gp[r] = -1; gl[r] = -1; }
        if (tid == 0) fa.sel_count[i] = cnt;
      }
    }
    tc_fence_before();
    __syncthreads();                                   // the scratch is dead; my list is in place; Q sits in tensor memory
    tc_fence_after();
    if (tid == 0) VX_TRACE_STAMP(cta, 3);
  }

  const int per_split = (cnt + num_splits - 1) / num_splits;
  const int r_begin = min(split * per_split, cnt), r_end = min(r_begin + per_split, cnt);
  const int n_pages = r_end - r_begin;
  auto list_phys = [&](int p) -> int { return s_mylist[0][p]; };   // my p-th page
  auto list_log = [&](int p) -> int { return s_mylist[1][p]; };
  const uint32_t p_base = base + OFF_P;

  if (n_pages == 0 && cluster_merge) {                 // empty split: a zero tile with weight zero
    for (int e = tid; e < NH * DV / 4; e += NT) reinterpret_cast<float4*>(sm + OFF_PAIR)[e] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid < NH)
      for (int r = 0; r < num_splits; ++r) dsmem_st_f32(dsmem_addr(smem_u32(&s_lse_all[split][tid]), r), -INFINITY);
  } else if (n_pages == 0) {                           // a request without pages to read (budget 0): zeros, lse = -inf
    for (int e = tid; e < num_q_heads * DV; e += NT) out[(int64_t)i * num_q_heads * DV + e] = __float2bfloat16_rn(0.f);
    if (tid < num_q_heads && lse_out) lse_out[(int64_t)i * num_q_heads + tid] = -INFINITY;
  } else if (warp == 0) {
    // ===== TMA producer: page p -> ring page p % 3 (4 pair slots + 1 RoPE slot), one full barrier per page =====
    static_assert(N_PAIR == N_ROPE * PAIRS_PER_PAGE, "the ring is a whole number of pages");
    int my_phys = 0;
    for (int p = 0; p < n_pages; ++p) {
      if ((p & 31) == 0) my_phys = p + lane < n_pages ? list_phys(p + lane) : 0;
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
  } else if (warp == 7) {
    // the fused step's spare warp: parked on the last PV's barrier (a hardware-suspended wait) rather than in the
    // cluster barrier below for the whole loop
    mbar_wait(bar(B_PV_DONE + ((n_pages - 1) & 1)), ((n_pages - 1) >> 1) & 1);
  } else if (warp <= 5) {
    // ===== warps 2..5: softmax (warp 4) + rescale helpers, then the epilogue ==============================
    const int sp = warp & 3;                             // TMEM sub-partition this warp may access
    const uint32_t t_lane = tmem + ((uint32_t)(sp * 32) << 16);
    const int pl = n_pages - 1;
    if (warp == SOFTMAX_WARP) {
      // thread = head `lane` (TMEM lane); columns = the 64 tokens of the page
      float m_ref = 0.f, l_sum = 0.f;
      int lg = list_log(0);
      for (int p = 0; p < n_pages; ++p) {
        const int b = p & 1;
        const int valid = min(PAGE, n_tok - lg * PAGE);
        if (p + 1 < n_pages) lg = list_log(p + 1);       // prefetch for the next page
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
      s_inv[lane] = 1.f / l_sum;
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
      const int lg_last = list_log(pl);
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
          *reinterpret_cast<uint4*>(summary_upd + (int64_t)list_phys(pl) * D + cc * 8) = *reinterpret_cast<const uint4*>(o8);
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
        __nv_bfloat16* dst = summary_upd + (int64_t)list_phys(pl) * 2 * D + cc * 8;
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
      if (lse_out) lse_out[(int64_t)i * num_q_heads + lane] = lse;
    }
  }

  // ---- (a5) the splits of the request merge inside their cluster; release TMEM ----------------------------------
  if (tid == 64) VX_TRACE_STAMP(cta, 8);                // epilogue stored
  tc_fence_before();
  if (cluster_merge) {
    cluster_sync();                                      // every split's tile and LSE are in place
    if (tid == 0) VX_TRACE_STAMP(cta, 9);
    merge_cluster<NT>(sm + OFF_PAIR, s_lse_all, reinterpret_cast<float (*)[NH]>(sm + OFF_PAIR + 96 * 1024), i, num_q_heads, num_splits, split,
                  out, lse_out);
    if (tid == 0) VX_TRACE_STAMP(cta, 10);
    cluster_sync();                                      // my tile stays until every peer has read it
  }
  __syncthreads();
  if (tid == 0) VX_TRACE_STAMP(cta, 11);
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
}

VX_TRACE_SETTER(vx_trace_set_step_mla)

bool step_mla_fused_applies(const vx_ctx* c, const vx_page_table& pt, const vx_kv_pool& pool, int32_t max_budget) {
  const vx_geom& g = c->g;
  return mla_tc_supported(g) && g.agg == VX_AGG_SUM && g.n_local >= 1 &&      // (n_local = 0: the summary kernel must run first)
         pt.max_pages_per_req <= mla::F_MAX_PAGES && max_budget <= 8 * mla::F_MAX_LIST && pool.num_pool_pages > 0;
}

// Where it pays (measured on the C4 geometry): batches of up to 8 requests, which run as 8 CTAs per
// request in one wave -- 47-49 us against 70-79 us for the three chained kernels.  From 16 requests on the chained kernels
// win: their score and decode kernels split the BATCH's pages evenly over all SMs, while a cluster streams its own
// request's summaries, so the longest request sets the pace (B = 64: 71.5 against 68.5 us).
bool step_mla_fused_pays(const vx_ctx*, const vx_page_table& pt) { return pt.batch <= 8; }

// splits = cluster size in {1, 2, 4, 8}: whole waves of clusters, cost = waves x (a CTA's share of the summary stream,
// in page equivalents, + its pages + ~3 pages of ramp, selection and epilogue)
static int step_mla_splits(const vx_ctx* c, int n_req, int max_pages_per_req, int max_budget) {
  const int row_bytes = (c->g.summary_kind == VX_SUMMARY_CENTROID ? 1 : 2) * mla::D * 2;
  const int summary_pages = (int)(((int64_t)max_pages_per_req * row_bytes + mla::PAGE_BYTES - 1) / mla::PAGE_BYTES);
  int best = 1, best_cost = 1 << 30;
  for (int sp = 1; sp <= 8 && sp <= max_budget; sp *= 2) {
    if ((max_budget + sp - 1) / sp > mla::F_MAX_LIST) continue;      // a CTA keeps its share of the block table in shared memory
    const int waves = (n_req * sp + c->num_sms - 1) / c->num_sms;
    const int cost = waves * ((summary_pages + max_budget + sp - 1) / sp + 3);
    if (cost < best_cost) { best_cost = cost; best = sp; }
  }
  return best;
}

cudaError_t launch_step_mla_fused(vx_ctx* c, const void* q, const vx_kv_pool& pool, const void* summary,
                                  const vx_page_table& pt, const int32_t* budget, int32_t max_budget, bool update_summary,
                                  int32_t* sel_phys, int32_t* sel_logical, int32_t* sel_count, void* out, float* lse,
                                  cudaStream_t s) {
  const vx_geom& g = c->g;
  if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(step_mla_kernel), c->device, mla::SMEM_BYTES)) return e;
  CUtensorMap kmap;
  if (cudaError_t e = make_latent_map(&kmap, pool)) return e;
  const int splits = step_mla_splits(c, pt.batch, pt.max_pages_per_req, max_budget);
  MlaStepArgs fa;
  fa.summary = static_cast<const __nv_bfloat16*>(summary);
  fa.page_indptr = pt.page_indptr;
  fa.page_indices = pt.page_indices;
  fa.budget = budget;
  fa.sel_count = sel_count;
  fa.n_sink = g.n_sink;
  fa.n_local = g.n_local;
  fa.row_chunks = (g.summary_kind == VX_SUMMARY_CENTROID ? 1 : 2) * mla::CHUNKS;
  fa.p_cap = (pt.max_pages_per_req + 31) / 32 * 32;
  dim3 grid(splits, 1, pt.batch);
  cudaError_t e = launch_kernel_cluster(step_mla_kernel, grid, dim3(mla::THREADS), (size_t)mla::SMEM_BYTES, s, false, splits, kmap,
                                static_cast<const __nv_bfloat16*>(q), g.num_q_heads, g.sm_scale * mla::kLog2e, pt.seq_lens,
                                sel_phys, sel_logical, max_budget, splits,
                                update_summary ? static_cast<__nv_bfloat16*>(const_cast<void*>(summary)) : nullptr, g.summary_kind,
                                static_cast<__nv_bfloat16*>(out), lse, fa);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace vx
