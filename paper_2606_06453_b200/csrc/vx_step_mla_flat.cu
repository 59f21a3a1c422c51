// vx_step_mla_flat.cu -- (a6) the whole decode step of an MLA BATCH in one persistent kernel, one CTA per SM:
// (a2) page scores -> (a3) top-k pages -> (a4) sparse paged decode -> (a5) split merge, (a1) folded in.
// PAPER.md:188 (persistent programs over the iteration's planned work list), :190 (fusion "to reduce intermediate memory
// traffic"), :202 / :262 (the role of the paper's cuda_mla backend).  The arithmetic of each step is that of
// vx_score.cu / vx_select.cuh / vx_decode_mla.cu; what is new is the schedule:
//
//   * The summary stream of the whole batch is cut FLAT over the CTAs (every CTA the same number of rows, whatever the
//     request lengths), in n_waves interleaved waves so that the requests complete one after the other while the
//     stream is still running; seven stream warps per CTA, each with a private ring of bulk copies.  The copies are
//     issued from flat row numbers alone (no look-up of the request before the first copy).
//   * The query vector [Qm | Qp] of request r is built once (by the selection warpgroup of CTA r mod grid) and
//     published through global memory; warp 0 of every CTA keeps the vectors its stream warps need next in three
//     shared-memory slots.
//   * Request r is SELECTED by a separate warpgroup (warps 8..11) of CTA r mod grid the moment its last score has
//     arrived (a release / acquire counter per request) -- while the other warps of that CTA, and all other CTAs, keep
//     streaming.  HBM never waits for a selection.
//   * Decode work is taken from a counter: item = (request, one of `splits` shares of its block table), in request
//     order, i.e. in the order in which the selections become ready.  The tcgen05 pipeline (TMA producer, QK issuer,
//     softmax, PV issuer; vx_decode_mla.cu) runs through a CTA's items with running barrier phases; the last share
//     of a request to arrive merges the partials by LSE.
//   * The last CTA to leave zeroes the step's counters: the kernel is replayable (CUDA graphs) without a memset.
#include <cuda.h>
#include <cstdlib>
#include "vx_mla.cuh"
#include "vx_select.cuh"

namespace vx {

namespace flat {
using namespace mla;
constexpr int NT = 384;                                   // 12 warps: the 8 of the decode pipeline + the selection warpgroup
constexpr int SEL_T0 = 256, SEL_NT = 128, SEL_BAR = 5;    // warps 8..11, their named barrier
constexpr int NQ = 3;                                     // query-vector slots in shared memory
constexpr int QV_FLOATS = 2 * D, QV_BYTES = QV_FLOATS * 4;   // [Qm | Qp] fp32: 4,608 B (centroid: the first half)
constexpr int MAX_WAVES = 8;
constexpr int MAX_BATCH = 224;                            // page_indptr and the CTA's request sequence are staged in the P region
// shared memory while the summaries stream (the P buffers and the page ring are idle until the first decode item):
//   [0, 4608)                        query-vector slot 0
//   [4608, +4 (MAX_BATCH + 1))       page_indptr
//   [OFF_SEQ, +4 (MAX_BATCH + MAX_WAVES))   the requests this CTA's rows belong to, in order
//   [OFF_PAIR + (k * F_WARPS + w) * F_STAGE_BYTES, ..)   slot k of stream warp w's ring
//   [tail, SMEM_BYTES)               query-vector slots 1, 2; the selection scratch; the selection keys (4 p_cap bytes)
constexpr int OFF_INDPTR = QV_BYTES;
constexpr int OFF_SEQ = OFF_INDPTR + 4 * (MAX_BATCH + 1) + 12;
static_assert(OFF_SEQ + 4 * (MAX_BATCH + MAX_WAVES) <= OFF_PAIR, "indptr and sequence fit below the ring");
constexpr int TAIL_FIXED = (NQ - 1) * QV_BYTES + ((int)sizeof(SelectScratch) + 15) / 16 * 16;
// sync words (workspace, zero between steps)
constexpr int SY_NEXT = 0, SY_DONE_CTAS = 1, SY_PER_REQ = 2;   // then qvec_ready[B], rows_done[B], sel_ready[B]
}  // namespace flat

struct MlaFlatArgs {
  const __nv_bfloat16* q;            // [batch, Hq, 576]
  const __nv_bfloat16* summary;      // summary pool, rows of row_chunks * 16 bytes, addressed by physical page id
  const int32_t* page_indptr;        // [batch + 1]
  const int32_t* page_indices;       // [total_pages]
  const int32_t* seq_lens;           // [batch]
  const int32_t* budget;             // [batch], pages incl. forced
  int32_t* sel_phys;                 // [batch, max_budget] out (the caller's arrays or the workspace)
  int32_t* sel_logical;
  int32_t* sel_count;                // [batch]
  float* scores;                     // [total_pages] workspace
  float* qvec;                       // [batch, 1152] workspace
  int32_t* sync;                     // [2 + 3 batch] workspace, zero on entry, zero on exit
  float* part_o;                     // [batch, splits, 512, 32] workspace
  float* part_lse;                   // [batch, Hq, splits]
  int32_t* unit_counter;             // [batch] split arrivals, zero between steps
  __nv_bfloat16* summary_upd;        // non-null: rebuild the newest page's summary row (a1)
  __nv_bfloat16* out;                // [batch, Hq, 512]
  float* lse_out;                    // [batch, Hq] or null
  int batch, total_pages, num_q_heads, max_budget, n_sink, n_local;
  int row_chunks;                    // 16-byte chunks per summary row: 144 envelope [min | max], 72 centroid
  int p_cap;                         // max pages per request rounded up to 32: sizes the selection keys
  int splits, n_waves, summary_kind;
  float scale_log2;
};

__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_gpu(int* p, int v) {
  asm volatile("red.release.gpu.global.add.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ uint4 ldcg_u32x4(const void* p) {
  uint4 v;
  asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ int ldcg_s32(const int* p) {
  int v;
  asm volatile("ld.global.cg.s32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ void flat_bulk_row_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// the request that owns flat row x: the r with indptr[r] <= x < indptr[r + 1] (requests without pages are skipped)
__device__ __forceinline__ int flat_find_request(const int* indptr, int batch, int x) {
  int lo = 0, hi = batch;                                // answer in [lo, hi)
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (indptr[mid] <= x) lo = mid; else hi = mid;
  }
  return lo;
}

__global__ void __launch_bounds__(flat::NT, 1)
step_mla_flat_kernel(const __grid_constant__ CUtensorMap kmap, const MlaFlatArgs a) {
  using namespace flat;
  extern __shared__ __align__(1024) uint8_t smem_raw[];   // swizzle atoms need 1024-byte alignment
  __shared__ __align__(8) uint64_t s_bar[N_BARS];
  __shared__ __align__(8) uint64_t s_qbar[2 * NQ];       // query-vector slot full (count 1) / empty (count F_WARPS)
  __shared__ int s_mylist[2][F_MAX_LIST];                // the item's share of the block table (physical, logical)
  __shared__ uint32_t s_tmem;
  __shared__ float s_fac[2][NH];
  __shared__ int s_flag[2];
  __shared__ float s_l[NH], s_m[NH], s_inv[NH];
  __shared__ int s_item, s_last, s_nseq;
  __shared__ int s_slice_a[MAX_WAVES], s_slice_b[MAX_WAVES], s_slice_g[MAX_WAVES + 1];   // my slices: first row, end row, first stage

  const int tid = threadIdx.x, warp = tid / kWarp, lane = tid % kWarp;
  const int cta = blockIdx.x, G = gridDim.x;
  if (tid == 0) { VX_TRACE_STAMP(cta, 0); VX_TRACE_SMID(cta); }
  const uint32_t base = smem_u32(smem_raw);
  if (base & 1023u) __trap();
  uint8_t* sm = smem_raw;
  const uint32_t bar0 = smem_u32(&s_bar[0]);
  auto bar = [&](int idx) -> uint32_t { return bar0 + 8u * (uint32_t)idx; };
  const uint32_t qbar0 = smem_u32(&s_qbar[0]);
  auto qfull = [&](int s) -> uint32_t { return qbar0 + 8u * (uint32_t)s; };
  auto qempty = [&](int s) -> uint32_t { return qbar0 + 8u * (uint32_t)(NQ + s); };
  const int B = a.batch, T = a.total_pages, NW = a.n_waves;
  int* const sy = a.sync;
  int* const qvec_ready = sy + SY_PER_REQ;
  int* const rows_done = sy + SY_PER_REQ + B;
  int* const sel_ready = sy + SY_PER_REQ + 2 * B;
  int* s_indptr = reinterpret_cast<int*>(sm + OFF_INDPTR);
  int* s_seq = reinterpret_cast<int*>(sm + OFF_SEQ);

  // ---- prologue: this CTA's slices of the flat row list (pure arithmetic), page_indptr, barriers, TMEM ------------------
  // wave w covers rows [T w / NW, T (w + 1) / NW); inside it CTA c takes the c-th of G equal parts; every boundary is
  // rounded down to a multiple of 4 rows (a stage of the stream is 4 consecutive rows)
  auto bound = [&](int w, int cc) -> int {
    if (cc == G) { ++w; cc = 0; }
    if (w >= NW) return T;
    const int64_t ws = (int64_t)T * w / NW, we = (int64_t)T * (w + 1) / NW;
    return (int)(ws + (we - ws) * cc / G) & ~3;
  };
  const int st = tid - SEL_T0;                           // thread of the selection warpgroup (warps 8..11)
  auto sel_sync = [&]() { asm volatile("bar.sync %0, %1;" ::"n"(SEL_BAR), "n"(SEL_NT) : "memory"); };
  const bool envelope = a.row_chunks == 2 * CHUNKS;
  if (warp >= 8) {
    // ---- the selection warpgroup starts with the query vectors of its requests: every stream of the batch waits for them,
    // so the Q rows (one contiguous block per request) are pulled into L2 at entry and nothing else comes first
    if (st == 0 && cta < B) l2_prefetch(a.q + (int64_t)cta * a.num_q_heads * D, (uint32_t)(a.num_q_heads * D * 2));
    for (int r = cta; r < B; r += G) {
      // [Qm | Qp] of the collapsed SUM form, in vx_score.cu's summation order (three head groups of ceil(g / 3) heads, each
      // summed head by head, then (p0 + p1) + p2); centroid summaries: [Qsum]
      if (st < CHUNKS) {
        const int c = st, per = (a.num_q_heads + 2) / 3;
        constexpr int PER_MAX = (NH + 2) / 3;            // heads per group: 11 loads in flight per thread
        float tp[8], tm[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) { tp[x] = 0.f; tm[x] = 0.f; }
#pragma unroll 1
        for (int gi = 0; gi < 3; ++gi) {
          const int h0 = gi * per, h1 = min(gi * per + per, a.num_q_heads);
          uint4 qv[PER_MAX];
#pragma unroll
          for (int u = 0; u < PER_MAX; ++u)
            qv[u] = h0 + u < h1 ? *reinterpret_cast<const uint4*>(a.q + ((int64_t)r * a.num_q_heads + h0 + u) * D + c * 8)
                                : make_uint4(0, 0, 0, 0);
          float qp[8], qm[8];
#pragma unroll
          for (int x = 0; x < 8; ++x) { qp[x] = 0.f; qm[x] = 0.f; }
#pragma unroll
          for (int u = 0; u < PER_MAX; ++u) {
            if (h0 + u < h1) {
              float f[8];
              Elem<__nv_bfloat16>::unpack(qv[u], f);
#pragma unroll
              for (int x = 0; x < 8; ++x) {
                if (envelope) { qp[x] += fmaxf(f[x], 0.f); qm[x] += fminf(f[x], 0.f); }
                else qp[x] += f[x];
              }
            }
          }
#pragma unroll
          for (int x = 0; x < 8; ++x) {
            tp[x] = gi == 0 ? qp[x] : tp[x] + qp[x];
            tm[x] = gi == 0 ? qm[x] : tm[x] + qm[x];
          }
        }
        float* dst = a.qvec + (int64_t)r * QV_FLOATS;
        if (envelope) {
          *reinterpret_cast<float4*>(dst + c * 8) = make_float4(tm[0], tm[1], tm[2], tm[3]);
          *reinterpret_cast<float4*>(dst + c * 8 + 4) = make_float4(tm[4], tm[5], tm[6], tm[7]);
          *reinterpret_cast<float4*>(dst + D + c * 8) = make_float4(tp[0], tp[1], tp[2], tp[3]);
          *reinterpret_cast<float4*>(dst + D + c * 8 + 4) = make_float4(tp[4], tp[5], tp[6], tp[7]);
        } else {
          *reinterpret_cast<float4*>(dst + c * 8) = make_float4(tp[0], tp[1], tp[2], tp[3]);
          *reinterpret_cast<float4*>(dst + c * 8 + 4) = make_float4(tp[4], tp[5], tp[6], tp[7]);
        }
      }
      sel_sync();
      if (st == 0) { __threadfence(); st_release_gpu(qvec_ready + r, 1); }
    }
    asm volatile("bar.sync 9, 384;" ::: "memory");       // ... then joins the prologue of warps 0..7
  } else {
  if (tid < NW) { s_slice_a[tid] = bound(tid, cta); s_slice_b[tid] = bound(tid, cta + 1); }
  for (int x = tid; x <= B; x += 256) s_indptr[x] = a.page_indptr[x];
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
    for (int s = 0; s < NQ; ++s) { mbar_init(qfull(s), 1); mbar_init(qempty(s), F_WARPS); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&kmap) : "memory");
  }
  tc_fence_before();
  asm volatile("bar.sync 8, 256;" ::: "memory");
  asm volatile("bar.arrive 9, 384;" ::: "memory");
  }
  tc_fence_after();
  if (tid == 0) VX_TRACE_STAMP(cta, 1);
  const uint32_t tmem = s_tmem;
  const int tail_off = SMEM_BYTES - (TAIL_FIXED + 4 * a.p_cap);
  const int nslot = min(F_SLOTS_MAX, (tail_off - OFF_PAIR) / (F_WARPS * F_STAGE_BYTES));   // stages per stream warp
  auto qslot = [&](int s) -> float* { return reinterpret_cast<float*>(s == 0 ? sm : sm + tail_off + (s - 1) * QV_BYTES); };
  const uint32_t row_bytes = (uint32_t)a.row_chunks * 16u;

  // ======================================= (a2) + (a3): the batch's summary stream =====================================
  if (warp == 0) {
    // ---- warp 0: the request sequence of this CTA's rows, then the query vectors its stream warps will need ----------
    if (lane == 0) {
      int n = 0;
      for (int w = 0; w < NW; ++w) {
        const int ra = s_slice_a[w], rb = s_slice_b[w];
        if (rb <= ra) continue;
        const int r_lo = flat_find_request(s_indptr, B, ra), r_hi = flat_find_request(s_indptr, B, rb - 1);
        for (int r = r_lo; r <= r_hi; ++r)
          if (s_indptr[r + 1] > s_indptr[r] && (n == 0 || s_seq[n - 1] != r)) s_seq[n++] = r;
      }
      s_nseq = n;
    }
    __syncwarp();
    asm volatile("bar.sync 4, 256;" ::: "memory");       // warps 0..7: the sequence is in place
    const int nseq = s_nseq;
    for (int k = 0; k < nseq; ++k) {
      const int slot = k % NQ, r = s_seq[k];
      if (k >= NQ) mbar_wait(qempty(slot), ((k / NQ) - 1) & 1);       // every stream warp is past the vector that was here
      if (lane == 0)
        while (ld_acquire_gpu(qvec_ready + r) == 0) __nanosleep(64);
      __syncwarp();
      const uint4* src = reinterpret_cast<const uint4*>(a.qvec + (int64_t)r * QV_FLOATS);
      uint4* dst = reinterpret_cast<uint4*>(qslot(slot));
      uint4 v[QV_BYTES / 16 / kWarp];
#pragma unroll
      for (int e = 0; e < QV_BYTES / 16 / kWarp; ++e) v[e] = ldcg_u32x4(src + lane + e * kWarp);
#pragma unroll
      for (int e = 0; e < QV_BYTES / 16 / kWarp; ++e) dst[lane + e * kWarp] = v[e];
      __syncwarp();
      if (lane == 0) mbar_arrive(qfull(slot));
    }
  } else if (warp < 8) {
    // ---- stream warps 1..7: each runs a PRIVATE ring of nslot stages of 4 consecutive flat rows (vx_step_mla.cu) -----
    const int cw = warp - 1;
    if (lane == 0 && cw == 0) {                          // stage prefix of my CTA's slices
      int g = 0;
      for (int w = 0; w < MAX_WAVES; ++w) {
        s_slice_g[w] = g;
        if (w < NW && s_slice_b[w] > s_slice_a[w]) g += (s_slice_b[w] - s_slice_a[w] + F_PG - 1) / F_PG;
      }
      s_slice_g[MAX_WAVES] = g;
    }
    asm volatile("bar.sync 3, 224;" ::: "memory");       // the stream warps
    const int n_groups = s_slice_g[MAX_WAVES];
    const int n_my = n_groups > cw ? (n_groups - cw + F_WARPS - 1) / F_WARPS : 0;
    // stage g of the CTA -> its first flat row and its row count
    auto stage_rows = [&](int g, int& first, int& count) {
      int w = 0;
#pragma unroll
      for (int x = 1; x < MAX_WAVES; ++x) w += (g >= s_slice_g[x] && s_slice_g[x] < n_groups) ? 1 : 0;
      first = s_slice_a[w] + F_PG * (g - s_slice_g[w]);
      count = min(F_PG, s_slice_b[w] - first);
    };
    // lane l of my m-th id block holds the page id of row l % 4 of my (8 m + l / 4)-th stage
    auto my_id = [&](int blk) -> int {
      const int mm = 8 * blk + (lane >> 2);
      if (mm >= n_my) return 0;
      int first, count;
      stage_rows(cw + F_WARPS * mm, first, count);
      return (lane & 3) < count ? a.page_indices[first + (lane & 3)] : 0;
    };
    int ids_cur = my_id(0), ids_nxt = my_id(1), blk = 0;
    // my m-th stage -> slot m % nslot, as 16-byte cp.async copies (one commit group per stage).  Bulk copies of single
    // 2,304-byte rows capped the stream near 30 GB/s per SM whatever the ring depth (the same rate vx_score.cu reaches on
    // this geometry); the LSU path takes 18 instructions per stage and is bound by HBM.
    constexpr int NIT = (2 * CHUNKS + kWarp - 1) / kWarp;     // 5 chunks per lane (envelope), 3 used by centroid rows
    auto issue = [&](int m) {
      const int slot = m % nslot;
      int first, count;
      stage_rows(cw + F_WARPS * m, first, count);
      const int idreg = (m >> 3) == blk ? ids_cur : ids_nxt;
      uint8_t* dst = sm + OFF_PAIR + (size_t)(slot * F_WARPS + cw) * F_STAGE_BYTES + lane * 16;
#pragma unroll
      for (int kk = 0; kk < F_PG; ++kk) {
        const int id = __shfl_sync(0xffffffffu, idreg, 4 * (m & 7) + kk);
        if (kk < count) {
          const uint8_t* src = reinterpret_cast<const uint8_t*>(a.summary) + (int64_t)id * row_bytes + lane * 16;
#pragma unroll
          for (int t = 0; t < NIT; ++t)
            if (lane + t * kWarp < a.row_chunks) cp_async16(dst + kk * F_MAX_ROW_BYTES + t * kWarp * 16, src + t * kWarp * 16);
        }
      }
      cp_async_commit();
    };
    for (int m = 0; m < nslot; ++m) {                    // (always nslot commit groups: the waits below count them)
      if (m < n_my) issue(m);
      else cp_async_commit();
    }
    if (cw == 0 && lane == 0) VX_TRACE_STAMP(cta, 2);
    asm volatile("bar.sync 4, 256;" ::: "memory");       // the request sequence (warp 0) is in place
    const int nseq = s_nseq;
    float qreg[NIT][8];
    int kcur = 0, cur_r = -1, cur_end = 0, acc_rows = 0;
    for (int m = 0; m < n_my; ++m) {
      const int slot = m % nslot;
      int first, count;
      stage_rows(cw + F_WARPS * m, first, count);
      if ((m & 7) == 0 && m > 0) {                       // my next block of 32 ids
        ++blk;
        ids_cur = ids_nxt;
        ids_nxt = my_id(blk + 1);
      }
      if (nslot == 3) cp_async_wait<2>();                // stage m has landed (the nslot - 1 younger groups may be pending)
      else cp_async_wait<1>();
      __syncwarp();
      if (m == 0 && cw == 0 && lane == 0) VX_TRACE_STAMP(cta, 3);
      const uint8_t* stage = sm + OFF_PAIR + (size_t)(slot * F_WARPS + cw) * F_STAGE_BYTES + lane * 16;
      // (the rows are read from shared memory pass by pass below; the slot is refilled after the last pass)
      int k0 = 0;
      while (k0 < count) {                               // (one pass, unless a request ends inside the stage)
        if (cur_r < 0 || first + k0 >= cur_end) {
          // ---- the rows from here on belong to another request: account for the finished one, take its query vector ----
          if (cur_r >= 0 && acc_rows > 0) {
            __syncwarp();
            if (lane == 0) red_release_gpu(rows_done + cur_r, acc_rows);
          }
          acc_rows = 0;
          int r = cur_r < 0 ? flat_find_request(s_indptr, B, first + k0) : cur_r + 1;
          while (s_indptr[r + 1] <= first + k0) ++r;
          while (s_seq[kcur] != r) {                     // (monotone: my rows only move forward through the sequence)
            // a vector I skip is released only once it has been loaded: my arrival must count for ITS phase of the slot
            mbar_wait(qfull(kcur % NQ), (kcur / NQ) & 1);
            if (lane == 0) mbar_arrive(qempty(kcur % NQ));
            ++kcur;
          }
          mbar_wait(qfull(kcur % NQ), (kcur / NQ) & 1);
          const float* qs = qslot(kcur % NQ);
#pragma unroll
          for (int t = 0; t < NIT; ++t) {
            const int c = lane + t * kWarp;
            if (c < a.row_chunks) {
              const float4 lo = *reinterpret_cast<const float4*>(qs + c * 8), hi = *reinterpret_cast<const float4*>(qs + c * 8 + 4);
              qreg[t][0] = lo.x; qreg[t][1] = lo.y; qreg[t][2] = lo.z; qreg[t][3] = lo.w;
              qreg[t][4] = hi.x; qreg[t][5] = hi.y; qreg[t][6] = hi.z; qreg[t][7] = hi.w;
            } else {
#pragma unroll
              for (int e = 0; e < 8; ++e) qreg[t][e] = 0.f;
            }
          }
          cur_r = r;
          cur_end = s_indptr[r + 1];
        }
        const int k1 = min(count, cur_end - first);     // rows [k0, k1) of the stage belong to cur_r
        // the four rows as independent accumulation chains; summation order = vx_score.cu's: per lane chunk by chunk,
        // then the xor tree 16, 8, 4, 2, 1 (in its transposed form)
        float part[4];
#pragma unroll
        for (int half = 0; half < 2; ++half) {           // two rows at a time: 40 registers of row data, not 80
          uint4 v[2][NIT];
#pragma unroll
          for (int kk = 0; kk < 2; ++kk) {
#pragma unroll
            for (int t = 0; t < NIT; ++t) {
              const bool ok = 2 * half + kk < count && lane + t * kWarp < a.row_chunks;
              v[kk][t] = ok ? *reinterpret_cast<const uint4*>(stage + (2 * half + kk) * F_MAX_ROW_BYTES + t * kWarp * 16) : make_uint4(0, 0, 0, 0);
            }
          }
#pragma unroll
          for (int kk = 0; kk < 2; ++kk) {
            float acc = 0.f;
#pragma unroll
            for (int t = 0; t < NIT; ++t) {
              float f[8];
              Elem<__nv_bfloat16>::unpack(v[kk][t], f);
#pragma unroll
              for (int e = 0; e < 8; ++e) acc = fmaf(qreg[t][e], f[e], acc);
            }
            part[2 * half + kk] = acc;
          }
        }
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
        const int rr = lane >> 3;                        // lanes [8k, 8k + 8) hold row k
        if ((lane & 7) == 0 && rr >= k0 && rr < k1) a.scores[first + rr] = tot;
        acc_rows += k1 - k0;
        k0 = k1;
      }
      // the stage's rows have been read: refill the slot with my stage m + nslot
      __syncwarp();
      if (m + nslot < n_my) issue(m + nslot);
      else cp_async_commit();
      // my next stage belongs to another request (or there is none): the finished request's rows count now, not a stage later
      {
        int nf = 0x7fffffff, nc;
        if (m + 1 < n_my) stage_rows(cw + F_WARPS * (m + 1), nf, nc);
        if (nf >= cur_end && acc_rows > 0) {
          if (lane == 0) red_release_gpu(rows_done + cur_r, acc_rows);
          acc_rows = 0;
        }
      }
    }
    if (cur_r >= 0 && acc_rows > 0) {
      __syncwarp();
      if (lane == 0) red_release_gpu(rows_done + cur_r, acc_rows);
    }
    for (; kcur < nseq; ++kcur) {
      mbar_wait(qfull(kcur % NQ), (kcur / NQ) & 1);
      if (lane == 0) mbar_arrive(qempty(kcur % NQ));
    }
    if (cw == 0 && lane == 0) VX_TRACE_STAMP(cta, 4);
  } else {
    // ---- warps 8..11, the selection warpgroup: (1) the query vectors of my requests, (2) their selections -----------
    if (st == 0) VX_TRACE_STAMP(cta, 5);
    SelectScratch& scratch = *reinterpret_cast<SelectScratch*>(sm + tail_off + (NQ - 1) * QV_BYTES);
    uint32_t* keys = reinterpret_cast<uint32_t*>(sm + tail_off + TAIL_FIXED);
    for (int r = cta; r < B; r += G) {
      const int row0 = s_indptr[r], rows = s_indptr[r + 1] - row0;
      const int n_tok = a.seq_lens[r];
      const int P = min(rows, (n_tok + PAGE - 1) / PAGE);
      const int k_budget = max(0, min(a.budget[r], a.max_budget));
      if (st == 0)
        while (ld_acquire_gpu(rows_done + r) < rows) __nanosleep(128);
      sel_sync();                                        // every score of the request has been written (and is visible)
      if (st == 0) VX_TRACE_STAMP(cta, 6);
      for (int j = st; j < P; j += SEL_NT) keys[j] = __float_as_uint(ldcg_f32(a.scores + row0 + j));
      sel_sync();
      const int cnt = cta_select_pages<SEL_NT, SEL_BAR, SEL_T0>(scratch, keys, P, k_budget, a.n_sink, a.n_local);
      int32_t* gp = a.sel_phys + (int64_t)r * a.max_budget;
      int32_t* gl = a.sel_logical + (int64_t)r * a.max_budget;
      for (int x = st; x < a.max_budget; x += SEL_NT) {
        const int j = x < cnt ? scratch.hist[x] : -1;
        gl[x] = j;
        gp[x] = j >= 0 ? a.page_indices[row0 + j] : -1;
      }
      if (st == 0) a.sel_count[r] = cnt;
      sel_sync();
      if (st == 0) { __threadfence(); st_release_gpu(sel_ready + r, 1); VX_TRACE_STAMP(cta, 7); }
    }
  }
  // every warp of the CTA is done with the stream: the ring, the P buffers and the tail now belong to the decode pipeline
  __syncthreads();
  if (tid == 0) VX_TRACE_STAMP(cta, 8);

  // ======================================= (a4) + (a5): decode items from the counter ==================================
  const int S = a.splits, n_items = B * S;
  const uint32_t p_base = base + OFF_P;
  constexpr int Q_PITCH = F_Q_PITCH;
  int pg0 = 0;                                           // pages this CTA's pipeline has run so far (barrier phases keep running)
  [[maybe_unused]] int n_done = 0;
  for (;;) {
    if (tid == 0) s_item = atomicAdd(sy + SY_NEXT, 1);
    __syncthreads();
    const int item = s_item;
    if (item >= n_items) break;
    const int i = item / S, split = item % S;
    if (tid == 0) {
      while (ld_acquire_gpu(sel_ready + i) == 0) __nanosleep(64);
      if (n_done == 0) VX_TRACE_STAMP(cta, 9);
    }
    __syncthreads();                                     // request i's block table is in global memory (and visible)
    const int n_tok = a.seq_lens[i];
    const int newest_page = (n_tok - 1) / PAGE;
    const int cnt = ldcg_s32(a.sel_count + i);
    const int per_split = (cnt + S - 1) / S;
    const int r_begin = min(split * per_split, cnt), r_end = min(r_begin + per_split, cnt);
    const int n_pages = r_end - r_begin;
    if (tid < n_pages) {
      s_mylist[0][tid] = ldcg_s32(a.sel_phys + (int64_t)i * a.max_budget + r_begin + tid);
      s_mylist[1][tid] = ldcg_s32(a.sel_logical + (int64_t)i * a.max_budget + r_begin + tid);
    }
    // Q rows -> the ring page this item will use LAST of the first three (its first two pages may already be on their way)
    const int q_page = (pg0 + 2) % N_ROPE;
    uint8_t* q_stage = sm + OFF_PAIR + q_page * PAIRS_PER_PAGE * PAIR_BYTES;
    if (n_pages > 0 && warp >= 2 && warp <= 5) {
      constexpr int Q_IT = NH * CHUNKS / SOFTMAX_THREADS;          // 18 independent 16-byte loads per thread
      uint4 qv[Q_IT];
#pragma unroll
      for (int k = 0; k < Q_IT; ++k) {
        const int x = tid - 64 + k * SOFTMAX_THREADS, h = x / CHUNKS, c = x % CHUNKS;
        qv[k] = h < a.num_q_heads ? *reinterpret_cast<const uint4*>(a.q + ((int64_t)i * a.num_q_heads + h) * D + c * 8)
                                  : make_uint4(0, 0, 0, 0);
      }
#pragma unroll
      for (int k = 0; k < Q_IT; ++k) {
        const int x = tid - 64 + k * SOFTMAX_THREADS, h = x / CHUNKS, c = x % CHUNKS;
        *reinterpret_cast<uint4*>(q_stage + h * Q_PITCH + c * 16) = qv[k];
      }
    }
    __syncthreads();                                     // the list and the staged Q rows are in shared memory
    auto list_phys = [&](int p) -> int { return s_mylist[0][p]; };
    auto list_log = [&](int p) -> int { return s_mylist[1][p]; };

    if (n_pages == 0) {                                  // an empty share: a zero partial of weight zero
      for (int e = tid; e < NH * DV; e += NT) {
        const int h = e / DV, d = e % DV;
        if (S > 1) a.part_o[(((int64_t)i * S + split) * DV + d) * NH + h] = 0.f;
        else if (h < a.num_q_heads) a.out[((int64_t)i * a.num_q_heads + h) * DV + d] = __float2bfloat16_rn(0.f);
      }
      if (tid < a.num_q_heads) {
        const int64_t row = (int64_t)i * a.num_q_heads + tid;
        if (S == 1) { if (a.lse_out) a.lse_out[row] = -INFINITY; }
        else a.part_lse[row * S + split] = -INFINITY;
      }
    } else if (warp == 0) {
      // ===== TMA producer: page p -> ring page (pg0 + p) % 3; the third page waits until Q has left its staging area =====
      int my_phys = 0;
      for (int p = 0; p < n_pages; ++p) {
        if ((p & 31) == 0) my_phys = p + lane < n_pages ? list_phys(p + lane) : 0;
        const int phys = __shfl_sync(0xffffffffu, my_phys, p & 31);
        if (p == 2) asm volatile("bar.sync 6, 64;" ::: "memory");          // (with the softmax warp, once Q is in tensor memory)
        if (elect_one()) {
          const int pg = pg0 + p, rs = pg % N_ROPE, u = pg / N_ROPE;
          const uint32_t full = bar(B_PAGE_FULL + rs);
          if (u >= 1) mbar_wait(bar(B_ROPE_EMPTY + rs), (u - 1) & 1);
          mbar_expect_tx(full, PAGE_BYTES);
          tma_box(base + OFF_ROPE + rs * K_ATOM_BYTES, &kmap, DV, phys, full);
#pragma unroll
          for (int j = 0; j < PAIRS_PER_PAGE; ++j) {
            const int ps = rs * PAIRS_PER_PAGE + j;
            if (u >= 1) mbar_wait(bar(B_PAIR_EMPTY + ps), (u - 1) & 1);
            const uint32_t dst = base + OFF_PAIR + ps * PAIR_BYTES;
            tma_box(dst, &kmap, 128 * j, phys, full);
            tma_box(dst + K_ATOM_BYTES, &kmap, 128 * j + 64, phys, full);
          }
        }
        __syncwarp();
      }
      if (n_pages <= 2) asm volatile("bar.sync 6, 64;" ::: "memory");
    } else if (warp == 1) {
      // ===== QK issuer =====
      asm volatile("bar.sync 7, 64;" ::: "memory");      // (with the softmax warp) Q is in tensor memory
      tc_fence_after();
      for (int p = 0; p < n_pages; ++p) {
        const int pg = pg0 + p, rs = pg % N_ROPE;
        if (pg >= 1) mbar_wait(bar(B_S_EMPTY), (pg - 1) & 1);
        mbar_wait(bar(B_PAGE_FULL + rs), (pg / N_ROPE) & 1);
        tc_fence_after();
        if (elect_one()) {
          if (p == 0 && n_done == 0) VX_TRACE_STAMP(cta, 12);
#pragma unroll
          for (int j = 0; j < PAIRS_PER_PAGE; ++j)
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
              const uint32_t kb = base + OFF_PAIR + (rs * PAIRS_PER_PAGE + j) * PAIR_BYTES + (ks >> 2) * K_ATOM_BYTES + (ks & 3) * 32;
              umma_ts(tmem + TM_S, tmem + TM_Q + 64 * j + 8 * ks, smem_desc(kb, 16, 1024), IDESC_QK, j > 0 || ks > 0);
            }
#pragma unroll
          for (int ks = 0; ks < 4; ++ks)
            umma_ts(tmem + TM_S, tmem + TM_Q + 256 + 8 * ks, smem_desc(base + OFF_ROPE + rs * K_ATOM_BYTES + ks * 32, 16, 1024),
                    IDESC_QK, true);
          umma_commit(bar(B_ROPE_EMPTY + rs));
          umma_commit(bar(B_S_FULL));
        }
        __syncwarp();
      }
    } else if (warp == PV_WARP) {
      // ===== PV issuer =====
      for (int p = 0; p < n_pages; ++p) {
        const int pg = pg0 + p, b = pg & 1, rs = pg % N_ROPE;
        mbar_wait(bar(B_P_FULL + b), (pg >> 1) & 1);
        tc_fence_after();
        if (elect_one()) {
#pragma unroll
          for (int ks = 0; ks < PAGE / 16; ++ks)
#pragma unroll
            for (int mb = 0; mb < PAIRS_PER_PAGE; ++mb)
              umma(tmem + TM_O + 32 * mb,
                   smem_desc(base + OFF_PAIR + (rs * PAIRS_PER_PAGE + mb) * PAIR_BYTES + ks * 2048, K_ATOM_BYTES, 1024),
                   smem_desc(p_base + b * P_BYTES + ks * 32, 16, 1024), IDESC_PV, p > 0 || ks > 0);
#pragma unroll
          for (int mb = 0; mb < PAIRS_PER_PAGE; ++mb) umma_commit(bar(B_PAIR_EMPTY + rs * PAIRS_PER_PAGE + mb));
          umma_commit(bar(B_PV_DONE + b));
          if (p == n_pages - 1 && n_done == 0) VX_TRACE_STAMP(cta, 13);
        }
        __syncwarp();
      }
    } else if (warp >= 2 && warp <= 5) {
      // ===== warps 2..5: Q -> tensor memory (warp 4), softmax (warp 4) + rescale helpers, then the epilogue ============
      const int sp = warp & 3;
      const uint32_t t_lane = tmem + ((uint32_t)(sp * 32) << 16);
      const int pl = n_pages - 1, pgl = pg0 + pl;
      if (warp == SOFTMAX_WARP) {
        {
          const uint4* qrow = reinterpret_cast<const uint4*>(q_stage + lane * Q_PITCH);
#pragma unroll 1
          for (int c = 0; c < D / 64; ++c) {
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
          asm volatile("bar.sync 7, 64;" ::: "memory");  // the QK issuer may start
          asm volatile("bar.sync 6, 64;" ::: "memory");  // the producer may overwrite the staging area
        }
        float m_ref = 0.f, l_sum = 0.f;
        int lg = list_log(0);
        for (int p = 0; p < n_pages; ++p) {
          const int pg = pg0 + p, b = pg & 1;
          const int valid = min(PAGE, n_tok - lg * PAGE);
          if (p + 1 < n_pages) lg = list_log(p + 1);
          mbar_wait(bar(B_S_FULL), pg & 1);
          tc_fence_after();
          float s[PAGE];
          tmem_ld32(t_lane + TM_S, *reinterpret_cast<float(*)[32]>(&s[0]));
          tmem_ld32(t_lane + TM_S + 32, *reinterpret_cast<float(*)[32]>(&s[32]));
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar(B_S_EMPTY));
          float tmax = -INFINITY;
#pragma unroll
          for (int t = 0; t < PAGE; ++t) {
            s[t] = t < valid ? s[t] * a.scale_log2 : -INFINITY;
            tmax = fmaxf(tmax, s[t]);
          }
          const bool grow = p > 0 && tmax > m_ref + kRescaleThreshold;
          const float fac = grow ? exp2f(m_ref - tmax) : 1.f;
          if (p == 0 || grow) m_ref = tmax;
          l_sum *= fac;
          const bool grow_any = __any_sync(0xffffffffu, grow);
          if (pg >= 2) mbar_wait(bar(B_ACK + b), ((pg >> 1) - 1) & 1);
          s_fac[b][lane] = fac;
          if (lane == 0) s_flag[b] = grow_any;
          __syncwarp();
          if (lane == 0) mbar_arrive(bar(B_DECIDE + b));
          if (pg >= 2) mbar_wait(bar(B_PV_DONE + b), ((pg >> 1) - 1) & 1);
          if (grow_any) {
            mbar_wait(bar(B_PV_DONE + ((pg - 1) & 1)), ((pg - 1) >> 1) & 1);
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
            mbar_wait(bar(B_ACK + b), (pg >> 1) & 1);
          }
          if (valid < PAGE) {                            // partial page: zero the stale value rows (0 x garbage must be 0)
            const int n_rows = PAGE - valid;
            for (int xx = lane; xx < n_rows * 64; xx += kWarp) {
              const int r = valid + xx / 64, at = (xx % 64) >> 3, c = xx & 7;
              const int ps = (pg * PAIRS_PER_PAGE + (at >> 1)) % N_PAIR;
              *reinterpret_cast<uint4*>(sm + OFF_PAIR + ps * PAIR_BYTES + (at & 1) * K_ATOM_BYTES + (r >> 3) * 1024 +
                                        (r & 7) * 128 + c * 16) = make_uint4(0, 0, 0, 0);
            }
          }
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
          fence_async_proxy();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar(B_P_FULL + b));
        }
        s_l[lane] = l_sum;
        s_m[lane] = m_ref;
        s_inv[lane] = 1.f / l_sum;
      } else {
        for (int p = 0; p < n_pages; ++p) {
          const int pg = pg0 + p, b = pg & 1;
          mbar_wait(bar(B_DECIDE + b), (pg >> 1) & 1);
          if (s_flag[b]) {
            mbar_wait(bar(B_PV_DONE + ((pg - 1) & 1)), ((pg - 1) >> 1) & 1);
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
        // (a1) the request's newest page is this item's last page: rebuild its summary row from the staged tile
        const int hidx = (warp == 5 ? 2 : warp - 2) * kWarp + lane;      // 0..95
        const int lg_last = list_log(pl);
        if (a.summary_upd != nullptr && lg_last == newest_page && hidx < CHUNKS) {
          mbar_wait(bar(B_S_FULL), pgl & 1);                             // QK(last) done: every box of the page has landed
          const int valid = min(PAGE, n_tok - lg_last * PAGE);
          const int cc = hidx, at = cc >> 3;
          const uint8_t* atom = at < 8 ? sm + OFF_PAIR + ((pgl * PAIRS_PER_PAGE + (at >> 1)) % N_PAIR) * PAIR_BYTES + (at & 1) * K_ATOM_BYTES
                                       : sm + OFF_ROPE + (pgl % N_ROPE) * K_ATOM_BYTES;
          if (a.summary_kind == VX_SUMMARY_CENTROID) {
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
            *reinterpret_cast<uint4*>(a.summary_upd + (int64_t)list_phys(pl) * D + cc * 8) = *reinterpret_cast<const uint4*>(o8);
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
            __nv_bfloat16* dst = a.summary_upd + (int64_t)list_phys(pl) * 2 * D + cc * 8;
            *reinterpret_cast<uint4*>(dst) = lo4;
            *reinterpret_cast<uint4*>(dst + D) = hi4;
          }
        }
      }
      // ---- epilogue (warps 2..5): O^T / l -> partial or final output ----------------------------------------
      softmax_barrier();
      mbar_wait(bar(B_PV_DONE + (pgl & 1)), (pgl >> 1) & 1);
      tc_fence_after();
#pragma unroll 1
      for (int mb = 0; mb < PAIRS_PER_PAGE; ++mb) {
        float o[NH];
        tmem_ld32(t_lane + TM_O + 32 * mb, o);
        const int d = mb * 128 + sp * 32 + lane;
        if (S > 1) {                                     // partial [request][split][channel][head]: 128 contiguous bytes per thread
          float4* dst = reinterpret_cast<float4*>(a.part_o + (((int64_t)i * S + split) * DV + d) * NH);
#pragma unroll
          for (int j4 = 0; j4 < NH / 4; ++j4)
            dst[j4] = make_float4(o[4 * j4] * s_inv[4 * j4], o[4 * j4 + 1] * s_inv[4 * j4 + 1],
                                  o[4 * j4 + 2] * s_inv[4 * j4 + 2], o[4 * j4 + 3] * s_inv[4 * j4 + 3]);
        } else {
#pragma unroll
          for (int j = 0; j < NH; ++j)
            if (j < a.num_q_heads) a.out[((int64_t)i * a.num_q_heads + j) * DV + d] = __float2bfloat16_rn(o[j] * s_inv[j]);
        }
      }
      tc_fence_before();
      if (warp == SOFTMAX_WARP && lane < a.num_q_heads) {
        const float lse = (s_m[lane] + log2f(s_l[lane])) * kLn2;
        const int64_t orow = (int64_t)i * a.num_q_heads + lane;
        if (S == 1) { if (a.lse_out) a.lse_out[orow] = lse; }
        else a.part_lse[orow * S + split] = lse;
      }
    }
    if (tid == 64 && n_done == 0) VX_TRACE_STAMP(cta, 14);
    // (warps 7..11 have no part in the pipeline: they wait here)
    // ---- (a5) the last share of the request to arrive merges the partials ------------------------------------------
    if (S > 1) {
      if (last_split_arrives(a.unit_counter + i, S, &s_last))
        merge_splits(a.part_o, a.part_lse, i, a.num_q_heads, S, a.out, a.lse_out, sm + OFF_PAIR);
    }
    pg0 += n_pages;
    ++n_done;
    tc_fence_before();
    __syncthreads();                                     // the merge scratch (ring) and TMEM are free for the next item
    tc_fence_after();
    if (tid == 0 && n_done == 1) VX_TRACE_STAMP(cta, 10);
  }
  if (tid == 0) VX_TRACE_STAMP(cta, 11);

  // ---- the last CTA to leave zeroes the step's counters (every other CTA has made its last access) -------------------
  if (tid == 0) {
    __threadfence();
    s_last = atomicAdd(sy + SY_DONE_CTAS, 1) == G - 1;
  }
  __syncthreads();
  if (s_last) {
    __threadfence();
    for (int x = tid; x < SY_PER_REQ + 3 * B; x += NT) sy[x] = 0;
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
}

VX_TRACE_SETTER(vx_trace_set_step_mla_flat)

size_t step_mla_flat_workspace_ints(int max_batch) { return (size_t)flat::SY_PER_REQ + 3 * (size_t)max_batch; }
size_t step_mla_flat_qvec_floats(int max_batch) { return (size_t)max_batch * flat::QV_FLOATS; }

// splits per request: about 1.75 items per CTA, so that the counter balances the tail, and no share above the list a CTA keeps
static int step_mla_flat_splits(const vx_ctx* c, int batch, int max_budget) {
  int s = (7 * c->num_sms / 4 + batch - 1) / batch;
  const int need = (max_budget + mla::F_MAX_LIST - 1) / mla::F_MAX_LIST;
  if (s < need) s = need;
  if (s > max_budget) s = max_budget;
  if (s > kMaxSplits) s = kMaxSplits;
  if (s > c->g.num_q_heads) s = c->g.num_q_heads;        // the partial buffer holds Hq splits per request
  return s < 1 ? 1 : s;
}

bool step_mla_flat_applies(const vx_ctx* c, const vx_page_table& pt, const vx_kv_pool& pool, int32_t max_budget) {
  const vx_geom& g = c->g;
  if (!(mla_tc_supported(g) && g.agg == VX_AGG_SUM && g.n_local >= 1 && pool.num_pool_pages > 0)) return false;
  if (pt.batch > flat::MAX_BATCH || pt.total_pages < 1) return false;
  const int p_cap = (pt.max_pages_per_req + 31) / 32 * 32;
  const int tail = flat::TAIL_FIXED + 4 * p_cap;
  if ((mla::SMEM_BYTES - tail - mla::OFF_PAIR) / (mla::F_WARPS * mla::F_STAGE_BYTES) < 2) return false;   // two stages per stream warp
  const int s = step_mla_flat_splits(c, pt.batch, max_budget);
  return (max_budget + s - 1) / s <= mla::F_MAX_LIST && max_budget <= kBins;
}

cudaError_t launch_step_mla_flat(vx_ctx* c, const void* q, const vx_kv_pool& pool, const void* summary,
                                 const vx_page_table& pt, const int32_t* budget, int32_t max_budget, bool update_summary,
                                 int32_t* sel_phys, int32_t* sel_logical, int32_t* sel_count, void* out, float* lse,
                                 cudaStream_t s) {
  const vx_geom& g = c->g;
  if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(step_mla_flat_kernel), c->device, mla::SMEM_BYTES)) return e;
  CUtensorMap kmap;
  if (cudaError_t e = make_latent_map(&kmap, pool)) return e;
  MlaFlatArgs a;
  a.q = static_cast<const __nv_bfloat16*>(q);
  a.summary = static_cast<const __nv_bfloat16*>(summary);
  a.page_indptr = pt.page_indptr;
  a.page_indices = pt.page_indices;
  a.seq_lens = pt.seq_lens;
  a.budget = budget;
  a.sel_phys = sel_phys;
  a.sel_logical = sel_logical;
  a.sel_count = sel_count;
  a.scores = c->ws.scores;
  a.qvec = c->ws.flat_qvec;
  a.sync = c->ws.flat_sync;
  a.part_o = c->ws.part_o;
  a.part_lse = c->ws.part_lse;
  a.unit_counter = c->ws.unit_counter;
  a.summary_upd = update_summary ? static_cast<__nv_bfloat16*>(const_cast<void*>(summary)) : nullptr;
  a.out = static_cast<__nv_bfloat16*>(out);
  a.lse_out = lse;
  a.batch = pt.batch;
  a.total_pages = pt.total_pages;
  a.num_q_heads = g.num_q_heads;
  a.max_budget = max_budget;
  a.n_sink = g.n_sink;
  a.n_local = g.n_local;
  a.row_chunks = (g.summary_kind == VX_SUMMARY_CENTROID ? 1 : 2) * mla::CHUNKS;
  a.p_cap = (pt.max_pages_per_req + 31) / 32 * 32;
  a.splits = c->flat_splits > 0 ? c->flat_splits : step_mla_flat_splits(c, pt.batch, max_budget);
  a.n_waves = c->flat_waves > 0 ? (c->flat_waves > flat::MAX_WAVES ? flat::MAX_WAVES : c->flat_waves) : 4;
  a.summary_kind = g.summary_kind;
  a.scale_log2 = g.sm_scale * mla::kLog2e;
  const int grid = c->num_sms;
  cudaError_t e = launch_kernel(step_mla_flat_kernel, dim3(grid), dim3(flat::NT), (size_t)mla::SMEM_BYTES, s, false, kmap, a);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace vx
