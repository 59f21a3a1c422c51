// vx_score.cu -- (a2) query-to-page scores from the page summaries.
// Envelope summaries (Quest): PAPER.md:552  u[h,j] = sum_c max(q_h[c]*M_j[c], q_h[c]*m_j[c]);  :92 / :119 aggregated
// over the query heads of one KV head by SUM (reading G2) or, for GQA groups, by MAX (:556).
// Centroid summaries (block top-k): Eq.2  s[j] = sum_h q_h . centroid_j.
//
// With SUM the per-head maxima collapse exactly (max(q*M, q*m) = max(q,0)*M + min(q,0)*m, M >= m):
//     S[kvh,j] = [Qm | Qp] . [m_j | M_j],   Qp = sum_h max(q_h,0),  Qm = sum_h min(q_h,0)
// i.e. one fp32 dot product per summary row (centroid: Qsum . centroid_j): 1 flop per byte, a pure HBM stream of
// 2*d*esz (centroid: d*esz) bytes per (page, KV head), gathered through the page table.
//
// Persistent kernel, two CTAs per SM.  All KV heads of a page are ONE contiguous chunk of the summary pool (4 KB
// at Hkv=8, d=128 bf16): a producer warp gathers PG pages per stage with cp.async.bulk (TMA bulk copy, completion
// on an mbarrier) into a 3..8-stage shared-memory ring sized to the shared-memory budget (no registers or LSU
// slots spent on the gather; the physical ids are prefetched 32 at a time); 8 consumer warps read rows from
// shared memory conflict-free (a warp reads one whole row per instruction -- two or four rows when a row is
// narrower than 512 bytes), multiply with their register-resident slice of the query vector and reduce with a
// shuffle butterfly.  Every CTA walks a contiguous range of the flat (ragged) page list, cut into
// groups that never straddle a request, so producer and consumers derive the same schedule independently; the
// request of the first page is found with independent strided loads (not a dependent binary search) and the
// query vector of a request is rebuilt with all its loads in flight at once.
#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

constexpr int kScConsumerWarps = 8;
constexpr int kScThreads = (kScConsumerWarps + 1) * kWarp;

__device__ __forceinline__ void sc_mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void sc_mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void sc_mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void sc_mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// (the summaries stream through once: evict-first, so that they do not push the scores, the page table and the queries
//  out of the L2 -- the next kernels read those)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}

// a page-table load that asks the L2 to keep its line (evict-last): the selection kernel gathers the same ids a few
// microseconds after 100+ MB of summaries have streamed through the cache
__device__ __forceinline__ int ld_keep_l2(const int32_t* p) {
  int v;
  asm volatile("{\n\t.reg .b64 pol;\n\tcreatepolicy.fractional.L2::evict_last.b64 pol, 1.0;\n\t"
               "ld.global.L2::cache_hint.s32 %0, [%1], pol;\n\t}" : "=r"(v) : "l"(p));
  return v;
}

// the schedule both roles follow: groups of <= PG pages inside one request, over flat pages [begin, end)
struct GroupIter {
  int flat, end, req, req_end;
  const int32_t* indptr;
  // Called by a converged warp.  The request holding flat page `begin` = number of indptr[1..batch] entries <= begin
  // (indptr is sorted): counted with independent strided loads -- one memory latency instead of the log2(batch)
  // dependent ones of a binary search (cold, that was several microseconds at the head of every CTA).
  __device__ GroupIter(int begin, int end_, int batch, const int32_t* page_indptr) : flat(begin), end(end_), indptr(page_indptr) {
    const int lane = threadIdx.x % kWarp;
    int below = 0;
    for (int r = lane; r < batch; r += kWarp) below += page_indptr[r + 1] <= begin;
#pragma unroll
    for (int o = kWarp / 2; o > 0; o >>= 1) below += __shfl_xor_sync(0xffffffffu, below, o);
    req = min(below, batch - 1);
    req_end = page_indptr[req + 1];
  }
  __device__ bool next(int pg, int& first, int& count, int& request) {
    if (flat >= end) return false;
    while (flat >= req_end) { ++req; req_end = indptr[req + 1]; }   // also skips empty requests
    first = flat;
    count = min(pg, min(req_end, end) - flat);
    request = req;
    flat += count;
    return true;
  }
};

template <typename T, int D, int PG, int HKV, int kScStages, int AGG, int KIND>
__global__ void __launch_bounds__(kScThreads, 2)
score_kernel(const T* __restrict__ q, const T* __restrict__ summary, int num_q_heads, int batch,
             const int32_t* __restrict__ page_indptr, const int32_t* __restrict__ page_indices, int total_pages,
             float* __restrict__ scores, int req_begin, int req_end, int flat_lo_host, int flat_span_host, int stream_once) {
  constexpr int PER = Elem<T>::kPerVec;
  // envelope: [min | max] of one (page, KV head); centroid (block top-k): the mean key, d elements
  constexpr int ROW_ELEMS = KIND == VX_SUMMARY_CENTROID ? D : 2 * D;
  constexpr int NCH = ROW_ELEMS / PER;           // 16-byte chunks per row
  constexpr int NIT = (NCH + kWarp - 1) / kWarp; // chunks per lane
  constexpr int RPW = PG * HKV / kScConsumerWarps;   // rows per warp per group
  constexpr int ROW_BYTES = ROW_ELEMS * (int)sizeof(T);
  constexpr int PAGE_BYTES = HKV * ROW_BYTES;
  constexpr int STAGE_BYTES = PG * PAGE_BYTES;
  static_assert(ROW_ELEMS % PER == 0 && kScConsumerWarps % HKV == 0, "shape");
  static_assert(RPW == 1 || RPW == 2 || RPW == 4 || RPW == 8, "rows per warp must be a power of two <= 8");
  // rows narrower than a warp-wide 512-byte read (256 B centroid rows, d = 64 envelopes): NCH lanes per row, 32 / NCH
  // rows per instruction, so that no lane idles
  constexpr int RPI = NCH < kWarp ? kWarp / NCH : 1;
  constexpr bool NARROW = AGG == VX_AGG_SUM && (NCH == 8 || NCH == 16) && RPW % RPI == 0;

  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t s_full[kScStages], s_empty[kScStages];
  float* s_q = reinterpret_cast<float*>(smem + (size_t)kScStages * STAGE_BYTES);   // SUM: [HKV][2*D] fp32: Qm | Qp
  T* s_qh = reinterpret_cast<T*>(smem + (size_t)kScStages * STAGE_BYTES);          // MAX: [Hq][2*D] in T: min(q_h,0) | max(q_h,0)

  const int warp = threadIdx.x / kWarp, lane = threadIdx.x % kWarp;
  if (threadIdx.x == 0) { VX_TRACE_STAMP(blockIdx.x, 0); VX_TRACE_SMID(blockIdx.x); }
  // this launch's request window in the flat page list (known to the host when the window is the whole batch: one
  // cold memory latency less at the head of every CTA)
  const int flat_lo = flat_span_host >= 0 ? flat_lo_host : page_indptr[req_begin];
  const int flat_span = flat_span_host >= 0 ? flat_span_host : page_indptr[req_end] - flat_lo;
  // The window's queries -> L2, a slice per CTA, before the summary stream saturates HBM: a CTA whose range crosses
  // into the next request rebuilds its query vector in mid-stream, and with the queries cold that stall was two
  // loaded memory latencies (~2 us) on the CTAs that finish last (profiles/r1e_trace.md).  The attention kernel
  // of the step reads the same queries later.
  if (threadIdx.x < kScConsumerWarps * kWarp) {    // (the consumers: the producer warp's first copies must not wait)
    const int64_t q_bytes = (int64_t)(req_end - req_begin) * num_q_heads * D * (int)sizeof(T);
    const int64_t per_cta = ((q_bytes + gridDim.x - 1) / gridDim.x + 127) / 128 * 128;
    const int64_t off = per_cta * blockIdx.x + (int64_t)threadIdx.x * 128;
    const uint8_t* qb = reinterpret_cast<const uint8_t*>(q + (int64_t)req_begin * num_q_heads * D);
    for (int64_t o = off; o < min(per_cta * (blockIdx.x + 1), q_bytes); o += kScConsumerWarps * kWarp * 128)
      asm volatile("prefetch.global.L2 [%0];" ::"l"(qb + o));
  }
  const int begin = flat_lo + (int)((int64_t)flat_span * blockIdx.x / gridDim.x);
  const int end = flat_lo + (int)((int64_t)flat_span * (blockIdx.x + 1) / gridDim.x);
  if (threadIdx.x == 0) {
    for (int s = 0; s < kScStages; ++s) {
      sc_mbar_init(smem_u32(&s_full[s]), 1);
      sc_mbar_init(smem_u32(&s_empty[s]), kScConsumerWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  pdl_trigger();                                // single-wave persistent grid: the selection kernel may queue up behind us
  if (begin >= end) return;
  int first, count, req;

  if (warp == kScConsumerWarps) {
    // ---- producer: one bulk copy per page (all KV heads of the page are contiguous) ----------
    // The physical ids of the CTA's flat page range are prefetched 32 at a time (one coalesced load, two chunks
    // in registers), so that no index load sits between a freed stage and its refill.
    const uint64_t stream_pol = l2_stream_policy(stream_once != 0);
    int chunk0 = begin;                                   // flat index of id_cur's lane 0
    int id_cur = chunk0 + lane < end ? ld_keep_l2(page_indices + chunk0 + lane) : 0;
    int id_nxt = chunk0 + kWarp + lane < end ? ld_keep_l2(page_indices + chunk0 + kWarp + lane) : 0;
    GroupIter it(begin, end, batch, page_indptr);         // (its loads fly together with the id loads above)
    if (lane == 0) VX_TRACE_STAMP(blockIdx.x, 1);
    for (int g = 0; it.next(PG, first, count, req); ++g) {
      const int s = g % kScStages;
      if (g >= kScStages) sc_mbar_wait(smem_u32(&s_empty[s]), ((g / kScStages) - 1) & 1);
      const uint32_t bar = smem_u32(&s_full[s]);
      if (lane == 0) sc_mbar_expect_tx(bar, (uint32_t)(count * PAGE_BYTES));
      __syncwarp();
      static_assert(PG <= kWarp, "a group is at most one id chunk long");
      if (first >= chunk0 + kWarp) {                      // the group starts in the next chunk: rotate, prefetch one more
        chunk0 += kWarp;
        id_cur = id_nxt;
        id_nxt = chunk0 + kWarp + lane < end ? ld_keep_l2(page_indices + chunk0 + kWarp + lane) : 0;
      }
      const int off = first + lane - chunk0;              // lane l copies page first + l (valid for l < count)
      const int a = __shfl_sync(0xffffffffu, id_cur, off & 31), b = __shfl_sync(0xffffffffu, id_nxt, off & 31);
      const int64_t phys = off < kWarp ? a : b;
      if (lane < count)
        bulk_g2s(smem_u32(smem + (size_t)s * STAGE_BYTES + (size_t)lane * PAGE_BYTES),
                 reinterpret_cast<const uint8_t*>(summary) + phys * PAGE_BYTES, (uint32_t)PAGE_BYTES, bar, stream_pol);
      if (lane == 0 && g == 0) VX_TRACE_STAMP(blockIdx.x, 2);
      if (lane == 0 && g == kScStages - 1) VX_TRACE_STAMP(blockIdx.x, 3);
    }
    if (lane == 0) VX_TRACE_STAMP(blockIdx.x, 4);
    return;
  }

  // ---- consumers: warp w owns KV head w % HKV and rows w + 8k of every group ---------------------
  GroupIter it(begin, end, batch, page_indptr);
  const int grp = num_q_heads / HKV;
  const int kvh = warp % HKV;
  float qreg[NIT][PER];
  int cur_req = -1;
  for (int g = 0; it.next(PG, first, count, req); ++g) {
    const int s = g % kScStages;
    if (req != cur_req) {                        // new request: rebuild [Qm | Qp] for all KV heads (rare)
      if (threadIdx.x == 0) VX_TRACE_STAMP(blockIdx.x, cur_req < 0 ? 5 : 7);
      asm volatile("bar.sync 1, %0;" ::"n"(kScConsumerWarps * kWarp));
      if constexpr (AGG == VX_AGG_MAX) {
        // per-head vectors (PAPER.md:556 max_h variant): u[h] = [min(q_h,0) | max(q_h,0)] . [m | M], exact in T
        constexpr int NVH = D / PER;
        for (int e = threadIdx.x; e < num_q_heads * NVH; e += kScConsumerWarps * kWarp) {
          const int h = e / NVH, c = e % NVH;
          const uint4 raw = *reinterpret_cast<const uint4*>(q + ((int64_t)req * num_q_heads + h) * D + c * PER);
          float f[PER];
          Elem<T>::unpack(raw, f);
#pragma unroll
          for (int x = 0; x < PER; ++x) {
            s_qh[h * ROW_ELEMS + c * PER + x] = Elem<T>::from_float(fminf(f[x], 0.f));
            s_qh[h * ROW_ELEMS + D + c * PER + x] = Elem<T>::from_float(fmaxf(f[x], 0.f));
          }
        }
      } else if constexpr (HKV == 1) {
        // one latent head shared by a large group (MLA, g = 32): three thread groups take a third of the heads each, so
        // that every load of the rebuild is in flight at once (one memory latency, not g / 8); the partial sums are
        // added in a fixed order (deterministic)
        constexpr int NV1 = D / PER, GS = 3, HMAX = 11;              // up to 33 heads
        float* s_part = s_q + ROW_ELEMS;                              // [GS][ROW_ELEMS]
        const int e = threadIdx.x;
        if (e < GS * NV1) {
          const int gi = e / NV1, c = e % NV1;
          const int per = (grp + GS - 1) / GS, h0 = gi * per, h1 = min(h0 + per, grp);
          const T* qbase = q + ((int64_t)req * num_q_heads + h0) * D + c * PER;
          uint4 v[HMAX];
#pragma unroll
          for (int k = 0; k < HMAX; ++k)
            v[k] = h0 + k < h1 ? *reinterpret_cast<const uint4*>(qbase + (int64_t)k * D) : make_uint4(0, 0, 0, 0);
          float qp[PER], qm[PER];
#pragma unroll
          for (int x = 0; x < PER; ++x) { qp[x] = 0.f; qm[x] = 0.f; }
#pragma unroll
          for (int k = 0; k < HMAX; ++k) {
            float f[PER];
            Elem<T>::unpack(v[k], f);
#pragma unroll
            for (int x = 0; x < PER; ++x) {
              if constexpr (KIND == VX_SUMMARY_CENTROID) qp[x] += f[x];
              else { qp[x] += fmaxf(f[x], 0.f); qm[x] += fminf(f[x], 0.f); }
            }
          }
#pragma unroll
          for (int x = 0; x < PER; ++x) {
            if constexpr (KIND == VX_SUMMARY_CENTROID) s_part[gi * ROW_ELEMS + c * PER + x] = qp[x];
            else {
              s_part[gi * ROW_ELEMS + c * PER + x] = qm[x];
              s_part[gi * ROW_ELEMS + D + c * PER + x] = qp[x];
            }
          }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(kScConsumerWarps * kWarp));
        for (int x = threadIdx.x; x < ROW_ELEMS; x += kScConsumerWarps * kWarp)
          s_q[x] = (s_part[x] + s_part[ROW_ELEMS + x]) + s_part[2 * ROW_ELEMS + x];
      } else {
      // one thread per (KV head, 16-byte channel vector); the group's heads are read 8 at a time with all
      // loads of a batch in flight together (a head-by-head loop costs one memory latency per head)
      constexpr int NV = D / PER;
      for (int e = threadIdx.x; e < HKV * NV; e += kScConsumerWarps * kWarp) {
        const int h = e / NV, c = e % NV;
        const T* qbase = q + ((int64_t)req * num_q_heads + h * grp) * D + c * PER;
        float qp[PER], qm[PER];
#pragma unroll
        for (int k = 0; k < PER; ++k) { qp[k] = 0.f; qm[k] = 0.f; }
        for (int r0 = 0; r0 < grp; r0 += 8) {
          uint4 v[8];
#pragma unroll
          for (int k = 0; k < 8; ++k)
            v[k] = r0 + k < grp ? *reinterpret_cast<const uint4*>(qbase + (int64_t)(r0 + k) * D) : make_uint4(0, 0, 0, 0);
#pragma unroll
          for (int k = 0; k < 8; ++k) {                  // zeros add nothing: heads past the group need no branch
            float f[PER];
            Elem<T>::unpack(v[k], f);
#pragma unroll
            for (int x = 0; x < PER; ++x) {
              if constexpr (KIND == VX_SUMMARY_CENTROID) qp[x] += f[x];        // Eq.2: sum_h q_h . centroid = (sum_h q_h) . centroid
              else { qp[x] += fmaxf(f[x], 0.f); qm[x] += fminf(f[x], 0.f); }
            }
          }
        }
#pragma unroll
        for (int x = 0; x < PER; ++x) {
          if constexpr (KIND == VX_SUMMARY_CENTROID) s_q[h * ROW_ELEMS + c * PER + x] = qp[x];
          else {
            s_q[h * ROW_ELEMS + c * PER + x] = qm[x];
            s_q[h * ROW_ELEMS + D + c * PER + x] = qp[x];
          }
        }
      }
      }
      asm volatile("bar.sync 1, %0;" ::"n"(kScConsumerWarps * kWarp));
      if (threadIdx.x == 0) VX_TRACE_STAMP(blockIdx.x, cur_req < 0 ? 6 : 8);
      cur_req = req;
      if constexpr (AGG == VX_AGG_SUM) {
#pragma unroll
        for (int t = 0; t < NIT; ++t) {
          const int c = NARROW ? lane % NCH : lane + t * kWarp;
#pragma unroll
          for (int e = 0; e < PER; ++e) qreg[t][e] = (NCH % kWarp == 0 || c < NCH) ? s_q[kvh * ROW_ELEMS + c * PER + e] : 0.f;
        }
      }
    }
    sc_mbar_wait(smem_u32(&s_full[s]), (g / kScStages) & 1);
    if (threadIdx.x == 0 && g == 0) VX_TRACE_STAMP(blockIdx.x, 9);
    const int rows = count * HKV;                // row r = page (r / HKV), head (r % HKV)
    if constexpr (NARROW) {
      constexpr int KIT = RPW / RPI;             // instructions per group; instruction i covers rows warp + 8 (i RPI + lane / NCH)
      const uint8_t* st = smem + (size_t)s * STAGE_BYTES + (lane % NCH) * 16;
      uint4 vn[KIT];
#pragma unroll
      for (int i = 0; i < KIT; ++i) {
        const int r = warp + (i * RPI + lane / NCH) * kScConsumerWarps;
        vn[i] = r < rows ? *reinterpret_cast<const uint4*>(st + r * ROW_BYTES) : make_uint4(0, 0, 0, 0);
      }
      __syncwarp();
      if (lane == 0) sc_mbar_arrive(smem_u32(&s_empty[s]));  // stage consumed: its rows are in registers
#pragma unroll
      for (int i = 0; i < KIT; ++i) {
        float f[PER];
        Elem<T>::unpack(vn[i], f);
        float acc = 0.f;
#pragma unroll
        for (int e = 0; e < PER; ++e) acc = fmaf(qreg[0][e], f[e], acc);
#pragma unroll
        for (int o = NCH / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);   // sum over the row's NCH lanes
        const int r = warp + (i * RPI + lane / NCH) * kScConsumerWarps;
        if (lane % NCH == 0 && r < rows) scores[(int64_t)kvh * total_pages + first + r / HKV] = acc;
      }
      continue;
    }
    const uint8_t* stage = smem + (size_t)s * STAGE_BYTES + lane * 16;
    uint4 v[RPW][NIT];
#pragma unroll
    for (int k = 0; k < RPW; ++k) {
      const int r = warp + k * kScConsumerWarps;
#pragma unroll
      for (int t = 0; t < NIT; ++t) {
        const bool ok = r < rows && (NCH % kWarp == 0 || lane + t * kWarp < NCH);
        v[k][t] = ok ? *reinterpret_cast<const uint4*>(stage + r * ROW_BYTES + t * kWarp * 16) : make_uint4(0, 0, 0, 0);
      }
    }
    __syncwarp();
    if (lane == 0) sc_mbar_arrive(smem_u32(&s_empty[s]));    // stage consumed: its rows are in registers
    if constexpr (AGG == VX_AGG_MAX) {
      // g dot products per row, the head vectors read from shared memory (conflict-free: a warp reads one row)
#pragma unroll
      for (int k = 0; k < RPW; ++k) {
        const int r = warp + k * kScConsumerWarps;
        float best = -INFINITY;
        for (int h = 0; h < grp; ++h) {
          float acc = 0.f;
#pragma unroll
          for (int t = 0; t < NIT; ++t) {
            const int c = lane + t * kWarp;
            if (NCH % kWarp == 0 || c < NCH) {
              float f[PER], qf[PER];
              Elem<T>::unpack(v[k][t], f);
              Elem<T>::unpack(*reinterpret_cast<const uint4*>(s_qh + (kvh * grp + h) * ROW_ELEMS + c * PER), qf);
#pragma unroll
              for (int e = 0; e < PER; ++e) acc = fmaf(qf[e], f[e], acc);
            }
          }
          best = fmaxf(best, warp_sum(acc));
        }
        if (lane == 0 && r < rows) scores[(int64_t)kvh * total_pages + first + r / HKV] = best;
      }
      continue;
    }
    float part[RPW];
#pragma unroll
    for (int k = 0; k < RPW; ++k) {
      float acc = 0.f;
#pragma unroll
      for (int t = 0; t < NIT; ++t) {
        float f[PER];
        Elem<T>::unpack(v[k][t], f);
#pragma unroll
        for (int e = 0; e < PER; ++e) acc = fmaf(qreg[t][e], f[e], acc);
      }
      part[k] = acc;
    }
    // transposed butterfly: RPW partial sums over 32 lanes -> lanes [k*32/RPW, (k+1)*32/RPW) hold the total of row k
    float tot;
    if constexpr (RPW == 8) {
      float a4[4], a2[2];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const bool up = lane & 16;
        a4[j] = (up ? part[j + 4] : part[j]) + __shfl_xor_sync(0xffffffffu, up ? part[j] : part[j + 4], 16);
      }
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const bool up = lane & 8;
        a2[j] = (up ? a4[j + 2] : a4[j]) + __shfl_xor_sync(0xffffffffu, up ? a4[j] : a4[j + 2], 8);
      }
      const bool up = lane & 4;
      tot = (up ? a2[1] : a2[0]) + __shfl_xor_sync(0xffffffffu, up ? a2[0] : a2[1], 4);
      tot += __shfl_xor_sync(0xffffffffu, tot, 2);
      tot += __shfl_xor_sync(0xffffffffu, tot, 1);
    } else if constexpr (RPW == 4) {
      float a2[2];
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const bool up = lane & 16;
        a2[j] = (up ? part[j + 2] : part[j]) + __shfl_xor_sync(0xffffffffu, up ? part[j] : part[j + 2], 16);
      }
      const bool up = lane & 8;
      tot = (up ? a2[1] : a2[0]) + __shfl_xor_sync(0xffffffffu, up ? a2[0] : a2[1], 8);
      tot += __shfl_xor_sync(0xffffffffu, tot, 4);
      tot += __shfl_xor_sync(0xffffffffu, tot, 2);
      tot += __shfl_xor_sync(0xffffffffu, tot, 1);
    } else if constexpr (RPW == 2) {
      const bool up = lane & 16;
      tot = (up ? part[1] : part[0]) + __shfl_xor_sync(0xffffffffu, up ? part[0] : part[1], 16);
      tot += __shfl_xor_sync(0xffffffffu, tot, 8);
      tot += __shfl_xor_sync(0xffffffffu, tot, 4);
      tot += __shfl_xor_sync(0xffffffffu, tot, 2);
      tot += __shfl_xor_sync(0xffffffffu, tot, 1);
    } else {
      tot = warp_sum(part[0]);
    }
    constexpr int LPR = kWarp / RPW;             // lanes per row after the butterfly
    const int r = warp + (lane / LPR) * kScConsumerWarps;
    if ((lane % LPR) == 0 && r < rows) scores[(int64_t)kvh * total_pages + first + r / HKV] = tot;
  }
  if (threadIdx.x == 0) VX_TRACE_STAMP(blockIdx.x, 11);
}

VX_TRACE_SETTER(vx_trace_set_score)

bool score_geometry_supported(const vx_geom& g) {
  if (g.agg != VX_AGG_SUM && g.agg != VX_AGG_MAX) return false;
  const int hkv = g.num_kv_heads;
  // MAX costs g flop per byte: CUDA cores carry it for GQA groups (g <= 8); the MLA group (16 or 32 heads on one
  // latent head) is a contraction on the tensor cores (vx_score_mla_max.cu)
  if (score_mla_max_supported(g)) return true;
  if (g.agg == VX_AGG_MAX && (g.kv_shared || g.num_q_heads / hkv > 8)) return false;
  if (g.summary_kind != VX_SUMMARY_ENVELOPE && g.summary_kind != VX_SUMMARY_CENTROID) return false;
  if (g.summary_kind == VX_SUMMARY_CENTROID && g.agg != VX_AGG_SUM) return false;       // Eq.2 is a mean over the group
  if (hkv != 1 && hkv != 2 && hkv != 4 && hkv != 8) return false;   // a consumer warp owns one KV head
  if (g.dtype == VX_DT_BF16) return g.qk_dim == 128 || g.qk_dim == 64 || g.qk_dim == 576 || g.qk_dim == 256;
  return g.qk_dim == 64 || g.qk_dim == 128;
}

constexpr int pow2_floor(int x) { int p = 1; while (2 * p <= x) p *= 2; return p; }
constexpr int clamp_int(int x, int lo, int hi) { return x < lo ? lo : (x > hi ? hi : x); }

template <typename T, int D, int PG, int HKV, int AGG, int KIND>
static cudaError_t launch_score_agg(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt,
                                  float* scores, cudaStream_t s, const ReqRange& rr) {
  const vx_geom& g = c->g;
  constexpr int ROW = KIND == VX_SUMMARY_CENTROID ? D : 2 * D;
  constexpr size_t page_bytes = (size_t)HKV * ROW * sizeof(T);
  // as many ~16-32 KB stages as two CTAs per SM can hold (>= 3): the bytes in flight, not the math, set the rate
  constexpr size_t q_bytes = AGG == VX_AGG_MAX ? (size_t)HKV * 8 * ROW * sizeof(T)
                                               : (size_t)HKV * ROW * sizeof(float) * (HKV == 1 ? 4 : 1);   // HKV 1: + 3 partial rows
  // measured (C2 / C3 / C4 sweep of stage size x footprint): GQA pools do best with ~16 KB stages in a 72 KB CTA,
  // the single-head MLA pool with ~18 KB stages in 110 KB
  constexpr int kFoot = (HKV == 1 ? 110 : 72) * 1024;
  constexpr int kScStages = clamp_int((int)((kFoot - q_bytes) / (PG * page_bytes)), 3, 8);
  constexpr size_t smem = kScStages * PG * page_bytes + q_bytes;
  if (cudaError_t e = ensure_dyn_smem(reinterpret_cast<const void*>(score_kernel<T, D, PG, HKV, kScStages, AGG, KIND>), c->device, (int)smem)) return e;
  int ctas = c->num_sms * (2 * smem + 4096 <= 227 * 1024 ? 2 : 1);   // two CTAs per SM when they fit
  const int min_pages = 2 * PG;                  // do not spread tiny inputs over every SM
  const int64_t est_pages = rr.count < 0 ? pt.total_pages : (int64_t)pt.total_pages * rr.count / (pt.batch > 0 ? pt.batch : 1) + 1;
  if ((int64_t)ctas * min_pages > est_pages) ctas = (int)((est_pages + min_pages - 1) / min_pages);
  if (ctas < 1) ctas = 1;
  score_kernel<T, D, PG, HKV, kScStages, AGG, KIND><<<ctas, kScThreads, smem, s>>>(
      static_cast<const T*>(q), static_cast<const T*>(summary), g.num_q_heads, pt.batch, pt.page_indptr,
      pt.page_indices, pt.total_pages, scores, rr.begin, rr.begin + (rr.count < 0 ? pt.batch : rr.count), 0,
      rr.count < 0 ? pt.total_pages : -1, l2_stream_once(c, (int64_t)est_pages * (int64_t)page_bytes) ? 1 : 0);
  c->launches += 1;
  return cudaGetLastError();
}

template <typename T, int D, int PG, int HKV, int KIND>
static cudaError_t launch_score_t(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt,
                                  float* scores, cudaStream_t s, const ReqRange& rr) {
  if constexpr (KIND == VX_SUMMARY_ENVELOPE) {
    if (c->g.agg == VX_AGG_MAX) return launch_score_agg<T, D, PG, HKV, VX_AGG_MAX, KIND>(c, q, summary, pt, scores, s, rr);
  }
  return launch_score_agg<T, D, PG, HKV, VX_AGG_SUM, KIND>(c, q, summary, pt, scores, s, rr);
}

// PG pages per stage so that a stage is ~32 KB and every consumer warp gets 1, 2, 4 or 8 rows of it
template <typename T, int D, int KIND>
static cudaError_t launch_score_k(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt,
                                  float* scores, cudaStream_t s, const ReqRange& rr) {
  constexpr int row_bytes = (KIND == VX_SUMMARY_CENTROID ? D : 2 * D) * (int)sizeof(T);
  constexpr int rows32k = pow2_floor(32768 / row_bytes < 8 ? 8 : 32768 / row_bytes);     // rows per ~32 KB stage, >= 8
  constexpr int rows16k = pow2_floor(16384 / row_bytes < 8 ? 8 : 16384 / row_bytes);     // rows per ~16 KB stage, >= 8
  switch (c->g.num_kv_heads) {                   // rows per stage = PG * HKV in [8, 64] (1..8 rows per consumer warp)
    case 8: return launch_score_t<T, D, clamp_int(rows16k, 8, 64) / 8, 8, KIND>(c, q, summary, pt, scores, s, rr);
    case 4: return launch_score_t<T, D, clamp_int(rows16k, 8, 64) / 4, 4, KIND>(c, q, summary, pt, scores, s, rr);
    case 2: return launch_score_t<T, D, clamp_int(rows16k, 8, 64) / 2, 2, KIND>(c, q, summary, pt, scores, s, rr);
    case 1: return launch_score_t<T, D, clamp_int(rows32k, 8, 32), 1, KIND>(c, q, summary, pt, scores, s, rr);
  }
  return cudaErrorInvalidValue;
}

template <typename T, int D>
static cudaError_t launch_score_d(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt,
                                  float* scores, cudaStream_t s, const ReqRange& rr) {
  if (c->g.summary_kind == VX_SUMMARY_CENTROID) return launch_score_k<T, D, VX_SUMMARY_CENTROID>(c, q, summary, pt, scores, s, rr);
  return launch_score_k<T, D, VX_SUMMARY_ENVELOPE>(c, q, summary, pt, scores, s, rr);
}

cudaError_t launch_page_score(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt,
                              float* scores, cudaStream_t s, const ReqRange& rr) {
  if (pt.batch == 0 || pt.total_pages == 0) return cudaSuccess;
  const vx_geom& g = c->g;
  if (kv_is_fp8(g)) return launch_score_fp8(c, q, summary, pt, scores, s);
  if (score_mla_max_supported(g)) return launch_score_mla_max(c, q, summary, pt, scores, s, rr);
  if (g.dtype == VX_DT_BF16) {
    switch (g.qk_dim) {
      case 64: return launch_score_d<__nv_bfloat16, 64>(c, q, summary, pt, scores, s, rr);
      case 128: return launch_score_d<__nv_bfloat16, 128>(c, q, summary, pt, scores, s, rr);
      case 256: return launch_score_d<__nv_bfloat16, 256>(c, q, summary, pt, scores, s, rr);
      case 576: return launch_score_d<__nv_bfloat16, 576>(c, q, summary, pt, scores, s, rr);
    }
  } else {
    switch (g.qk_dim) {
      case 64: return launch_score_d<float, 64>(c, q, summary, pt, scores, s, rr);
      case 128: return launch_score_d<float, 128>(c, q, summary, pt, scores, s, rr);
    }
  }
  return cudaErrorInvalidValue;
}

}  // namespace vx
