// vx_internal.h -- context, workspace carving and kernel launcher prototypes (host side).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/vortex_b200.h"
#include "../../include/vortex_b200_trace.h"

namespace vx {

constexpr int kMaxSplits = 32;   // split-KV fan-out bound (workspace is sized for it)

struct Workspace {               // device pointers carved from the caller's workspace
  float* scores;                 // [Hkv, max_total_pages]
  int32_t* sel_phys;             // [max_batch, Hkv, max_budget]
  int32_t* sel_logical;          // [max_batch, Hkv, max_budget]
  int32_t* sel_count;            // [max_batch, Hkv]
  float* part_o;                 // [max_batch, Hq, kMaxSplits, v_dim]
  float* part_lse;               // [max_batch, Hq, kMaxSplits]
  int32_t* unit_counter;         // [max_batch, Hkv] split-arrival counters; zero between steps
  // staging for vx_sparse_decode_step_host
  void* h_q;                     // [max_batch, Hq, qk_dim] elements
  int32_t* h_indptr;             // [max_batch + 1]
  int32_t* h_indices;            // [max_total_pages]
  int32_t* h_seq_lens;           // [max_batch]
  int32_t* h_budget;             // [max_batch]
  void* h_out;                   // [max_batch, Hq, v_dim] elements
  float* h_lse;                  // [max_batch, Hq]
  // the flat MLA step kernel (vx_step_mla_flat.cu)
  float* flat_qvec;              // [max_batch, 2 qk_dim] query vectors [Qm | Qp]
  int32_t* flat_sync;            // counters and per-request flags; zero between steps
  int32_t* blk_indptr;           // blocks finer than the page: the page table expanded into a block table, [max_batch + 1]
  int32_t* blk_indices;          // [max_total_pages * bpp] physical block ids
  float* topk_remap;             // [kTopkRemapMaxKnots] the knot table of vx_set_topk_remap
  void* mla_stage;               // fp8 latent cache: [max_batch * max_budget] selected pages widened to bf16 (vx_decode_mla_fp8.cu)
  int32_t* mla_stage_sel;        // [max_batch, max_budget] their ids in that pool
  float* fp8_qvec;               // fp8 KV cache: [max_batch, Hkv, 2 qk_dim] query vectors [Qm | Qp] of the score kernel (vx_score_fp8.cu)
  size_t bytes;                  // total
};

// carve (base may be null: only sizes are computed)
Workspace carve_workspace(const vx_geom& g, void* base, int32_t max_batch, int32_t max_total_pages,
                          int32_t max_budget);

// Approximate radix top-k (PAPER.md:196 stochastic early termination, :538 `approxTopK`):
// tolerate_ratio <= 0 is the exact selection.
// remap (App. D.2, reading G29): an offline-profiled monotone knot table through which the first radix pass
// bins the normalised scores; remap_n == 0: none.  A plan with a remap runs the approximate kernels' code (which carry the
// remapped pass) even at tolerate_ratio 0, where their result is the exact selection.
constexpr int kTopkRemapMaxKnots = 65;
struct ApproxPlan {
  float tolerate_ratio = 0.f;
  uint64_t seed = 0;
  const float* remap = nullptr;                  // device, remap_n floats in [0, 1], non-decreasing
  int remap_n = 0;
  __host__ __device__ bool active() const { return tolerate_ratio > 0.f || remap_n > 0; }
};
constexpr int kTopkRegMaxPages = 8 * 1024;       // register-resident selection kernel: pages per request
constexpr int kTopkApproxMaxPages = 48 * 1024;   // the lossy selection beyond that: the shared-memory-key kernel's key cache
constexpr int kTopkApproxMaxBudgetLong = 2048;   // ... which stages at most this many selected pages
inline bool approx_topk_supported(int max_pages_per_req, int max_budget) {
  return max_pages_per_req <= kTopkRegMaxPages || (max_pages_per_req <= kTopkApproxMaxPages && max_budget <= kTopkApproxMaxBudgetLong);
}

}  // namespace vx

struct vx_ctx;
inline bool l2_stream_once(const vx_ctx* c, int64_t bytes);
struct vx_ctx {
  vx_geom g;
  int device;
  int num_sms;
  int64_t l2_bytes;              // the device's L2 size (streams larger than half of it are read evict-first)
  int32_t max_batch, max_total_pages, max_pages_per_req, max_budget;
  vx::Workspace ws;
  int32_t launches;              // kernels enqueued by the last compute call
  vx::ApproxPlan approx;         // vx_set_topk_approx: used by a fused step with VX_STEP_APPROX_TOPK
  int32_t mla_step;              // VX_OPT_MLA_STEP
  int32_t bpp;                   // selection blocks per physical page (vx_geom.block_size); g.page_size holds the BLOCK size
  int32_t user_page_size;        // tokens per physical page as the caller gave it
  int32_t* pinned_small;         // pinned host staging [3 max_batch + 1] for vx_sparse_decode_step_host's small arrays
  int32_t flat_splits, flat_waves;   // VX_OPT_MLA_FLAT_*: 0 = the library's choice
  char err[512];
};
inline bool l2_stream_once(const vx_ctx* c, int64_t bytes) { return bytes > c->l2_bytes / 2; }


namespace vx {

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) holds per DEVICE: the opt-in is remembered per (kernel, device),
// so contexts on several GPUs of one process each get it (a process-wide flag would skip the second device).
cudaError_t ensure_dyn_smem(const void* kernel, int device, int bytes);

// One kernel launch; pdl = allow it to start while its predecessor in the stream drains (the kernel
// itself calls pdl_wait() before touching what the predecessor wrote).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                                 bool pdl, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ... as thread-block clusters of cluster_x CTAs along x (grid.x must be a multiple of it)
template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel_cluster(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                                         bool pdl, int cluster_x, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[2];
  int n = 0;
  if (cluster_x > 1) {
    at[n].id = cudaLaunchAttributeClusterDimension;
    at[n].val.clusterDim.x = (unsigned)cluster_x;
    at[n].val.clusterDim.y = 1;
    at[n].val.clusterDim.z = 1;
    ++n;
  }
  if (pdl) {
    at[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[n].val.programmaticStreamSerializationAllowed = 1;
    ++n;
  }
  cfg.attrs = at;
  cfg.numAttrs = n;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// a window of requests [begin, begin + count) of the page table; count < 0 = the whole batch
struct ReqRange {
  int begin = 0;
  int count = -1;
};

// What the selection kernel prefetches into L2 for the decode kernel that follows it in a step: the first
// `pages_per_split` pages of every split of every (request, KV head), K and V chunks (`chunk_bytes` contiguous
// bytes each).  Between the end of the selection and the decode kernel's first loads HBM would sit idle; the
// prefetch moves a few MB of the decode kernel's stream into that gap.  k == nullptr: no prefetch.
struct PrefetchPlan {
  const void* k = nullptr;
  const void* v = nullptr;                       // nullptr: K only (MLA latent)
  int64_t page_bytes = 0, head_bytes = 0;        // byte strides of a page / a KV head in the pool
  uint32_t chunk_bytes = 0;                      // page_size * row bytes, contiguous
  int splits = 1, pages_per_split = 0;
};
// phase tracing (-DVX_TRACE builds; cudaErrorNotSupported otherwise): one setter per kernel file
cudaError_t vx_trace_set_score(long long* buf, int ctas);
cudaError_t vx_trace_set_topk(long long* buf, int ctas);
cudaError_t vx_trace_set_decode_gqa(long long* buf, int ctas);
cudaError_t vx_trace_set_decode_mla(long long* buf, int ctas);
cudaError_t vx_trace_set_step_mla(long long* buf, int ctas);
int decode_gqa_splits(const vx_ctx* c, int n_req, int max_budget);
int decode_mla_splits(const vx_ctx* c, int n_req, int max_budget);

// how a decode launch is embedded in a step
struct DecodeOpts {
  ReqRange rr;
  void* summary_upd = nullptr;   // non-null: also rebuild the summary of each request's newest page (a1), whose
                                 // keys the kernel stages anyway (it is a forced local page)
  bool pdl = false;              // launched as a programmatic dependent of the preceding kernel
  float scale_mul = 1.f;         // multiplies sm_scale (an fp8 pool's k_scale when the kernel runs on widened codes)
  float out_scale = 1.f;         // multiplies the output (its v_scale)
  const int32_t* budget = nullptr;   // fused step: sel_count[i, h] is known to be min(budget[i], max_budget, P_i), so the kernel
                                 // need not wait for the selection kernel to read it (one L2 round trip less after the wait)
};

// every launcher returns cudaGetLastError() after its launches and adds to ctx->launches
cudaError_t launch_summary_update(vx_ctx* c, const vx_kv_pool& pool, const vx_page_table& pt,
                                  const int32_t* first_new_pos, void* summary, cudaStream_t s);
cudaError_t launch_page_score(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt,
                              float* scores, cudaStream_t s, const ReqRange& rr = ReqRange());
cudaError_t launch_topk_pages(vx_ctx* c, const float* scores, const vx_page_table& pt,
                              const int32_t* budget, int32_t max_budget, int32_t* sel_phys,
                              int32_t* sel_logical, int32_t* sel_count, cudaStream_t s, bool pdl = false,
                              const ReqRange& rr = ReqRange(), const PrefetchPlan& pf = PrefetchPlan(),
                              const ApproxPlan& ap = ApproxPlan());
// the same selection with each problem on a cluster of two CTAs (vx_topk_pair.cu)
bool topk_pair_applies(const vx_ctx* c, int n_problems, int max_pages_per_req);
cudaError_t launch_topk_pair(vx_ctx* c, const float* scores, const vx_page_table& pt, const int32_t* budget,
                             int32_t max_budget, int32_t* sel_phys, int32_t* sel_logical, int32_t* sel_count,
                             cudaStream_t s, bool pdl, const ReqRange& rr, const PrefetchPlan& pf);
// VX_AGG_MAX over the MLA head group on the tensor cores (vx_score_mla_max.cu)
bool score_mla_max_supported(const vx_geom& g);
cudaError_t launch_score_mla_max(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt, float* scores,
                                 cudaStream_t s, const ReqRange& rr);
cudaError_t launch_union_pages(vx_ctx* c, const vx_page_table& pt, const int32_t* sel_logical, const int32_t* sel_count,
                               int32_t max_budget, int32_t max_union, int32_t* union_phys, int32_t* union_logical,
                               int32_t* union_count, cudaStream_t s);
cudaError_t launch_decode_gqa(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                              const int32_t* sel_phys, const int32_t* sel_logical,
                              const int32_t* sel_count, int32_t max_budget, void* out, float* lse,
                              cudaStream_t s, const DecodeOpts& opt = DecodeOpts());
cudaError_t launch_decode_gqa_mma(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                  const int32_t* sel_phys, const int32_t* sel_logical,
                                  const int32_t* sel_count, int32_t max_budget, void* out, float* lse,
                                  cudaStream_t s, const DecodeOpts& opt = DecodeOpts());
bool gqa_mma_supported(const vx_geom& g);
bool decode_folds_summary(const vx_ctx* c);   // the decode path of this context can take DecodeOpts::summary_upd
cudaError_t launch_decode_mla(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                              const int32_t* sel_phys, const int32_t* sel_logical,
                              const int32_t* sel_count, int32_t max_budget, void* out, float* lse,
                              cudaStream_t s, const DecodeOpts& opt = DecodeOpts());
cudaError_t launch_decode_mla_tc(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                 const int32_t* sel_phys, const int32_t* sel_logical,
                                 const int32_t* sel_count, int32_t max_budget, void* out, float* lse,
                                 cudaStream_t s, const DecodeOpts& opt = DecodeOpts());
bool mla_tc_supported(const vx_geom& g);
// the whole step of a request (score -> select -> decode -> merge) in one kernel on the cluster that owns it
bool step_mla_fused_applies(const vx_ctx* c, const vx_page_table& pt, const vx_kv_pool& pool, int32_t max_budget);   // it can run
bool step_mla_fused_pays(const vx_ctx* c, const vx_page_table& pt);                                                  // ... and is the faster schedule
cudaError_t launch_step_mla_fused(vx_ctx* c, const void* q, const vx_kv_pool& pool, const void* summary,
                                  const vx_page_table& pt, const int32_t* budget, int32_t max_budget, bool update_summary,
                                  int32_t* sel_phys, int32_t* sel_logical, int32_t* sel_count, void* out, float* lse,
                                  cudaStream_t s);
// the whole step of the batch in one persistent kernel (flat summary stream, selection warpgroups, decode items from a counter)
bool step_mla_flat_applies(const vx_ctx* c, const vx_page_table& pt, const vx_kv_pool& pool, int32_t max_budget);
size_t step_mla_flat_workspace_ints(int max_batch);
size_t step_mla_flat_qvec_floats(int max_batch);
cudaError_t launch_step_mla_flat(vx_ctx* c, const void* q, const vx_kv_pool& pool, const void* summary,
                                 const vx_page_table& pt, const int32_t* budget, int32_t max_budget, bool update_summary,
                                 int32_t* sel_phys, int32_t* sel_logical, int32_t* sel_count, void* out, float* lse,
                                 cudaStream_t s);
cudaError_t vx_trace_set_step_mla_flat(long long* buf, int ctas);
cudaError_t launch_combine(vx_ctx* c, int32_t batch, int num_splits, void* out, float* lse,
                           cudaStream_t s);

// fp8 KV cache (vx_kv_format): one-byte K / V / summary elements
inline bool kv_is_fp8(const vx_geom& g) { return g.kv_format != VX_KV_SAME; }
inline size_t kv_elem_size(const vx_geom& g) { return kv_is_fp8(g) ? 1 : (g.dtype == VX_DT_BF16 ? 2 : 4); }
bool fp8_geometry_supported(const vx_geom& g);
cudaError_t launch_score_fp8(vx_ctx* c, const void* q, const void* summary, const vx_page_table& pt, float* scores, cudaStream_t s);
bool mla_fp8_staged_supported(const vx_geom& g);
size_t mla_fp8_stage_elems(const vx_geom& g, int max_batch, int max_budget);
cudaError_t launch_decode_mla_fp8_staged(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                         const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                         int32_t max_budget, void* out, float* lse, cudaStream_t s, const DecodeOpts& opt);
cudaError_t launch_decode_fp8(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                              const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                              int32_t max_budget, void* out, float* lse, cudaStream_t s);

bool gqa_fp8_fast_supported(const vx_geom& g);           // the mma kernel of vx_decode_gqa_fp8.cu (page 16, d = 128)
cudaError_t launch_decode_gqa_fp8(vx_ctx* c, const void* q, const vx_kv_pool& pool, const vx_page_table& pt,
                                  const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                  int32_t max_budget, void* out, float* lse, cudaStream_t s, bool pdl, const int32_t* budget,
                                  void* summary_upd);

// geometry support predicates (used by vx_create validation)
bool gqa_geometry_supported(const vx_geom& g);
bool mla_geometry_supported(const vx_geom& g);
bool score_geometry_supported(const vx_geom& g);

}  // namespace vx
