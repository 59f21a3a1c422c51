// vx_api.cu -- the C ABI of include/vortex_b200.h: context, workspace, validation, dispatch.
// Every step of the path runs in the kernels of this directory; there is no CPU fallback.
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <set>
#include <utility>

#include "vx_internal.h"

namespace vx {

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static size_t elem_size(int32_t dtype) { return dtype == VX_DT_BF16 ? 2 : 4; }

Workspace carve_workspace(const vx_geom& g, void* base, int32_t max_batch, int32_t max_total_pages,
                          int32_t max_budget) {
  Workspace w{};
  size_t off = 0;
  char* b = static_cast<char*>(base);
  auto take = [&](size_t bytes) -> void* {
    void* p = b ? b + off : nullptr;
    off = align_up(off + bytes, 256);
    return p;
  };
  const size_t B = (size_t)max_batch, Hq = (size_t)g.num_q_heads, Hkv = (size_t)g.num_kv_heads;
  const size_t esz = elem_size(g.dtype);
  // (carved from the CALLER's geometry: page_size is the physical page, block_size the selection block)
  const size_t bpp = (g.block_size > 0 && g.block_size < g.page_size) ? (size_t)(g.page_size / g.block_size) : 1;
  w.scores = static_cast<float*>(take(Hkv * (size_t)max_total_pages * bpp * 4));
  w.sel_phys = static_cast<int32_t*>(take(B * Hkv * (size_t)max_budget * 4));
  w.sel_logical = static_cast<int32_t*>(take(B * Hkv * (size_t)max_budget * 4));
  w.sel_count = static_cast<int32_t*>(take(B * Hkv * 4));
  w.part_o = static_cast<float*>(take(B * Hq * kMaxSplits * (size_t)g.v_dim * 4));
  w.part_lse = static_cast<float*>(take(B * Hq * kMaxSplits * 4));
  w.unit_counter = static_cast<int32_t*>(take(B * Hkv * 4));
  w.h_q = take(B * Hq * (size_t)g.qk_dim * esz);
  // page_indptr | seq_lens | budget are one contiguous block (one host->device copy), each part 4-byte aligned
  w.h_indptr = static_cast<int32_t*>(take((3 * B + 1) * 4));
  w.h_seq_lens = w.h_indptr ? w.h_indptr + (B + 1) : nullptr;
  w.h_budget = w.h_indptr ? w.h_indptr + (2 * B + 1) : nullptr;
  w.h_indices = static_cast<int32_t*>(take((size_t)max_total_pages * 4));
  w.h_out = take(B * Hq * (size_t)g.v_dim * esz);
  w.h_lse = static_cast<float*>(take(B * Hq * 4));
  const bool mla = g.kv_shared != 0;
  w.flat_qvec = static_cast<float*>(take(mla ? step_mla_flat_qvec_floats(max_batch) * 4 : 0));
  w.flat_sync = static_cast<int32_t*>(take(mla ? step_mla_flat_workspace_ints(max_batch) * 4 : 0));
  w.blk_indptr = static_cast<int32_t*>(take(bpp > 1 ? (B + 1) * 4 : 0));
  w.blk_indices = static_cast<int32_t*>(take(bpp > 1 ? (size_t)max_total_pages * bpp * 4 : 0));
  w.topk_remap = static_cast<float*>(take(kTopkRemapMaxKnots * 4));
  w.mla_stage = take(mla_fp8_stage_elems(g, max_batch, max_budget) * 2);
  w.mla_stage_sel = static_cast<int32_t*>(take(mla_fp8_staged_supported(g) ? B * (size_t)max_budget * 4 : 0));
  w.fp8_qvec = static_cast<float*>(take(kv_is_fp8(g) ? B * Hkv * 2 * (size_t)g.qk_dim * 4 : 0));
  w.bytes = off;
  return w;
}

static char g_create_err[512] = "";

cudaError_t ensure_dyn_smem(const void* kernel, int device, int bytes) {
  static std::mutex mu;
  static std::set<std::pair<const void*, int>> done;
  std::lock_guard<std::mutex> lock(mu);
  if (done.count({kernel, device})) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess) done.insert({kernel, device});
  return e;
}

static vx_status fail(vx_ctx* c, vx_status st, const char* fmt, ...) {
  char* dst = c ? c->err : g_create_err;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(dst, 512, fmt, ap);
  va_end(ap);
  return st;
}

static const char* check_geom(const vx_geom* g, vx_status* st) {
  *st = VX_ERR_INVALID_ARG;
  if (!g) return "geom is NULL";
  if (g->dtype != VX_DT_BF16 && g->dtype != VX_DT_F32) return "dtype must be VX_DT_BF16 or VX_DT_F32";
  if (g->num_q_heads <= 0 || g->num_kv_heads <= 0 || g->num_q_heads % g->num_kv_heads != 0)
    return "num_q_heads must be a positive multiple of num_kv_heads";
  if (g->qk_dim <= 0 || g->v_dim <= 0 || g->page_size <= 0) return "qk_dim, v_dim, page_size must be positive";
  if (g->n_sink < 0 || g->n_local < 0) return "n_sink, n_local must be >= 0";
  if (g->kv_shared && g->v_dim > g->qk_dim) return "kv_shared needs v_dim <= qk_dim";
  if (g->block_size < 0 || (g->block_size > 0 && g->page_size % g->block_size != 0))
    return "block_size must be 0 (= page_size) or divide page_size";
  *st = VX_ERR_UNSUPPORTED;
  if (g->agg != VX_AGG_SUM && g->agg != VX_AGG_MAX) return "agg must be VX_AGG_SUM or VX_AGG_MAX";
  if (g->summary_kind != VX_SUMMARY_ENVELOPE && g->summary_kind != VX_SUMMARY_CENTROID)
    return "summary_kind must be VX_SUMMARY_ENVELOPE or VX_SUMMARY_CENTROID";
  if (g->kv_format != VX_KV_SAME) {            // fp8 KV cache: its own kernels (vx_score_fp8.cu, the generic decode path)
    if (g->kv_format != VX_KV_FP8_E4M3 && g->kv_format != VX_KV_FP8_E5M2) return "kv_format must be VX_KV_SAME, VX_KV_FP8_E4M3 or VX_KV_FP8_E5M2";
    if (!fp8_geometry_supported(*g))
      return "fp8 KV cache: bf16 queries, envelope summaries, VX_AGG_SUM; GQA head widths 64 / 128 (groups of <= 8 heads) or the 576 / 512 MLA latent";
    *st = VX_OK;
    return nullptr;
  }
  if (!score_geometry_supported(*g)) return "qk_dim / dtype / aggregation not supported by the score kernel (VX_AGG_MAX: GQA groups of <= 8 heads, or the bf16 MLA group of 16 / 32 heads)";
  if (g->kv_shared ? !mla_geometry_supported(*g) : !gqa_geometry_supported(*g))
    return "(dtype, qk_dim, v_dim, heads) not supported by the decode kernels";
  *st = VX_OK;
  return nullptr;
}

static vx_status check_cuda(vx_ctx* c, cudaError_t e, const char* what) {
  if (e == cudaSuccess) return VX_OK;
  return fail(c, VX_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

// every compute call: the context's kernels, workspace and per-device attributes belong to c->device
static vx_status check_device(vx_ctx* c) {
  int cur = -1;
  const cudaError_t e = cudaGetDevice(&cur);
  if (e != cudaSuccess) return fail(c, VX_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (cur != c->device)
    return fail(c, VX_ERR_INVALID_ARG, "the context is bound to device %d but the calling thread's current device is %d",
                c->device, cur);
  return VX_OK;
}

static vx_status check_table(vx_ctx* c, const vx_page_table* pt) {
  if (vx_status st = check_device(c)) return st;
  if (!pt) return fail(c, VX_ERR_INVALID_ARG, "page table is NULL");
  if (pt->batch < 0 || pt->total_pages < 0 || pt->max_pages_per_req < 0)
    return fail(c, VX_ERR_INVALID_ARG, "negative size in page table");
  if (pt->batch > 0 && (!pt->page_indptr || !pt->page_indices || !pt->seq_lens))
    return fail(c, VX_ERR_INVALID_ARG, "page table has NULL arrays");
  if (pt->batch > c->max_batch || pt->total_pages > c->max_total_pages)
    return fail(c, VX_ERR_WORKSPACE, "batch %d / total_pages %d exceed the context's maxima %d / %d",
                pt->batch, pt->total_pages, c->max_batch, c->max_total_pages);
  return VX_OK;
}

static vx_status check_pool(vx_ctx* c, const vx_kv_pool* pool) {
  if (!pool || !pool->k) return fail(c, VX_ERR_INVALID_ARG, "kv pool / k is NULL");
  if (!c->g.kv_shared && !pool->v) return fail(c, VX_ERR_INVALID_ARG, "kv pool v is NULL");
  const int64_t per16 = 16 / (int64_t)kv_elem_size(c->g);
  if (kv_is_fp8(c->g) && !(pool->k_scale > 0.f && (c->g.kv_shared || pool->v_scale > 0.f)))
    return fail(c, VX_ERR_INVALID_ARG, "fp8 KV cache: k_scale / v_scale must be positive");
  if (pool->stride_page % per16 || pool->stride_token % per16 || pool->stride_head % per16 ||
      ((uintptr_t)pool->k & 15) || (!c->g.kv_shared && ((uintptr_t)pool->v & 15)))
    return fail(c, VX_ERR_INVALID_ARG, "pool pointers and strides must be multiples of 16 bytes");
  return VX_OK;
}

// the page table the kernels work on: the caller's, or (blocks finer than the page) its expansion into a block table in
// the workspace -- request i's blocks are page_indptr[i] * bpp .., block (page, s) has the physical id page id * bpp + s
__global__ void expand_block_table_kernel(const int32_t* __restrict__ indptr, const int32_t* __restrict__ indices, int batch,
                                          int total_pages, int bpp, int32_t* __restrict__ out_indptr, int32_t* __restrict__ out_indices) {
  const int n = total_pages * bpp;
  for (int x = blockIdx.x * blockDim.x + threadIdx.x; x < n; x += gridDim.x * blockDim.x) out_indices[x] = indices[x / bpp] * bpp + x % bpp;
  for (int x = blockIdx.x * blockDim.x + threadIdx.x; x <= batch; x += gridDim.x * blockDim.x) out_indptr[x] = indptr[x] * bpp;
}

static vx_status effective_table(vx_ctx* c, const vx_page_table* pt, cudaStream_t s, vx_page_table* out) {
  *out = *pt;
  if (c->bpp == 1 || pt->batch == 0) return VX_OK;
  const int n = pt->total_pages * c->bpp;
  int blocks = (n + 255) / 256;
  if (blocks < 1) blocks = 1;
  if (blocks > c->num_sms * 8) blocks = c->num_sms * 8;
  expand_block_table_kernel<<<blocks, 256, 0, s>>>(pt->page_indptr, pt->page_indices, pt->batch, pt->total_pages, c->bpp,
                                                   c->ws.blk_indptr, c->ws.blk_indices);
  c->launches += 1;
  if (vx_status st = check_cuda(c, cudaGetLastError(), "block table")) return st;
  out->page_indptr = c->ws.blk_indptr;
  out->page_indices = c->ws.blk_indices;
  out->total_pages = n;
  out->max_pages_per_req = pt->max_pages_per_req * c->bpp;
  return VX_OK;
}

}  // namespace vx

using namespace vx;

extern "C" {

size_t vx_workspace_bytes(const vx_geom* g, int32_t max_batch, int32_t max_total_pages,
                          int32_t max_pages_per_req, int32_t max_budget) {
  vx_status st;
  if (check_geom(g, &st) || max_batch < 0 || max_total_pages < 0 || max_pages_per_req < 0 || max_budget < 0)
    return 0;
  return carve_workspace(*g, nullptr, max_batch, max_total_pages, max_budget).bytes;
}

vx_status vx_create(vx_ctx** out, const vx_geom* g, int device, void* workspace, size_t workspace_bytes,
                    int32_t max_batch, int32_t max_total_pages, int32_t max_pages_per_req,
                    int32_t max_budget) {
  if (!out) return fail(nullptr, VX_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  vx_status st;
  if (const char* why = check_geom(g, &st)) return fail(nullptr, st, "%s", why);
  if (max_batch < 0 || max_total_pages < 0 || max_pages_per_req < 0 || max_budget < 0)
    return fail(nullptr, VX_ERR_INVALID_ARG, "negative maximum");
  const size_t need = carve_workspace(*g, nullptr, max_batch, max_total_pages, max_budget).bytes;
  if (!workspace || ((uintptr_t)workspace & 255))
    return fail(nullptr, VX_ERR_INVALID_ARG, "workspace must be a 256-byte aligned device pointer");
  if (workspace_bytes < need)
    return fail(nullptr, VX_ERR_WORKSPACE, "workspace has %zu bytes, %zu needed", workspace_bytes, need);
  cudaError_t e = cudaSetDevice(device);
  if (e != cudaSuccess) return fail(nullptr, VX_ERR_CUDA, "cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, device);
  if (e != cudaSuccess) return fail(nullptr, VX_ERR_CUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(e));
  if (prop.major != 10)
    return fail(nullptr, VX_ERR_UNSUPPORTED, "device %d is sm_%d%d; this library is built for sm_100a only",
                device, prop.major, prop.minor);
  vx_ctx* c = new (std::nothrow) vx_ctx();
  if (!c) return fail(nullptr, VX_ERR_INVALID_ARG, "out of host memory");
  c->g = *g;
  // blocks finer than the page: from here on the kernels' "page" is the selection block (G28); the physical page survives
  // in user_page_size / bpp, which only the kernels that address the KV pool need
  c->user_page_size = g->page_size;
  c->bpp = (g->block_size > 0 && g->block_size < g->page_size) ? g->page_size / g->block_size : 1;
  c->g.page_size = g->page_size / c->bpp;
  c->g.block_size = c->g.page_size;
  c->device = device;
  c->num_sms = prop.multiProcessorCount;
  c->l2_bytes = prop.l2CacheSize;
  c->max_batch = max_batch;
  c->max_total_pages = max_total_pages;
  c->max_pages_per_req = max_pages_per_req;
  c->max_budget = max_budget;
  c->ws = carve_workspace(*g, workspace, max_batch, max_total_pages, max_budget);
  c->launches = 0;
  c->err[0] = 0;
  c->mla_step = VX_MLA_STEP_AUTO;
  c->pinned_small = nullptr;
  e = cudaHostAlloc(reinterpret_cast<void**>(&c->pinned_small), (3 * (size_t)(max_batch > 0 ? max_batch : 1) + 1) * 4, cudaHostAllocDefault);
  if (e != cudaSuccess) {
    delete c;
    return fail(nullptr, VX_ERR_CUDA, "pinned staging for the host entry point: %s", cudaGetErrorString(e));
  }
  c->flat_splits = c->flat_waves = 0;
  // split-arrival counters start at zero and every step leaves them at zero
  e = cudaMemset(c->ws.unit_counter, 0, (size_t)(max_batch > 0 ? max_batch : 1) * g->num_kv_heads * 4);
  if (e == cudaSuccess && g->kv_shared) e = cudaMemset(c->ws.flat_sync, 0, step_mla_flat_workspace_ints(max_batch) * 4);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  if (e != cudaSuccess) {
    cudaFreeHost(c->pinned_small);
    delete c;
    return fail(nullptr, VX_ERR_CUDA, "workspace initialisation: %s", cudaGetErrorString(e));
  }
  *out = c;
  return VX_OK;
}

void vx_destroy(vx_ctx* ctx) {
  if (ctx && ctx->pinned_small) cudaFreeHost(ctx->pinned_small);
  delete ctx;
}

const char* vx_last_error(const vx_ctx* ctx) { return ctx ? ctx->err : g_create_err; }

int32_t vx_last_launch_count(const vx_ctx* ctx) { return ctx ? ctx->launches : 0; }

vx_status vx_trace_attach(vx_ctx* c, void* buffer, int32_t max_ctas, int32_t kernels) {
  if (!c) return VX_ERR_INVALID_ARG;
  if (max_ctas < 0) return fail(c, VX_ERR_INVALID_ARG, "negative max_ctas");
  if (cudaError_t e = cudaSetDevice(c->device)) return check_cuda(c, e, "vx_trace_attach");
  long long* b = static_cast<long long*>(buffer);
  const int n = buffer ? max_ctas : 0;
  // one kind: its CTAs' rows start at row 0.  Several kinds at once (a whole step on one time line): the score kernel's
  // rows start at 0, the selection kernels' at 1024, the decode kernels' at 4096
  const bool many = (kernels & (kernels - 1)) != 0;
  const int o_topk = many ? 1024 : 0, o_dec = many ? 4096 : 0;
  auto at = [&](int off) -> long long* { return b ? b + (long long)off * 16 : nullptr; };
  auto left = [&](int off) -> int { return n > off ? n - off : 0; };
  cudaError_t e = vx_trace_set_score((kernels & VX_TRACE_SCORE) ? b : nullptr, n);
  if (e == cudaErrorNotSupported) return fail(c, VX_ERR_UNSUPPORTED, "this library was built without -DVX_TRACE");
  if (e == cudaSuccess) e = vx_trace_set_topk((kernels & VX_TRACE_TOPK) ? at(o_topk) : nullptr, left(o_topk));
  if (e == cudaSuccess) e = vx_trace_set_decode_gqa((kernels & VX_TRACE_DECODE) ? at(o_dec) : nullptr, left(o_dec));
  if (e == cudaSuccess) e = vx_trace_set_decode_mla((kernels & VX_TRACE_DECODE) ? at(o_dec) : nullptr, left(o_dec));
  if (e == cudaSuccess) e = vx_trace_set_step_mla((kernels & VX_TRACE_DECODE) ? at(o_dec) : nullptr, left(o_dec));
  if (e == cudaSuccess) e = vx_trace_set_step_mla_flat((kernels & VX_TRACE_DECODE) ? at(o_dec) : nullptr, left(o_dec));
  return check_cuda(c, e, "vx_trace_attach");
}

vx_status vx_page_summary_update(vx_ctx* c, const vx_kv_pool* pool, const vx_page_table* pt,
                                 const int32_t* first_new_pos, void* summary, vx_stream stream) {
  if (!c) return VX_ERR_INVALID_ARG;
  c->launches = 0;
  if (vx_status st = check_table(c, pt)) return st;
  vx_page_table pt_eff;                          // (the block table when blocks are finer than the page)
  if (vx_status st = effective_table(c, pt, (cudaStream_t)stream, &pt_eff)) return st;
  pt = &pt_eff;
  if (vx_status st = check_pool(c, pool)) return st;
  if (!summary) return fail(c, VX_ERR_INVALID_ARG, "summary is NULL");
  return check_cuda(c, launch_summary_update(c, *pool, *pt, first_new_pos, summary, (cudaStream_t)stream),
                    "vx_page_summary_update");
}

vx_status vx_page_score(vx_ctx* c, const void* q, const void* summary, const vx_page_table* pt, float* scores,
                        vx_stream stream) {
  if (!c) return VX_ERR_INVALID_ARG;
  c->launches = 0;
  if (vx_status st = check_table(c, pt)) return st;
  vx_page_table pt_eff;                          // (the block table when blocks are finer than the page)
  if (vx_status st = effective_table(c, pt, (cudaStream_t)stream, &pt_eff)) return st;
  pt = &pt_eff;
  if (!q || !summary || !scores) return fail(c, VX_ERR_INVALID_ARG, "q / summary / scores is NULL");
  return check_cuda(c, launch_page_score(c, q, summary, *pt, scores, (cudaStream_t)stream), "vx_page_score");
}

vx_status vx_topk_pages(vx_ctx* c, const float* scores, const vx_page_table* pt, const int32_t* budget,
                        int32_t max_budget, int32_t* sel_phys, int32_t* sel_logical, int32_t* sel_count,
                        vx_stream stream) {
  if (!c) return VX_ERR_INVALID_ARG;
  c->launches = 0;
  if (vx_status st = check_table(c, pt)) return st;
  vx_page_table pt_eff;                          // (the block table when blocks are finer than the page)
  if (vx_status st = effective_table(c, pt, (cudaStream_t)stream, &pt_eff)) return st;
  pt = &pt_eff;
  if (!scores || !budget || !sel_phys || !sel_count)
    return fail(c, VX_ERR_INVALID_ARG, "scores / budget / sel_phys / sel_count is NULL");
  if (max_budget <= 0) return fail(c, VX_ERR_INVALID_ARG, "max_budget must be positive");
  return check_cuda(c, launch_topk_pages(c, scores, *pt, budget, max_budget, sel_phys, sel_logical, sel_count,
                                         (cudaStream_t)stream), "vx_topk_pages");
}

vx_status vx_topk_pages_approx(vx_ctx* c, const float* scores, const vx_page_table* pt, const int32_t* budget,
                               int32_t max_budget, float tolerate_ratio, uint64_t seed, int32_t* sel_phys,
                               int32_t* sel_logical, int32_t* sel_count, vx_stream stream) {
  if (!c) return VX_ERR_INVALID_ARG;
  c->launches = 0;
  if (vx_status st = check_table(c, pt)) return st;
  vx_page_table pt_eff;                          // (the block table when blocks are finer than the page)
  if (vx_status st = effective_table(c, pt, (cudaStream_t)stream, &pt_eff)) return st;
  pt = &pt_eff;
  if (!scores || !budget || !sel_phys || !sel_count)
    return fail(c, VX_ERR_INVALID_ARG, "scores / budget / sel_phys / sel_count is NULL");
  if (max_budget <= 0) return fail(c, VX_ERR_INVALID_ARG, "max_budget must be positive");
  if (!(tolerate_ratio >= 0.f && tolerate_ratio <= 1.f))
    return fail(c, VX_ERR_INVALID_ARG, "tolerate_ratio %g outside [0, 1]", (double)tolerate_ratio);
  ApproxPlan ap = c->approx;                     // (the remap table, if one is installed)
  ap.tolerate_ratio = tolerate_ratio;
  ap.seed = seed;
  if (ap.active() && !approx_topk_supported(pt->max_pages_per_req, max_budget))
    return fail(c, VX_ERR_UNSUPPORTED, "approximate top-k handles at most %d pages per request (budgets above %d: %d pages); got %d",
                kTopkApproxMaxPages, kTopkApproxMaxBudgetLong, kTopkRegMaxPages, pt->max_pages_per_req);
  return check_cuda(c, launch_topk_pages(c, scores, *pt, budget, max_budget, sel_phys, sel_logical, sel_count,
                                         (cudaStream_t)stream, false, ReqRange(), PrefetchPlan(), ap),
                    "vx_topk_pages_approx");
}

vx_status vx_set_topk_approx(vx_ctx* c, float tolerate_ratio, uint64_t seed) {
  if (!c) return VX_ERR_INVALID_ARG;
  if (!(tolerate_ratio >= 0.f && tolerate_ratio <= 1.f))
    return fail(c, VX_ERR_INVALID_ARG, "tolerate_ratio %g outside [0, 1]", (double)tolerate_ratio);
  c->approx.tolerate_ratio = tolerate_ratio;
  c->approx.seed = seed;
  return VX_OK;
}

vx_status vx_set_topk_remap(vx_ctx* c, const float* knots, int32_t n_knots) {
  if (!c) return VX_ERR_INVALID_ARG;
  if (n_knots == 0) {                            // back to the per-request linear map
    c->approx.remap = nullptr;
    c->approx.remap_n = 0;
    return VX_OK;
  }
  if (!knots || n_knots < 2 || n_knots > kTopkRemapMaxKnots)
    return fail(c, VX_ERR_INVALID_ARG, "remap: 2..%d knots (0 clears the table); got %d", kTopkRemapMaxKnots, n_knots);
  for (int i = 0; i < n_knots; ++i)
    if (!(knots[i] >= 0.f && knots[i] <= 1.f) || (i > 0 && knots[i] < knots[i - 1]))
      return fail(c, VX_ERR_INVALID_ARG, "remap: knot %d = %g; knots must lie in [0, 1] and never decrease", i, (double)knots[i]);
  if (vx_status st = check_device(c)) return st;
  // (synchronous set-up call: the table is in place when it returns; a selection already in flight may read either table)
  if (vx_status st = check_cuda(c, cudaMemcpy(c->ws.topk_remap, knots, (size_t)n_knots * 4, cudaMemcpyHostToDevice), "remap table"))
    return st;
  c->approx.remap = c->ws.topk_remap;
  c->approx.remap_n = n_knots;
  return VX_OK;
}

vx_status vx_set_option(vx_ctx* c, int32_t option, int32_t value) {
  if (!c) return VX_ERR_INVALID_ARG;
  if (option == VX_OPT_MLA_STEP && value >= VX_MLA_STEP_AUTO && value <= VX_MLA_STEP_FLAT) {
    c->mla_step = value;
    return VX_OK;
  }
  if (option == VX_OPT_MLA_FLAT_SPLITS && value >= 0 && value <= kMaxSplits) { c->flat_splits = value; return VX_OK; }
  if (option == VX_OPT_MLA_FLAT_WAVES && value >= 0 && value <= 8) { c->flat_waves = value; return VX_OK; }
  return fail(c, VX_ERR_INVALID_ARG, "unknown option %d / value %d", option, value);
}

vx_status vx_union_pages(vx_ctx* c, const vx_page_table* pt, const int32_t* sel_logical, const int32_t* sel_count,
                         int32_t max_budget, int32_t max_union, int32_t* union_phys, int32_t* union_logical,
                         int32_t* union_count, vx_stream stream) {
  if (!c) return VX_ERR_INVALID_ARG;
  c->launches = 0;
  if (vx_status st = check_table(c, pt)) return st;
  vx_page_table pt_eff;                          // (the block table when blocks are finer than the page)
  if (vx_status st = effective_table(c, pt, (cudaStream_t)stream, &pt_eff)) return st;
  pt = &pt_eff;
  if (!sel_logical || !sel_count || !union_phys || !union_count)
    return fail(c, VX_ERR_INVALID_ARG, "sel_logical / sel_count / union_phys / union_count is NULL");
  if (max_budget <= 0) return fail(c, VX_ERR_INVALID_ARG, "max_budget must be positive");
  const int64_t largest = (int64_t)c->g.num_kv_heads * max_budget;
  const int64_t bound = largest < pt->max_pages_per_req ? largest : pt->max_pages_per_req;
  if (max_union < bound)
    return fail(c, VX_ERR_INVALID_ARG, "max_union %d below the largest possible union %lld", max_union, (long long)bound);
  cudaError_t e = launch_union_pages(c, *pt, sel_logical, sel_count, max_budget, max_union, union_phys, union_logical,
                                     union_count, (cudaStream_t)stream);
  if (e == cudaErrorNotSupported) return fail(c, VX_ERR_UNSUPPORTED, "more than 393,184 pages per request");
  return check_cuda(c, e, "vx_union_pages");
}

static vx_status decode_dispatch(vx_ctx* c, const void* q, const vx_kv_pool* pool, const vx_page_table* pt,
                                 const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                 int32_t max_budget, void* out, float* lse, cudaStream_t s,
                                 const DecodeOpts& opt = DecodeOpts()) {
  if (gqa_fp8_fast_supported(c->g))
    return check_cuda(c, launch_decode_gqa_fp8(c, q, *pool, *pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s,
                                               opt.pdl, opt.budget, opt.summary_upd), "vx_sparse_paged_decode (fp8 KV cache)");
  if (mla_fp8_staged_supported(c->g) && c->bpp == 1 && opt.rr.count < 0 && max_budget <= c->max_budget)
    return check_cuda(c, launch_decode_mla_fp8_staged(c, q, *pool, *pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s, opt),
                      "vx_sparse_paged_decode (fp8 latent cache)");
  if (kv_is_fp8(c->g))
    return check_cuda(c, launch_decode_fp8(c, q, *pool, *pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s),
                      "vx_sparse_paged_decode (fp8 KV cache)");
  cudaError_t e = c->g.kv_shared
                      ? launch_decode_mla(c, q, *pool, *pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s, opt)
                      : launch_decode_gqa(c, q, *pool, *pt, sel_phys, sel_logical, sel_count, max_budget, out, lse, s, opt);
  return check_cuda(c, e, "vx_sparse_paged_decode");
}

vx_status vx_sparse_paged_decode(vx_ctx* c, const void* q, const vx_kv_pool* pool, const vx_page_table* pt,
                                 const int32_t* sel_phys, const int32_t* sel_logical, const int32_t* sel_count,
                                 int32_t max_budget, void* out, float* lse, vx_stream stream) {
  if (!c) return VX_ERR_INVALID_ARG;
  c->launches = 0;
  if (vx_status st = check_table(c, pt)) return st;
  vx_page_table pt_eff;                          // (the block table when blocks are finer than the page)
  if (vx_status st = effective_table(c, pt, (cudaStream_t)stream, &pt_eff)) return st;
  pt = &pt_eff;
  if (vx_status st = check_pool(c, pool)) return st;
  if (!q || !sel_phys || !sel_logical || !sel_count || !out)
    return fail(c, VX_ERR_INVALID_ARG, "q / sel_phys / sel_logical / sel_count / out is NULL");
  if (max_budget <= 0) return fail(c, VX_ERR_INVALID_ARG, "max_budget must be positive");
  if (pt->batch == 0) return VX_OK;
  return decode_dispatch(c, q, pool, pt, sel_phys, sel_logical, sel_count, max_budget, out, lse,
                         (cudaStream_t)stream);
}

vx_status vx_sparse_decode_step(vx_ctx* c, const void* q, const vx_kv_pool* pool, void* summary,
                                const vx_page_table* pt, const int32_t* budget, int32_t max_budget,
                                uint32_t flags, void* out, float* lse, int32_t* sel_phys, int32_t* sel_logical,
                                int32_t* sel_count, vx_stream stream) {
  if (!c) return VX_ERR_INVALID_ARG;
  c->launches = 0;
  if (vx_status st = check_table(c, pt)) return st;
  vx_page_table pt_eff;                          // (the block table when blocks are finer than the page)
  if (vx_status st = effective_table(c, pt, (cudaStream_t)stream, &pt_eff)) return st;
  pt = &pt_eff;
  if (vx_status st = check_pool(c, pool)) return st;
  if (!q || !summary || !budget || !out) return fail(c, VX_ERR_INVALID_ARG, "q / summary / budget / out is NULL");
  if (max_budget <= 0 || max_budget > c->max_budget)
    return fail(c, VX_ERR_WORKSPACE, "max_budget %d outside (0, %d]", max_budget, c->max_budget);
  if (pt->batch == 0) return VX_OK;
  ApproxPlan ap;                                 // exact unless the caller asks for the lossy selection
  if (flags & VX_STEP_APPROX_TOPK) {
    ap = c->approx;
    if (ap.active() && !approx_topk_supported(pt->max_pages_per_req, max_budget))
      return fail(c, VX_ERR_UNSUPPORTED, "approximate top-k handles at most %d pages per request (budgets above %d: %d pages); got %d",
                  kTopkApproxMaxPages, kTopkApproxMaxBudgetLong, kTopkRegMaxPages, pt->max_pages_per_req);
  }
  cudaStream_t s = (cudaStream_t)stream;
  int32_t* sp = sel_phys ? sel_phys : c->ws.sel_phys;
  int32_t* sl = sel_logical ? sel_logical : c->ws.sel_logical;
  int32_t* sc = sel_count ? sel_count : c->ws.sel_count;
  // (a1) With n_local >= 1 the newest page is a forced page: its score never decides the selection and its keys
  // are staged by the decode kernel anyway, so the decode kernel rebuilds its summary (same result, no extra
  // launch, no extra HBM bytes).  Otherwise the summary kernel runs first.
  // MLA: the whole step of a request runs in one kernel on the cluster that owns it (vx_decode_mla.cu, FUSED)
  // MLA, small batches: the whole step of a request runs in one kernel on the cluster that owns it (vx_step_mla.cu)
  if (c->g.kv_shared && !(flags & VX_STEP_APPROX_TOPK) && c->mla_step == VX_MLA_STEP_FLAT &&
      step_mla_flat_applies(c, *pt, *pool, max_budget))
    return check_cuda(c, launch_step_mla_flat(c, q, *pool, summary, *pt, budget, max_budget,
                                              (flags & VX_STEP_UPDATE_SUMMARY) != 0, sp, sl, sc, out, lse, s),
                      "flat MLA step");
  if (c->g.kv_shared && !(flags & VX_STEP_APPROX_TOPK) && c->mla_step != VX_MLA_STEP_CHAINED && c->mla_step != VX_MLA_STEP_FLAT &&
      step_mla_fused_applies(c, *pt, *pool, max_budget) && (c->mla_step == VX_MLA_STEP_FUSED || step_mla_fused_pays(c, *pt)))
    return check_cuda(c, launch_step_mla_fused(c, q, *pool, summary, *pt, budget, max_budget,
                                               (flags & VX_STEP_UPDATE_SUMMARY) != 0, sp, sl, sc, out, lse, s),
                      "fused MLA step");
  DecodeOpts opt;
  opt.pdl = true;                                // the kernels of a step are chained by programmatic dependent launch
  opt.budget = budget;
  if (flags & VX_STEP_UPDATE_SUMMARY) {
    if (c->g.n_local >= 1 && decode_folds_summary(c)) {
      opt.summary_upd = summary;
    } else if (vx_status st = check_cuda(c, launch_summary_update(c, *pool, *pt, nullptr, summary, s), "summary update")) {
      return st;
    }
  }
  if (vx_status st = check_cuda(c, launch_page_score(c, q, summary, *pt, c->ws.scores, s), "page score")) return st;
  // L2 prefetch plan for the decode kernel's first pages (fast decode paths with contiguous page chunks only): the
  // selection kernel's emission issues it while HBM would otherwise idle between the two kernels.
  // GQA: the first 6 pages of every split, at most 16 MB in all (measured on C3: 88.8 us against 89.8 without;
  // 4 / 8 pages 89.2-89.4, 48 MB and more slower -- the prefetch then delays the selection kernel's own tail), none
  // when a big batch leaves fewer than 4 (C5).  MLA (73.7 KB pages): the first page only (C4 71.0 -> 70.1 us with 1
  // page, 72.1 / 74.0 / 75.8 with 2 / 3 / 4 -- the decode kernel's first TMA boxes queue behind the prefetches).
  PrefetchPlan pf;
  const int64_t esz = (int64_t)elem_size(c->g.dtype);
  if (decode_folds_summary(c) && !kv_is_fp8(c->g) && pool->stride_token == c->g.qk_dim && c->bpp == 1) {
    pf.k = pool->k;
    pf.v = c->g.kv_shared ? nullptr : pool->v;
    pf.page_bytes = pool->stride_page * esz;
    pf.head_bytes = pool->stride_head * esz;
    pf.chunk_bytes = (uint32_t)(c->g.page_size * c->g.qk_dim * esz);
    pf.splits = c->g.kv_shared ? decode_mla_splits(c, pt->batch, max_budget) : decode_gqa_splits(c, pt->batch, max_budget);
    const int64_t per_page = (int64_t)pf.chunk_bytes * (pf.v ? 2 : 1);
    const int64_t units = (int64_t)pt->batch * c->g.num_kv_heads * pf.splits;
    const int64_t cap = ((int64_t)16 << 20) / (units * per_page > 0 ? units * per_page : 1);
    const int want = c->g.kv_shared ? 1 : 6;
    pf.pages_per_split = (int)(want < cap ? want : cap);
    if (!c->g.kv_shared && cap < 4) pf.pages_per_split = 0;
    if (pf.pages_per_split < 1) pf.k = nullptr;
  }
  if (vx_status st = check_cuda(c, launch_topk_pages(c, c->ws.scores, *pt, budget, max_budget, sp, sl, sc, s, true,
                                                     ReqRange(), pf, ap), "top-k pages"))
    return st;
  return decode_dispatch(c, q, pool, pt, sp, sl, sc, max_budget, out, lse, s, opt);
}

vx_status vx_sparse_decode_step_host(vx_ctx* c, const void* h_q, const vx_kv_pool* pool, void* summary,
                                     int32_t batch, const int32_t* h_page_indptr, const int32_t* h_page_indices,
                                     const int32_t* h_seq_lens, const int32_t* h_budget, int32_t max_budget,
                                     uint32_t flags, void* h_out, float* h_lse, vx_stream stream) {
  if (!c) return VX_ERR_INVALID_ARG;
  c->launches = 0;
  if (batch < 0 || batch > c->max_batch) return fail(c, VX_ERR_WORKSPACE, "batch %d outside [0, %d]", batch, c->max_batch);
  if (batch == 0) return VX_OK;
  if (!h_q || !h_page_indptr || !h_page_indices || !h_seq_lens || !h_budget || !h_out)
    return fail(c, VX_ERR_INVALID_ARG, "a host input / output pointer is NULL");
  const int32_t total = h_page_indptr[batch];
  if (total < 0 || total > c->max_total_pages)
    return fail(c, VX_ERR_WORKSPACE, "total_pages %d outside [0, %d]", total, c->max_total_pages);
  int32_t max_pages = 0;
  for (int32_t i = 0; i < batch; ++i) {
    const int32_t p = h_page_indptr[i + 1] - h_page_indptr[i];
    if (p < 0) return fail(c, VX_ERR_INVALID_ARG, "page_indptr is not non-decreasing at %d", i);
    if (p > max_pages) max_pages = p;
  }
  const vx_geom& g = c->g;
  const size_t esz = elem_size(g.dtype);
  cudaStream_t s = (cudaStream_t)stream;
  Workspace& w = c->ws;
  const size_t q_bytes = (size_t)batch * g.num_q_heads * g.qk_dim * esz;
  const size_t o_bytes = (size_t)batch * g.num_q_heads * g.v_dim * esz;
  // three copies in: the page ids first (the score kernel's first loads), then the three small arrays packed into the
  // context's pinned staging block (a few hundred bytes; one transfer instead of three), then the queries.  The call is
  // synchronous, so the staging block is free again when it returns.
  const size_t B = (size_t)batch;
  memcpy(c->pinned_small, h_page_indptr, (B + 1) * 4);
  memcpy(c->pinned_small + (B + 1), h_seq_lens, B * 4);
  memcpy(c->pinned_small + (2 * B + 1), h_budget, B * 4);
  int32_t* d_indptr = w.h_indptr;                       // device block laid out like the staging block for THIS batch
  int32_t* d_seq = d_indptr + (B + 1);
  int32_t* d_budget = d_indptr + (2 * B + 1);
  cudaError_t e = cudaMemcpyAsync(w.h_indices, h_page_indices, (size_t)total * 4, cudaMemcpyHostToDevice, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_indptr, c->pinned_small, (3 * B + 1) * 4, cudaMemcpyHostToDevice, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(w.h_q, h_q, q_bytes, cudaMemcpyHostToDevice, s);
  if (vx_status st = check_cuda(c, e, "host->device copies")) return st;
  vx_page_table pt{batch, d_indptr, w.h_indices, d_seq, total, max_pages};
  vx_status st = vx_sparse_decode_step(c, w.h_q, pool, summary, &pt, d_budget, max_budget, flags, w.h_out,
                                       w.h_lse, nullptr, nullptr, nullptr, stream);
  if (st != VX_OK) return st;
  e = cudaMemcpyAsync(h_out, w.h_out, o_bytes, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess && h_lse)
    e = cudaMemcpyAsync(h_lse, w.h_lse, (size_t)batch * g.num_q_heads * 4, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  return check_cuda(c, e, "device->host copies");
}

}  // extern "C"
