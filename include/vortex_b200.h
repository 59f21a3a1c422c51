/*
 * vortex_b200.h -- C ABI of the B200 (sm_100a) sparse decode hot path of
 * arxiv/paper_2606_06453 ("Vortex": dynamic sparse attention over a paged KV cache).
 *
 * One decode step, per layer (PAPER.md:87-99 section 3.1; :546 App. G shared pipeline):
 *   (a1) page summaries      channel-wise min / max of the keys of each page          (:546)
 *   (a2) page scores         u[h,j] = sum_c max(q_h[c]*M_j[c], q_h[c]*m_j[c]),
 *                            aggregated over the query heads of one KV head            (:552, :92)
 *   (a3) top-k pages         per (request, KV head); first n_sink and last n_local
 *                            pages always kept; ties -> lower logical page             (:92 Eq.3, :280)
 *   (a4) sparse attention    softmax(q K_I^T * sm_scale) V_I over the selected pages,
 *                            reached through the page table, split along pages         (:92 Eq.4, :200)
 *   (a5) combine             merge the splits by log-sum-exp                           (:75)
 *
 * Conventions
 *  - All pointers are DEVICE pointers unless the parameter is marked "host".  Buffers are
 *    caller-owned; the library never allocates or frees device memory and keeps scratch
 *    only in the workspace given to vx_create.
 *  - Calls are asynchronous on `stream` (a cudaStream_t passed as void*; NULL = default
 *    stream), never synchronise, never read device memory on the host, and can be captured
 *    in a CUDA graph -- except vx_sparse_decode_step_host, which is synchronous.
 *  - Return value is a vx_status; nothing throws or aborts across the ABI.  Only
 *    host-visible arguments are validated.  vx_last_error gives a text for the last
 *    failure on that context.
 *  - A context is bound to one geometry and one device and is not thread-safe.
 *  - Inputs must be finite; behaviour on NaN/Inf is undefined (padding uses -1 / -inf).
 *  - There is no CPU fallback: without a CUDA device every compute call returns VX_ERR_CUDA.
 *
 * Page table = the paper's layout metadata C = (b, p, I) (PAPER.md:166 Eq.5, :438):
 * request i owns logical pages 0..P_i-1, P_i = ceil(seq_lens[i] / page_size); logical page j
 * lives in physical page page_indices[page_indptr[i] + j]; only the last page may be partial.
 * Named caches (the summaries) are paged with the SAME physical ids as the KV pool (:180).
 */
#ifndef VORTEX_B200_H_
#define VORTEX_B200_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vx_ctx vx_ctx; /* opaque */
typedef void *vx_stream;      /* cudaStream_t */

typedef enum {
  VX_OK = 0,
  VX_ERR_INVALID_ARG = 1, /* null pointer, negative size, inconsistent sizes */
  VX_ERR_UNSUPPORTED = 2, /* geometry / dtype / option the kernels are not built for */
  VX_ERR_WORKSPACE = 3,   /* workspace too small for this call's sizes */
  VX_ERR_CUDA = 4         /* CUDA runtime / launch failure (text in vx_last_error) */
} vx_status;

typedef enum { VX_DT_BF16 = 0, VX_DT_F32 = 1 } vx_dtype;

/* aggregation of per-head envelope scores over the heads of one KV head.
 * SUM ranks like the paper's mean ("topK(Sum(s))"); MAX is the max_h variant of
 * App. G (:556): built for GQA groups of <= 8 heads (g flop per byte on CUDA cores) and, as a tensor-core
 * contraction, for the bf16 MLA group of 16 or 32 heads on one 576-wide latent head with envelope summaries;
 * any other (geometry, MAX) pair makes vx_create return VX_ERR_UNSUPPORTED. */
typedef enum { VX_AGG_SUM = 0, VX_AGG_MAX = 1 } vx_agg;

/* what a page summary is (the query-independent cache of the flow):
 *  ENVELOPE  Quest: channel-wise min / max of the page's keys (:546); score = envelope upper bound (:552).
 *            summary: [num_pool_pages, Hkv, 2, qk_dim], [..,0,:] = min, [..,1,:] = max.
 *  CENTROID  block top-k (:85-99 section 3.1): mean of the page's valid keys, rounded to the KV dtype (:92 Eq.1);
 *            score = sum over the head group of q_h . centroid (:92 Eq.2; ranks like the paper's mean).
 *            summary: [num_pool_pages, Hkv, qk_dim] -- half the bytes.  VX_AGG_SUM only. */
typedef enum { VX_SUMMARY_ENVELOPE = 0, VX_SUMMARY_CENTROID = 1 } vx_summary_kind;

/* storage format of the KV cache (PAPER.md:200 "fp8 KV cache", :520 / :525 kv_cache_dtype "fp8_e4m3", "fp8_e5m2"):
 *  SAME      K, V pools and summaries hold elements of geom.dtype.
 *  FP8_E4M3  OCP E4M3 (bias 7, no infinities, S.1111.111 = NaN, max 448) / FP8_E5M2  OCP E5M2 (bias 15, IEEE-like):
 *            K, V pools and the summary pool hold one-byte codes; a code c stands for  scale * decode(c)  with one
 *            fp32 scale per pool tensor (vx_kv_pool.k_scale / .v_scale; the MLA latent pool uses k_scale for both
 *            roles).  q, out and lse stay in geom.dtype, which must be VX_DT_BF16.  Summaries are the min / max CODES
 *            (exact); page scores are computed on decoded codes without k_scale -- a positive factor common to every
 *            page changes no selection -- so vx_page_score returns  oracle score / k_scale  (G25-G27).
 *            Envelope summaries and VX_AGG_SUM only; pool strides are in one-byte elements.
 *            Workspace: for the absorbed-MLA geometry (kv_shared, d 576, dv 512, page 64) a context holds a bf16
 *            staging pool of max_batch * max_budget pages (73,728 B each), into which the selected fp8 pages are widened
 *            (exactly) before the tensor-core decode kernel runs on them -- vx_workspace_bytes includes it. */
typedef enum { VX_KV_SAME = 0, VX_KV_FP8_E4M3 = 1, VX_KV_FP8_E5M2 = 2 } vx_kv_format;

typedef struct {
  int32_t dtype;        /* vx_dtype of q, K, V, summaries and out */
  int32_t num_q_heads;  /* Hq */
  int32_t num_kv_heads; /* Hkv; Hq % Hkv == 0; MLA: 1 */
  int32_t qk_dim;       /* d: width of q and K rows (MLA: 576 = 512 latent + 64 RoPE) */
  int32_t v_dim;        /* dv: width of V rows and of out (MLA: 512) */
  int32_t page_size;    /* b tokens per page */
  int32_t kv_shared;    /* 1 = MLA absorbed: V_t = K_t[0:v_dim]; pool.v is ignored */
  float sm_scale;       /* softmax scale of (a4); scores of (a2) are unscaled (:92 Eq.2) */
  int32_t n_sink;       /* first pages always selected (:280) */
  int32_t n_local;      /* last pages always selected (:280); precondition n_sink+n_local <= budget[i] */
  int32_t agg;          /* vx_agg */
  int32_t summary_kind; /* vx_summary_kind */
  int32_t kv_format;    /* vx_kv_format: storage of the K, V and summary pools (0 = elements of dtype) */
  int32_t block_size;   /* selection block b_s in tokens (PAPER.md:518-519 `block_size: 16` inside `page_size: 32`; :202):
                         * 0 or page_size = the page; otherwise it must divide page_size.  A block is b_s consecutive tokens
                         * inside one physical page; everything the calls below do per page they then do per BLOCK:
                         * summaries are [num_pool_pages * (page_size / b_s), Hkv, ..] addressed by the physical block id
                         * page id * (page_size / b_s) + block in page, scores are [Hkv, total_pages * (page_size / b_s)]
                         * (request i's blocks start at page_indptr[i] * page_size / b_s), budget / n_sink / n_local count
                         * blocks, sel_logical / sel_phys hold logical / physical block ids.  The page table stays the
                         * caller's page table (G28).  Fast decode kernels: GQA with b_s = 16. */
} vx_geom;

typedef struct {
  int32_t batch;               /* host: number of requests B */
  const int32_t *page_indptr;  /* dev [B+1], page_indptr[0] = 0 */
  const int32_t *page_indices; /* dev [total_pages] physical page ids in logical order */
  const int32_t *seq_lens;     /* dev [B] tokens incl. the one just appended, >= 1 */
  int32_t total_pages;         /* host copy of page_indptr[B] */
  int32_t max_pages_per_req;   /* host upper bound of P_i (sizes grids) */
} vx_page_table;

/* K and V pools, addressed in ELEMENTS:
 *   elem(page p, token t, head h, channel c) = p*stride_page + t*stride_token + h*stride_head + c
 * The same strides serve k and v.  Rows (qk_dim channels) are contiguous and 16-byte aligned:
 * base pointers and all strides must be multiples of 16 bytes. */
typedef struct {
  const void *k;
  const void *v; /* ignored when geom.kv_shared */
  int64_t stride_page, stride_token, stride_head;
  int32_t num_pool_pages;
  float k_scale, v_scale; /* fp8 pools only (geom.kv_format != VX_KV_SAME): value = scale * decode(code); must be > 0 */
} vx_kv_pool;

/* ---- context ------------------------------------------------------------------------ */

/* Bytes of device workspace a context needs for calls with batch <= max_batch,
 * total_pages <= max_total_pages, max_pages_per_req <= max_pages_per_req, max_budget <= max_budget.
 * Returns 0 if the geometry is invalid. */
size_t vx_workspace_bytes(const vx_geom *g, int32_t max_batch, int32_t max_total_pages,
                          int32_t max_pages_per_req, int32_t max_budget);

/* Create a context on CUDA device `device` (host int).  `workspace` is device memory of
 * `workspace_bytes` (256-byte aligned), owned by the caller and kept alive until vx_destroy.
 * The max_* values are the ones given to vx_workspace_bytes. */
vx_status vx_create(vx_ctx **out, const vx_geom *g, int device, void *workspace,
                    size_t workspace_bytes, int32_t max_batch, int32_t max_total_pages,
                    int32_t max_pages_per_req, int32_t max_budget);
void vx_destroy(vx_ctx *ctx);

/* Text of the last error on this context (ctx == NULL: last vx_create failure).  Owned by
 * the library; valid until the next call on the same context. */
const char *vx_last_error(const vx_ctx *ctx);

/* Number of kernel launches the last compute call on this context enqueued (host counter). */
int32_t vx_last_launch_count(const vx_ctx *ctx);

/* Context options (host side, persistent until changed).  VX_ERR_INVALID_ARG for an unknown option or value.
 *  VX_OPT_MLA_STEP   how vx_sparse_decode_step schedules the MLA geometry:
 *      VX_MLA_STEP_AUTO     (default) the faster of the two for the batch at hand
 *      VX_MLA_STEP_FUSED    one kernel: a thread-block cluster per request runs score -> select -> decode -> merge
 *                           (falls back to CHAINED when the request / budget sizes exceed what it keeps on chip)
 *      VX_MLA_STEP_CHAINED  three kernels chained by programmatic dependent launch (score, select, decode)
 *      VX_MLA_STEP_FLAT     one persistent kernel for the whole batch: the summary stream cut flat over the SMs, a
 *                           selection warpgroup per request running beside the stream, decode shares taken from a
 *                           counter (falls back to CHAINED for batches / requests beyond what it keeps on chip)
 *    All schedules compute the same selection bit for bit; outputs agree to rounding (different split sizes).
 *  VX_OPT_MLA_FLAT_SPLITS / VX_OPT_MLA_FLAT_WAVES   0 (default) = chosen by the library; > 0 = decode shares per request /
 *                           interleaved waves of the summary stream of the FLAT schedule (tuning knobs) */
enum { VX_OPT_MLA_STEP = 1, VX_OPT_MLA_FLAT_SPLITS = 2, VX_OPT_MLA_FLAT_WAVES = 3 };
enum { VX_MLA_STEP_AUTO = 0, VX_MLA_STEP_FUSED = 1, VX_MLA_STEP_CHAINED = 2, VX_MLA_STEP_FLAT = 3 };
vx_status vx_set_option(vx_ctx *ctx, int32_t option, int32_t value);

/* ---- (a1) summaries: PAPER.md:546 envelope, :89 query-independent, :529 per block ---- */
/* For request i, rebuilds from the K pool the summary of every logical page
 * j >= first_new_pos[i] / page_size (first_new_pos == NULL: only the last page, i.e. the page
 * the newest token fell into; first_new_pos[i] = 0 rebuilds all pages of the request):
 *   summary[p, h, 0, c] = min_t K[p, t, h, c],  summary[p, h, 1, c] = max_t K[p, t, h, c]
 * over the page's VALID tokens (position < seq_lens[i]).  Idempotent.
 * summary: dev [num_pool_pages, Hkv, 2, qk_dim] in the K dtype (min/max are exact).
 * VX_SUMMARY_CENTROID: summary[p, h, c] = mean_t K[p, t, h, c] over the valid tokens, computed exactly and rounded
 * once (nearest even) to the K dtype; summary: dev [num_pool_pages, Hkv, qk_dim]. */
vx_status vx_page_summary_update(vx_ctx *ctx, const vx_kv_pool *pool, const vx_page_table *pt,
                                 const int32_t *first_new_pos /* dev [B] or NULL */,
                                 void *summary, vx_stream stream);

/* ---- (a2) scores: PAPER.md:552, aggregated per KV head (:92) ------------------------- */
/* scores[kvh * total_pages + page_indptr[i] + j] (fp32, ragged layout of PAPER.md:436)
 *   = AGG_{h in group(kvh)} sum_c max(q[i,h,c] * max_c, q[i,h,c] * min_c)  of page j of request i.
 * q: dev [B, Hq, qk_dim].  fp32 accumulation. */
vx_status vx_page_score(vx_ctx *ctx, const void *q, const void *summary, const vx_page_table *pt,
                        float *scores /* dev [Hkv, total_pages] */, vx_stream stream);

/* ---- (a3) selection: PAPER.md:92 Eq.3, :194 radix top-k, :280 forced pages ----------- */
/* Per (request i, KV head kvh), k = budget[i] pages INCLUDING the forced ones:
 * k >= P_i selects every page; otherwise the first n_sink and last n_local logical pages plus
 * the k - #forced best-scoring of the rest (ties: lower logical index).  Exact.
 * sel_phys / sel_logical: dev [B, Hkv, max_budget], entries in ASCENDING logical order,
 * padded with -1; sel_logical may be NULL.  sel_count: dev [B, Hkv] = min(k, P_i).
 * max_budget (host) >= every budget[i].  budget[i] lives on the device and is not validated on the host:
 * a value above max_budget is clamped to it, a negative one selects nothing, and budget[i] < n_sink + n_local
 * breaks the precondition of vx_geom.n_local (the first budget[i] forced pages in logical order are taken, so the
 * newest page may be dropped and vx_sparse_decode_step then leaves its summary as it was). */
vx_status vx_topk_pages(vx_ctx *ctx, const float *scores, const vx_page_table *pt,
                        const int32_t *budget /* dev [B] */, int32_t max_budget,
                        int32_t *sel_phys, int32_t *sel_logical, int32_t *sel_count,
                        vx_stream stream);

/* ---- NEXT-3: approximate radix top-k, PAPER.md:194-196 (stochastic early termination), :538 (`approxTopK`,
 * "tolerate_ratio in [0,1] trades exactness for speed"), :495-509 (judged by recall@k) -----------------------
 * Same inputs / outputs / layout as vx_topk_pages.  The radix select stops refining as soon as the pages still
 * to be taken from the threshold bin number at most floor(tolerate_ratio * k): those are drawn from the bin's
 * members as a cyclic window in page order whose start is SplitMix64(seed, problem = i * Hkv + kvh) >> 32 modulo
 * the member count (every member equally likely; the same seed reproduces the selection bit for bit).  Forced
 * pages and every page above the threshold bin are always taken, so at most floor(tolerate_ratio * k) selected
 * pages differ from the exact set: recall@k >= 1 - tolerate_ratio.  tolerate_ratio = 0 is vx_topk_pages.
 * The paper prints no pseudo-code; the choices made are readings G20-G23 of DESIGN.md section 12.
 * VX_ERR_INVALID_ARG if tolerate_ratio is outside [0, 1]; VX_ERR_UNSUPPORTED if tolerate_ratio > 0 and
 * pt->max_pages_per_req > 49152, or > 8192 with max_budget > 2048 (requests of up to 8,192 pages are selected with their
 * keys in registers, longer ones with their keys in shared memory, which stages at most 2,048 selected pages). */
vx_status vx_topk_pages_approx(vx_ctx *ctx, const float *scores, const vx_page_table *pt,
                               const int32_t *budget /* dev [B] */, int32_t max_budget,
                               float tolerate_ratio, uint64_t seed, int32_t *sel_phys,
                               int32_t *sel_logical, int32_t *sel_count, vx_stream stream);
/* tolerate_ratio and seed used by vx_sparse_decode_step when its flags carry VX_STEP_APPROX_TOPK
 * (context state, host side; default 0 = exact).  VX_ERR_INVALID_ARG outside [0, 1]. */
vx_status vx_set_topk_approx(vx_ctx *ctx, float tolerate_ratio, uint64_t seed);
/* The remap of PAPER.md:495 (App. D.2: "a monotonic transformation x' = f(x) that preserves ordering while reshaping the
 * value distribution ... selected offline through profiling and fused into the histogram pass"; reading G29).
 * knots: HOST array of n_knots floats (2 <= n_knots <= 65), each in [0, 1], never decreasing: f on the score normalised
 * by the request's own min / max, piecewise linear between the knots at 0, 1/(n-1), ..., 1 (copied into the workspace
 * before the call returns; the caller keeps its array).  n_knots = 0 (knots ignored) removes the table.
 * With a table installed, vx_topk_pages_approx and a fused step with VX_STEP_APPROX_TOPK bin the FIRST radix pass through
 * f instead of the linear map; a monotone f changes how many pages share the threshold bin, never which pages an exact
 * selection returns: at tolerate_ratio 0 those calls still return exactly vx_topk_pages' selection (through the
 * approximate kernels' code, so vx_topk_pages_approx's size limits apply).  vx_topk_pages itself never uses the table.
 * paper_2606_06453_b200/remap_profile.py fits a table to sample scores (their empirical distribution function).
 * Synchronous set-up call (one cudaMemcpy); do not call it while a selection of this context is in flight.
 * VX_ERR_INVALID_ARG for a bad count, a NULL table, a value outside [0, 1] or a decreasing pair. */
vx_status vx_set_topk_remap(vx_ctx *ctx, const float *knots /* host */, int32_t n_knots);

/* ---- NEXT-4: head-union block table, PAPER.md:538 (Table 1 "TopK, Union: block-table selection and its
 * deduplicated union (trtllm backend)"), :200 (a paged decode backend that takes one table per request) ------
 * union[i] = the set union over the KV heads of sel_logical[i, kvh, 0:sel_count[i, kvh]], duplicates removed,
 * in ASCENDING logical order; union_phys holds the physical ids through the page table.
 * sel_logical / sel_count: dev, as written by vx_topk_pages (entries outside [0, P_i) are ignored).
 * union_phys / union_logical: dev [B, max_union], padded with -1; union_logical may be NULL.
 * union_count: dev [B].  max_union (host) must be >= min(Hkv * max_budget, pt->max_pages_per_req), the largest
 * union possible, else VX_ERR_INVALID_ARG.  VX_ERR_UNSUPPORTED above 393,184 pages per request. */
vx_status vx_union_pages(vx_ctx *ctx, const vx_page_table *pt, const int32_t *sel_logical,
                         const int32_t *sel_count, int32_t max_budget, int32_t max_union,
                         int32_t *union_phys, int32_t *union_logical, int32_t *union_count,
                         vx_stream stream);

/* ---- (a4)+(a5) attention over the selected pages: PAPER.md:92 Eq.4, :200, :75 -------- */
/* out[i,h,:] = softmax_t(sm_scale * q[i,h].K_t) V_t over the valid tokens of the pages listed
 * in sel_logical/sel_phys[i, h/g, 0:sel_count]; lse[i,h] = natural log of the softmax
 * denominator.  Split-KV partials live in the workspace and are merged by LSE.
 * out: dev [B, Hq, v_dim] in geom.dtype; lse: dev [B, Hq] fp32 (may be NULL). */
vx_status vx_sparse_paged_decode(vx_ctx *ctx, const void *q, const vx_kv_pool *pool,
                                 const vx_page_table *pt, const int32_t *sel_phys,
                                 const int32_t *sel_logical, const int32_t *sel_count,
                                 int32_t max_budget, void *out, float *lse, vx_stream stream);

/* ---- (a6) the fused step: (a1 append rows) -> a2 -> a3 -> a4 -> a5 in one call -------- */
#define VX_STEP_UPDATE_SUMMARY 1u /* flags bit 0: first rebuild the last page's summary of each request */
#define VX_STEP_APPROX_TOPK 2u    /* flags bit 1: select with vx_topk_pages_approx (vx_set_topk_approx's values) */
/* sel_phys / sel_logical / sel_count are optional outputs (NULL = keep them in the workspace). */
vx_status vx_sparse_decode_step(vx_ctx *ctx, const void *q, const vx_kv_pool *pool, void *summary,
                                const vx_page_table *pt, const int32_t *budget, int32_t max_budget,
                                uint32_t flags, void *out, float *lse, int32_t *sel_phys,
                                int32_t *sel_logical, int32_t *sel_count, vx_stream stream);

/* The same step fed from HOST buffers (the serving loop's per-step inputs): copies q, the page
 * table arrays and the budgets host->device into the workspace, runs the fused step, copies
 * out (and lse if not NULL) device->host and synchronises `stream`.  The KV and summary pools
 * are resident device state.  h_* are host pointers (pinned memory recommended). */
vx_status vx_sparse_decode_step_host(vx_ctx *ctx, const void *h_q, const vx_kv_pool *pool,
                                     void *summary, int32_t batch, const int32_t *h_page_indptr,
                                     const int32_t *h_page_indices, const int32_t *h_seq_lens,
                                     const int32_t *h_budget, int32_t max_budget, uint32_t flags,
                                     void *h_out, float *h_lse, vx_stream stream);

/* ---- (a4)+(a5) without a context, a workspace or any allocation ------------------------------------------------
 * vx_sparse_paged_decode_static computes what vx_sparse_paged_decode computes (Eq.4 over the selected pages,
 * :75 split + LSE merge) for callers that cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it.  It takes the geometry by value instead of a context, and its split-KV partials live in a
 * file-scope device array of vx_static_scratch_bytes() = 8 MiB that every GPU loading the library holds until the
 * process exits; the call itself performs no cudaMalloc / cudaFree and calls no allocating routine.  It runs the
 * geometry-agnostic CUDA-core kernels (every geometry vx_create accepts; not the tensor-core paths), on the calling
 * thread's current device, asynchronously on `stream`.
 * Limits and hazards: batch * num_q_heads * 4 (GQA; 1 for MLA) * (v_dim + 1) * 4 bytes must fit the array, else
 * VX_ERR_WORKSPACE (the split count shrinks to fit first); all calls share the array, which keeps the last call's
 * contents (nothing in it needs clearing), so calls that overlap on the GPU -- different streams -- race: serialise them.
 * Arguments as vx_sparse_paged_decode.  Errors: text in vx_static_last_error() (process-wide, not thread-safe). */
vx_status vx_sparse_paged_decode_static(const vx_geom *geom, const void *q, const vx_kv_pool *pool,
                                        const vx_page_table *pt, const int32_t *sel_phys, const int32_t *sel_logical,
                                        const int32_t *sel_count, int32_t max_budget, void *out, float *lse,
                                        vx_stream stream);
size_t vx_static_scratch_bytes(void);
const char *vx_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* VORTEX_B200_H_ */
