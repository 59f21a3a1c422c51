/*
 * vx_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, fp64 CPU statement of the sparse decode hot path of
 * arxiv/paper_2606_06453 ("Vortex"), written from PAPER.md, used to check the
 * CUDA path.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with paper_2606_06453_b200/csrc/ and does not include
 * include/vortex_b200.h.
 *
 * What it computes (notation of SURVEY.md section 8(c); citations are PAPER.md
 * line numbers):
 *   summary   M[j,c] = max_t K[page j, t, c],  m[j,c] = min_t ...   (:546 "feature-wise
 *             key envelope k_j^max, k_j^min"; :89 query-independent; :529 per block)
 *   score     u[h,j] = sum_c max(q[h,c]*M[j,c], q[h,c]*m[j,c])      (:552)
 *             S[kvh,j] = sum_{h in group} u[h,j]  (or max_h)        (:92 group mean; :556 max_h)
 *   top-k     forced first n_sink + last n_local pages (:280), plus arg-top-k of the
 *             remaining pages (:92 Eq. 3), ties -> lower logical index
 *   attention o = softmax(q K_I^T * sm_scale) V_I over the tokens of the selected
 *             pages (:92 Eq. 4), lse = natural log of the softmax denominator
 *   combine   split-softmax merge by log-sum-exp (:75 Flash-Decoding)
 *   block top-k flow: centroid = mean of the block's keys, rounded to the KV dtype
 *             (:92 Eq. 1); score = group sum of q_h . centroid (:92 Eq. 2); pins in tests/test_oracle_centroid.py
 *
 * Every function is the plain definition: no blocking, no fusion, no reordering.
 * All arithmetic is double.  Inputs are read in their storage dtype (bf16 bits or
 * fp32) and widened exactly; fp8 KV pools arrive as the doubles scale * decode(code) (vx_oracle_fp8.py).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closed forms of softmax attention,
 * dense == sparse when the budget covers all pages, split+combine == unsplit,
 * brute-force top-k / subset enumeration on tiny inputs, the upper-bound invariant
 * u[h,j] >= q_h . K_t, summary envelope attained, pool-permutation invariance.
 * The paper prints no worked numeric example for this path, so there are no
 * paper-printed golden values: numeric outputs are pinned by invariants only.
 *
 * Layouts.  K/V pools are addressed with element strides:
 *   elem(page p, token t, head h, channel c) = p*stride_page + t*stride_token + h*stride_head + c
 * Page table is the paper's C = (b, p, I) (:166, :438): page_indptr[batch+1],
 * page_indices[total_pages] physical ids in logical order, seq_lens[batch].
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libvx_oracle.so vx_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define VXO_BF16 0
#define VXO_F32 1
#define VXO_F64 2 /* values that are already doubles: fp8 pools widened and scaled by oracle/vx_oracle_fp8.py (readings G25-G27) */

/* exact widening of one stored element to double */
static double ld_elem(const void *base, int dtype, int64_t idx) {
  if (dtype == VXO_F64) return ((const double *)base)[idx];
  if (dtype == VXO_F32) return (double)((const float *)base)[idx];
  uint32_t bits = ((uint32_t)((const uint16_t *)base)[idx]) << 16;
  float f;
  memcpy(&f, &bits, sizeof f);
  return (double)f;
}

static int num_pages_of(int n_tokens, int page_size) {
  return (n_tokens + page_size - 1) / page_size; /* G3: P = ceil(n / b) */
}

/* number of threads the parallel loops use (reported by bench.py) */
#ifdef _OPENMP
#include <omp.h>
int vxo_num_threads(void) { return omp_get_max_threads(); }
#else
int vxo_num_threads(void) { return 1; }
#endif

/* ------------------------------------------------------------------------- *
 * summary: channel-wise min / max over the VALID tokens of each
 * logical page of each request.  summary[phys, head, 0, c] = min, [.., 1, c] = max.
 * Pages not referenced by the page table are left untouched.
 * first_page[i] (may be NULL = 0): only logical pages >= first_page[i] are rebuilt.
 * ------------------------------------------------------------------------- */
void vxo_page_summary(const void *k, int dtype, int64_t stride_page, int64_t stride_token,
                      int64_t stride_head, int num_kv_heads, int qk_dim, int page_size,
                      int batch, const int32_t *page_indptr, const int32_t *page_indices,
                      const int32_t *seq_lens, const int32_t *first_page, double *summary) {
#pragma omp parallel for schedule(dynamic)
  for (int i = 0; i < batch; ++i) {
    int n = seq_lens[i];
    int P = num_pages_of(n, page_size);
    for (int j = first_page ? first_page[i] : 0; j < P; ++j) {
      int64_t phys = page_indices[page_indptr[i] + j];
      int t_end = n - j * page_size;
      if (t_end > page_size) t_end = page_size;
      for (int h = 0; h < num_kv_heads; ++h) {
        double *mn = summary + ((phys * num_kv_heads + h) * 2 + 0) * (int64_t)qk_dim;
        double *mx = summary + ((phys * num_kv_heads + h) * 2 + 1) * (int64_t)qk_dim;
        for (int c = 0; c < qk_dim; ++c) {
          double lo = INFINITY, hi = -INFINITY;
          for (int t = 0; t < t_end; ++t) {
            double x = ld_elem(k, dtype, phys * stride_page + t * stride_token + h * stride_head + c);
            if (x < lo) lo = x;
            if (x > hi) hi = x;
          }
          mn[c] = lo;
          mx[c] = hi;
        }
      }
    }
  }
}

/* ------------------------------------------------------------------------- *
 * score (PAPER.md:552 per-head envelope; :92 / :119 group sum; :556 group max).
 *   u[h, T0+j] = sum_c max(q[i,h,c]*M[j,c], q[i,h,c]*m[j,c])   T0 = page_indptr[i]
 *   S[kvh, T0+j] = agg_{h in group(kvh)} u[h, T0+j],   agg: 0 = sum, 1 = max
 * Query head h belongs to KV head h / (Hq/Hkv).  Scores carry no softmax scale (G7).
 * u_out may be NULL.
 * ------------------------------------------------------------------------- */
void vxo_page_score(const void *q, int dtype, const double *summary, int num_q_heads,
                    int num_kv_heads, int qk_dim, int batch, const int32_t *page_indptr,
                    const int32_t *page_indices, const int32_t *seq_lens, int page_size, int agg,
                    double *u_out /* [Hq, T] */, double *s_out /* [Hkv, T] */) {
  int g = num_q_heads / num_kv_heads;
  int64_t T = page_indptr[batch];
#pragma omp parallel for schedule(dynamic)
  for (int i = 0; i < batch; ++i) {
    int P = num_pages_of(seq_lens[i], page_size);
    for (int j = 0; j < P; ++j) {
      int64_t col = page_indptr[i] + j;
      int64_t phys = page_indices[col];
      for (int kvh = 0; kvh < num_kv_heads; ++kvh) {
        const double *mn = summary + ((phys * num_kv_heads + kvh) * 2 + 0) * (int64_t)qk_dim;
        const double *mx = summary + ((phys * num_kv_heads + kvh) * 2 + 1) * (int64_t)qk_dim;
        double agg_val = 0.0;
        for (int r = 0; r < g; ++r) {
          int h = kvh * g + r;
          double u = 0.0;
          for (int c = 0; c < qk_dim; ++c) {
            double qc = ld_elem(q, dtype, ((int64_t)i * num_q_heads + h) * qk_dim + c);
            double a = qc * mx[c], b = qc * mn[c];
            u += (a > b) ? a : b;
          }
          if (u_out) u_out[(int64_t)h * T + col] = u;
          if (r == 0) agg_val = u;
          else if (agg == 0) agg_val += u;
          else if (u > agg_val) agg_val = u;
        }
        s_out[(int64_t)kvh * T + col] = agg_val;
      }
    }
  }
}

/* ------------------------------------------------------------------------- *
 * Block top-k flow (section 3.1, the equations around "(2)" at :92):
 *   centroid  kc[j,c] = mean_t K[page j, t, c] over the page's VALID tokens         (Eq. 1)
 *   score     s[j]    = mean_{h in group} q_h . kc[j]                               (Eq. 2)
 * The centroid is stored in the KV dtype: for bf16 pools the exact mean (a sum of at most a few
 * hundred bf16 values is exact in double) is rounded to bf16, round-to-nearest-even, and returned
 * as that bf16 value widened to double.  Scores are returned as the group SUM (ranks like the mean,
 * same convention as the envelope score; reading G2).
 * ------------------------------------------------------------------------- */
static double round_to_storage(double x, int dtype) {
  float f = (float)x;                         /* fp32 storage: one rounding */
  if (dtype == VXO_F32) return (double)f;
  if (dtype == VXO_F64) return x;             /* (fp8 pools have no centroid flow; doubles pass through) */
  /* bf16: round the DOUBLE to 8 significand bits directly (no double rounding through float) */
  if (x == 0.0 || x != x) return x;
  int e;
  double m = frexp(x, &e);                    /* x = m * 2^e, 0.5 <= |m| < 1 */
  double scaled = ldexp(m, 8);                /* 8 significand bits: |scaled| in [128, 256) */
  double r = nearbyint(scaled);               /* default rounding mode: to nearest, ties to even */
  return ldexp(r, e - 8);
}

void vxo_page_centroid(const void *k, int dtype, int64_t stride_page, int64_t stride_token,
                       int64_t stride_head, int num_kv_heads, int qk_dim, int page_size,
                       int batch, const int32_t *page_indptr, const int32_t *page_indices,
                       const int32_t *seq_lens, const int32_t *first_page,
                       double *centroid /* [num_pool_pages, Hkv, d] */) {
#pragma omp parallel for schedule(dynamic)
  for (int i = 0; i < batch; ++i) {
    int n = seq_lens[i];
    int P = num_pages_of(n, page_size);
    for (int j = first_page ? first_page[i] : 0; j < P; ++j) {
      int64_t phys = page_indices[page_indptr[i] + j];
      int t_end = n - j * page_size;
      if (t_end > page_size) t_end = page_size;
      for (int h = 0; h < num_kv_heads; ++h) {
        double *kc = centroid + (phys * num_kv_heads + h) * (int64_t)qk_dim;
        for (int c = 0; c < qk_dim; ++c) {
          double sum = 0.0;
          for (int t = 0; t < t_end; ++t)
            sum += ld_elem(k, dtype, phys * stride_page + t * stride_token + h * stride_head + c);
          kc[c] = round_to_storage(sum / (double)t_end, dtype);
        }
      }
    }
  }
}

void vxo_centroid_score(const void *q, int dtype, const double *centroid, int num_q_heads,
                        int num_kv_heads, int qk_dim, int batch, const int32_t *page_indptr,
                        const int32_t *page_indices, const int32_t *seq_lens, int page_size,
                        double *u_out /* [Hq, T] per-head q_h . kc, may be NULL */,
                        double *s_out /* [Hkv, T] group sum */) {
  int g = num_q_heads / num_kv_heads;
  int64_t T = page_indptr[batch];
#pragma omp parallel for schedule(dynamic)
  for (int i = 0; i < batch; ++i) {
    int P = num_pages_of(seq_lens[i], page_size);
    for (int j = 0; j < P; ++j) {
      int64_t col = page_indptr[i] + j;
      int64_t phys = page_indices[col];
      for (int kvh = 0; kvh < num_kv_heads; ++kvh) {
        const double *kc = centroid + (phys * num_kv_heads + kvh) * (int64_t)qk_dim;
        double total = 0.0;
        for (int r = 0; r < g; ++r) {
          int h = kvh * g + r;
          double u = 0.0;
          for (int c = 0; c < qk_dim; ++c)
            u += ld_elem(q, dtype, ((int64_t)i * num_q_heads + h) * qk_dim + c) * kc[c];
          if (u_out) u_out[(int64_t)h * T + col] = u;
          total += u;
        }
        s_out[(int64_t)kvh * T + col] = total;
      }
    }
  }
}

/* ------------------------------------------------------------------------- *
 * top-k pages (PAPER.md:92 Eq. 3 arg-top-k; :280 forced first / last blocks;
 * readings G4, G5, G6 of SURVEY.md section 8(c)).
 * Per (request i, KV head kvh), P = pages of request i, k = budget[i]:
 *   F = {0..min(n_sink,P)-1} U {max(P-n_local,0)..P-1}
 *   k >= P : all pages;  else  F plus the first max(k-|F|,0) of the pages not in F
 *   sorted by (score descending, logical index ascending).
 * Output in ascending logical order, padded with -1 up to max_budget.
 * thr_out[i,kvh] = score of the last non-forced page taken (NaN if none taken or
 * nothing was left out) -- used by the tests' 1e-3 near-tie rule.
 * Returns 0, or 1 if the precondition |F| <= k failed somewhere.
 * ------------------------------------------------------------------------- */
typedef struct { double s; int32_t j; } vxo_cand;

static int cand_cmp(const void *a, const void *b) {
  const vxo_cand *x = (const vxo_cand *)a, *y = (const vxo_cand *)b;
  if (x->s > y->s) return -1;
  if (x->s < y->s) return 1;
  return (x->j > y->j) - (x->j < y->j);
}

static int int_cmp(const void *a, const void *b) {
  int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
  return (x > y) - (x < y);
}

int vxo_topk_pages(const double *scores /* [Hkv, T] */, int num_kv_heads, int batch,
                   const int32_t *page_indptr, const int32_t *page_indices,
                   const int32_t *seq_lens, int page_size, const int32_t *budget, int n_sink,
                   int n_local, int max_budget, int32_t *sel_logical, int32_t *sel_phys,
                   int32_t *sel_count, double *thr_out) {
  int64_t T = page_indptr[batch];
  int bad = 0;
#pragma omp parallel for schedule(dynamic) reduction(| : bad)
  for (int i = 0; i < batch; ++i) {
    int P = num_pages_of(seq_lens[i], page_size);
    int k = budget[i];
    vxo_cand *cand = (vxo_cand *)malloc(sizeof(vxo_cand) * (size_t)(P > 0 ? P : 1));
    int32_t *chosen = (int32_t *)malloc(sizeof(int32_t) * (size_t)(P > 0 ? P : 1));
    for (int kvh = 0; kvh < num_kv_heads; ++kvh) {
      int64_t o = ((int64_t)i * num_kv_heads + kvh) * max_budget;
      int n_sel = 0, n_cand = 0;
      double thr = NAN;
      if (k >= P) {
        for (int j = 0; j < P; ++j) chosen[n_sel++] = j;
      } else {
        for (int j = 0; j < P; ++j) {
          int forced = (j < n_sink) || (j >= P - n_local);
          if (forced) chosen[n_sel++] = j;
          else { cand[n_cand].s = scores[(int64_t)kvh * T + page_indptr[i] + j]; cand[n_cand].j = j; ++n_cand; }
        }
        if (n_sel > k) bad |= 1;
        int take = k - n_sel;
        if (take < 0) take = 0;
        if (take > n_cand) take = n_cand;
        qsort(cand, (size_t)n_cand, sizeof(vxo_cand), cand_cmp);
        for (int r = 0; r < take; ++r) chosen[n_sel++] = cand[r].j;
        if (take > 0 && take < n_cand) thr = cand[take - 1].s;
        qsort(chosen, (size_t)n_sel, sizeof(int32_t), int_cmp);
      }
      if (n_sel > max_budget) { bad |= 1; n_sel = max_budget; }
      for (int r = 0; r < max_budget; ++r) {
        sel_logical[o + r] = r < n_sel ? chosen[r] : -1;
        sel_phys[o + r] = r < n_sel ? page_indices[page_indptr[i] + chosen[r]] : -1;
      }
      sel_count[(int64_t)i * num_kv_heads + kvh] = n_sel;
      if (thr_out) thr_out[(int64_t)i * num_kv_heads + kvh] = thr;
    }
    free(cand);
    free(chosen);
  }
  return bad;
}

/* ------------------------------------------------------------------------- *
 * attention over a list of logical pages (Eq. 4), one (request, q head):
 *   x_t = sm_scale * sum_c q[c] K_t[c];  mx = max_t x_t;  Z = sum_t exp(x_t - mx)
 *   o = sum_t exp(x_t - mx) V_t / Z;     lse = mx + ln Z
 * over the valid tokens (position < n) of the listed pages, in list order.
 * An empty token set gives o = 0, lse = -inf.
 * ------------------------------------------------------------------------- */
static void attend_pages(const void *q, int q_dtype, int64_t q_off, const void *k, const void *v,
                         int kv_dtype, int64_t stride_page, int64_t stride_token, int64_t head_off,
                         int qk_dim, int v_dim, int page_size, int n_tokens,
                         const int32_t *page_row /* physical ids by logical page */,
                         const int32_t *logical, int n_pages, double sm_scale, double *out,
                         double *lse) {
  int n_tok = 0;
  for (int r = 0; r < n_pages; ++r) {
    int left = n_tokens - logical[r] * page_size;
    n_tok += left > page_size ? page_size : (left > 0 ? left : 0);
  }
  double *x = (double *)malloc(sizeof(double) * (size_t)(n_tok > 0 ? n_tok : 1));
  int64_t *row = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n_tok > 0 ? n_tok : 1));
  int w = 0;
  double mx = -INFINITY;
  for (int r = 0; r < n_pages; ++r) {
    int j = logical[r];
    int64_t phys = page_row[j];
    for (int t = 0; t < page_size && j * page_size + t < n_tokens; ++t) {
      int64_t base = phys * stride_page + t * stride_token + head_off;
      double dot = 0.0;
      for (int c = 0; c < qk_dim; ++c)
        dot += ld_elem(q, q_dtype, q_off + c) * ld_elem(k, kv_dtype, base + c);
      x[w] = sm_scale * dot;
      row[w] = base;
      if (x[w] > mx) mx = x[w];
      ++w;
    }
  }
  for (int c = 0; c < v_dim; ++c) out[c] = 0.0;
  double Z = 0.0;
  for (int t = 0; t < n_tok; ++t) Z += exp(x[t] - mx);
  for (int t = 0; t < n_tok; ++t) {
    double p = exp(x[t] - mx) / Z;
    for (int c = 0; c < v_dim; ++c) out[c] += p * ld_elem(v, kv_dtype, row[t] + c);
  }
  *lse = n_tok > 0 ? mx + log(Z) : -INFINITY;
  free(x);
  free(row);
}

/* sparse attention on a given selection (sel_logical [batch, Hkv, max_budget], first
 * sel_count entries valid).  MLA (kv_shared): pass v = k; V_t = K_t[0:v_dim] (G8). */
void vxo_sparse_attention(const void *q, int q_dtype, const void *k, const void *v, int kv_dtype,
                          int64_t stride_page, int64_t stride_token, int64_t stride_head,
                          int num_q_heads, int num_kv_heads, int qk_dim, int v_dim, int page_size,
                          int batch, const int32_t *page_indptr, const int32_t *page_indices,
                          const int32_t *seq_lens, const int32_t *sel_logical,
                          const int32_t *sel_count, int max_budget, double sm_scale,
                          double *out /* [batch, Hq, v_dim] */, double *lse /* [batch, Hq] */) {
  int g = num_q_heads / num_kv_heads;
#pragma omp parallel for schedule(dynamic) collapse(2)
  for (int i = 0; i < batch; ++i) {
    for (int h = 0; h < num_q_heads; ++h) {
      int kvh = h / g;
      int64_t so = ((int64_t)i * num_kv_heads + kvh) * max_budget;
      attend_pages(q, q_dtype, ((int64_t)i * num_q_heads + h) * qk_dim, k, v, kv_dtype,
                   stride_page, stride_token, kvh * stride_head, qk_dim, v_dim, page_size,
                   seq_lens[i], page_indices + page_indptr[i], sel_logical + so,
                   sel_count[(int64_t)i * num_kv_heads + kvh], sm_scale,
                   out + ((int64_t)i * num_q_heads + h) * v_dim, lse + (int64_t)i * num_q_heads + h);
    }
  }
}

/* dense attention over ALL tokens of every request: the limit case budget >= P
 * (PAPER.md:290 full-attention baseline; :517 skip_layers). */
void vxo_dense_attention(const void *q, int q_dtype, const void *k, const void *v, int kv_dtype,
                         int64_t stride_page, int64_t stride_token, int64_t stride_head,
                         int num_q_heads, int num_kv_heads, int qk_dim, int v_dim, int page_size,
                         int batch, const int32_t *page_indptr, const int32_t *page_indices,
                         const int32_t *seq_lens, double sm_scale, double *out, double *lse) {
  int g = num_q_heads / num_kv_heads;
#pragma omp parallel for schedule(dynamic) collapse(2)
  for (int i = 0; i < batch; ++i) {
    for (int h = 0; h < num_q_heads; ++h) {
      int P = num_pages_of(seq_lens[i], page_size);
      int32_t *all = (int32_t *)malloc(sizeof(int32_t) * (size_t)(P > 0 ? P : 1));
      for (int j = 0; j < P; ++j) all[j] = j;
      attend_pages(q, q_dtype, ((int64_t)i * num_q_heads + h) * qk_dim, k, v, kv_dtype,
                   stride_page, stride_token, (h / g) * stride_head, qk_dim, v_dim, page_size,
                   seq_lens[i], page_indices + page_indptr[i], all, P, sm_scale,
                   out + ((int64_t)i * num_q_heads + h) * v_dim, lse + (int64_t)i * num_q_heads + h);
      free(all);
    }
  }
}

/* combine S partial results by log-sum-exp (PAPER.md:75 Flash-Decoding):
 *   lse = ln sum_s exp(lse_s);  o = sum_s exp(lse_s - lse) o_s.
 * o_part [rows, S, v_dim], lse_part [rows, S]; parts with lse = -inf contribute 0. */
void vxo_combine(const double *o_part, const double *lse_part, int64_t rows, int num_splits,
                 int v_dim, double *out, double *lse) {
  for (int64_t r = 0; r < rows; ++r) {
    double mx = -INFINITY;
    for (int s = 0; s < num_splits; ++s)
      if (lse_part[r * num_splits + s] > mx) mx = lse_part[r * num_splits + s];
    for (int c = 0; c < v_dim; ++c) out[r * v_dim + c] = 0.0;
    if (mx == -INFINITY) { lse[r] = -INFINITY; continue; }
    double Z = 0.0;
    for (int s = 0; s < num_splits; ++s) Z += exp(lse_part[r * num_splits + s] - mx);
    lse[r] = mx + log(Z);
    for (int s = 0; s < num_splits; ++s) {
      double wgt = exp(lse_part[r * num_splits + s] - lse[r]);
      if (wgt == 0.0) continue;
      for (int c = 0; c < v_dim; ++c) out[r * v_dim + c] += wgt * o_part[(r * num_splits + s) * v_dim + c];
    }
  }
}
