// vx_union.cu -- NEXT-4: the deduplicated union of a request's per-KV-head selections (Table 1,
// "TopK, Union: block-table selection and its deduplicated union (trtllm backend)"; :200 the sparse block table
// handed to a paged decode backend that takes ONE table per request).
//
// One CTA per request.  The selected logical page ids of all KV heads set bits of a shared-memory bitmap over the
// request's pages (atomicOr: duplicates collapse); the bitmap is then emitted in ascending logical order -- every
// thread owns a contiguous run of words, a block-wide exclusive scan of the runs' popcounts gives its first
// output position -- with the physical id gathered from the page table.  Integer work on a few KB per request.
#include "vx_common.cuh"
#include "vx_internal.h"

namespace vx {

constexpr int kUnionThreads = 256;

__global__ void __launch_bounds__(kUnionThreads)
union_kernel(int num_kv_heads, const int32_t* __restrict__ page_indptr, const int32_t* __restrict__ page_indices,
             const int32_t* __restrict__ seq_lens, int page_size, const int32_t* __restrict__ sel_logical,
             const int32_t* __restrict__ sel_count, int max_budget, int max_union, int32_t* __restrict__ union_phys,
             int32_t* __restrict__ union_logical, int32_t* __restrict__ union_count) {
  constexpr int WARPS = kUnionThreads / kWarp;
  extern __shared__ uint32_t s_bits[];
  __shared__ int s_wsum[WARPS];
  const int i = blockIdx.x, tid = threadIdx.x, lane = tid % kWarp, warp = tid / kWarp;
  const int n_pages = (seq_lens[i] + page_size - 1) / page_size;
  const int words = (n_pages + 31) / 32;
  const int row0 = page_indptr[i];
  for (int w = tid; w < words; w += kUnionThreads) s_bits[w] = 0u;
  __syncthreads();
  for (int idx = tid; idx < num_kv_heads * max_budget; idx += kUnionThreads) {
    const int h = idx / max_budget, r = idx - h * max_budget;
    if (r < sel_count[i * num_kv_heads + h]) {
      const int j = sel_logical[((int64_t)i * num_kv_heads + h) * max_budget + r];
      if (j >= 0 && j < n_pages) atomicOr(&s_bits[j >> 5], 1u << (j & 31));
    }
  }
  __syncthreads();
  // my run of words, its popcount, and the exclusive prefix over the block
  const int per = (words + kUnionThreads - 1) / kUnionThreads;
  const int w0 = min(tid * per, words), w1 = min(w0 + per, words);
  int mine = 0;
  for (int w = w0; w < w1; ++w) mine += __popc(s_bits[w]);
  int inc = mine;
#pragma unroll
  for (int o = 1; o < kWarp; o <<= 1) {
    const int a = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += a;
  }
  if (lane == kWarp - 1) s_wsum[warp] = inc;
  __syncthreads();
  int pos = inc - mine, total = 0;
#pragma unroll
  for (int w = 0; w < WARPS; ++w) {
    pos += (w < warp) ? s_wsum[w] : 0;
    total += s_wsum[w];
  }
  const int64_t out0 = (int64_t)i * max_union;
  for (int w = w0; w < w1; ++w) {
    uint32_t bits = s_bits[w];
    while (bits) {
      const int j = w * 32 + __ffs(bits) - 1;
      bits &= bits - 1;
      if (pos < max_union) {
        union_phys[out0 + pos] = page_indices[row0 + j];
        if (union_logical) union_logical[out0 + pos] = j;
      }
      ++pos;
    }
  }
  const int n_out = min(total, max_union);
  if (tid == 0) union_count[i] = n_out;
  for (int r = n_out + tid; r < max_union; r += kUnionThreads) {
    union_phys[out0 + r] = -1;
    if (union_logical) union_logical[out0 + r] = -1;
  }
}

cudaError_t launch_union_pages(vx_ctx* c, const vx_page_table& pt, const int32_t* sel_logical, const int32_t* sel_count,
                               int32_t max_budget, int32_t max_union, int32_t* union_phys, int32_t* union_logical,
                               int32_t* union_count, cudaStream_t s) {
  if (pt.batch == 0) return cudaSuccess;
  const size_t smem = (size_t)((pt.max_pages_per_req + 31) / 32 + 1) * sizeof(uint32_t);
  if (smem > 48 * 1024) return cudaErrorNotSupported;             // > 393,184 pages per request
  cudaError_t e = launch_kernel(union_kernel, dim3(pt.batch), dim3(kUnionThreads), smem, s, false, c->g.num_kv_heads,
                                pt.page_indptr, pt.page_indices, pt.seq_lens, c->g.page_size, sel_logical, sel_count,
                                max_budget, max_union, union_phys, union_logical, union_count);
  c->launches += 1;
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace vx
