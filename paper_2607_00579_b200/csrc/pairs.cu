// Pair-list builder (DESIGN.md row a-P4).  Integer work on the device; results are bit-reproducible.
//   PAPER.md:70  the viewgraph is the set of valid pairs; PAPER.md:478-483 (Alg. 3) batches pairs.
// Canonical order = ascending (target, source), stable w.r.t. the user's order, so that all pairs
// sampling the same target distance field are adjacent in the fused kernel's work list (L2 reuse).
#include "epo_internal.h"

namespace {

__global__ void k_hist(const int32_t* __restrict__ key, int64_t n, int stride, int32_t* __restrict__ cnt) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) atomicAdd(&cnt[key[i * stride]], 1);
}

// single-CTA exclusive scan (n+1 outputs)
__global__ void k_scan_small(const int32_t* __restrict__ in, int32_t* __restrict__ out, int64_t n) {
  __shared__ int32_t warp_sums[32];
  __shared__ int32_t carry_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) carry_s = 0;
  __syncthreads();
  for (int64_t base = 0; base < n; base += blockDim.x) {
    int64_t i = base + tid;
    int32_t v = (i < n) ? in[i] : 0, x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) warp_sums[warp] = x;
    __syncthreads();
    if (warp == 0) {
      int32_t w = (lane < (blockDim.x >> 5)) ? warp_sums[lane] : 0;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { int32_t y = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += y; }
      warp_sums[lane] = w;
    }
    __syncthreads();
    int32_t prefix = carry_s + (warp > 0 ? warp_sums[warp - 1] : 0) + x - v;
    if (i < n) out[i] = prefix;
    __syncthreads();
    if (tid == blockDim.x - 1) carry_s = prefix + v;
    __syncthreads();
  }
  if (tid == 0) out[n] = carry_s;
}

// unordered bucketing of item ids by key (order inside a bucket is fixed by k_rank_*)
__global__ void k_bucket(const int32_t* __restrict__ key, int64_t n, int stride, const int32_t* __restrict__ off,
                         int32_t* __restrict__ cursor, int32_t* __restrict__ bucket) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int k = key[i * stride];
  bucket[off[k] + atomicAdd(&cursor[k], 1)] = (int32_t)i;
}

// canonical position of user pair k inside its target bucket: number of bucket members with a smaller
// (source, user index).  Writes the canonical list and the permutation.
__global__ void k_rank_targets(const int32_t* __restrict__ user, const int32_t* __restrict__ tgt_off,
                               const int32_t* __restrict__ bucket, int64_t P, int2* __restrict__ canon,
                               int32_t* __restrict__ perm) {
  int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= P) return;
  int k = bucket[e];
  int s = user[2 * (int64_t)k], t = user[2 * (int64_t)k + 1];
  int lo = tgt_off[t], hi = tgt_off[t + 1], rank = 0;
  for (int j = lo; j < hi; ++j) {
    int k2 = bucket[j];
    int s2 = user[2 * (int64_t)k2];
    rank += (s2 < s) || (s2 == s && k2 < k);
  }
  canon[lo + rank] = make_int2(s, t);
  perm[lo + rank] = k;
}

// per-source incidence lists of canonical ids, ascending
__global__ void k_rank_sources(const int2* __restrict__ canon, const int32_t* __restrict__ src_off,
                               const int32_t* __restrict__ bucket, int64_t P, int32_t* __restrict__ inc) {
  int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= P) return;
  int p = bucket[e];
  int s = canon[p].x;
  int lo = src_off[s], hi = src_off[s + 1], rank = 0;
  for (int j = lo; j < hi; ++j) rank += bucket[j] < p;
  inc[lo + rank] = p;
}

__global__ void k_chunk_counts(const int2* __restrict__ canon, const int32_t* __restrict__ edge_off, int64_t P,
                               int chunk, int32_t* __restrict__ cnt) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  int s = canon[p].x;
  int n = edge_off[s + 1] - edge_off[s];
  cnt[p] = (n + chunk - 1) / chunk;
}

// work item = {source, target, first point of the chunk (absolute index into the point list), samples of the
// source's list from there on}: the fused kernel needs no other table before it can start loading points
__global__ void k_fill_work(const int32_t* __restrict__ work_off, const int2* __restrict__ canon,
                            const int32_t* __restrict__ edge_off, int64_t P, int chunk, int4* __restrict__ work) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const int2 st = canon[p];
  const int e0 = edge_off[st.x], n = edge_off[st.x + 1] - e0;
  int lo = work_off[p], hi = work_off[p + 1];
  for (int w = lo; w < hi; ++w) work[w] = make_int4(st.x, st.y, e0 + (w - lo) * chunk, n - (w - lo) * chunk);
}

}  // namespace

epo_status epo_build_pairs(epo_ctx* ctx, const int32_t* d_user, int64_t P, int2** out_pairs, int32_t** out_perm,
                           int32_t** out_tgt_off, int32_t** out_src_off, int32_t** out_src_inc, int4** out_work,
                           int32_t** out_work_off, int64_t* out_n_work, int chunk) {
  const int N = ctx->N;
  cudaStream_t st = ctx->stream;
  int2* canon = nullptr;
  int4* work = nullptr;
  int32_t *perm = nullptr, *tgt_off = nullptr, *src_off = nullptr, *src_inc = nullptr;
  int32_t *cnt = nullptr, *cursor = nullptr, *bucket = nullptr, *chunk_cnt = nullptr, *work_off = nullptr;
  auto free_all = [&]() {
    cudaFree(canon); cudaFree(work); cudaFree(perm); cudaFree(tgt_off); cudaFree(src_off); cudaFree(src_inc); cudaFree(work_off);
  };
  auto free_tmp = [&]() { cudaFree(cnt); cudaFree(cursor); cudaFree(bucket); cudaFree(chunk_cnt); };
#define PR_CUDA(call)                                                                                \
  do {                                                                                               \
    cudaError_t e_ = (call);                                                                         \
    if (e_ != cudaSuccess) {                                                                         \
      epo_status rc_ = epo_fail(ctx, e_ == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, \
                                "%s failed: %s", #call, cudaGetErrorString(e_));                     \
      free_all(); free_tmp();                                                                        \
      return rc_;                                                                                    \
    }                                                                                                \
  } while (0)
  PR_CUDA(cudaMalloc(&canon, P * sizeof(int2)));
  PR_CUDA(cudaMalloc(&perm, P * sizeof(int32_t)));
  PR_CUDA(cudaMalloc(&tgt_off, (N + 1) * sizeof(int32_t)));
  PR_CUDA(cudaMalloc(&src_off, (N + 1) * sizeof(int32_t)));
  PR_CUDA(cudaMalloc(&src_inc, P * sizeof(int32_t)));
  PR_CUDA(cudaMalloc(&cnt, (N + 1) * sizeof(int32_t)));
  PR_CUDA(cudaMalloc(&cursor, (N + 1) * sizeof(int32_t)));
  PR_CUDA(cudaMalloc(&bucket, P * sizeof(int32_t)));
  PR_CUDA(cudaMalloc(&chunk_cnt, (P + 1) * sizeof(int32_t)));
  PR_CUDA(cudaMalloc(&work_off, (P + 1) * sizeof(int32_t)));
  const int gridP = (int)((P + 255) / 256);
  // by target
  PR_CUDA(cudaMemsetAsync(cnt, 0, (N + 1) * sizeof(int32_t), st));
  PR_CUDA(cudaMemsetAsync(cursor, 0, (N + 1) * sizeof(int32_t), st));
  k_hist<<<gridP, 256, 0, st>>>(d_user + 1, P, 2, cnt);
  k_scan_small<<<1, 1024, 0, st>>>(cnt, tgt_off, N);
  k_bucket<<<gridP, 256, 0, st>>>(d_user + 1, P, 2, tgt_off, cursor, bucket);
  k_rank_targets<<<gridP, 256, 0, st>>>(d_user, tgt_off, bucket, P, canon, perm);
  // by source, over canonical ids
  PR_CUDA(cudaMemsetAsync(cnt, 0, (N + 1) * sizeof(int32_t), st));
  PR_CUDA(cudaMemsetAsync(cursor, 0, (N + 1) * sizeof(int32_t), st));
  k_hist<<<gridP, 256, 0, st>>>(reinterpret_cast<const int32_t*>(canon), P, 2, cnt);
  k_scan_small<<<1, 1024, 0, st>>>(cnt, src_off, N);
  k_bucket<<<gridP, 256, 0, st>>>(reinterpret_cast<const int32_t*>(canon), P, 2, src_off, cursor, bucket);
  k_rank_sources<<<gridP, 256, 0, st>>>(canon, src_off, bucket, P, src_inc);
  // work list of the fused kernel: (pair, first edge of the chunk), target-major
  k_chunk_counts<<<gridP, 256, 0, st>>>(canon, ctx->d_edge_off, P, chunk, chunk_cnt);
  k_scan_small<<<1, 1024, 0, st>>>(chunk_cnt, work_off, P);
  ctx->launches += 10;
  int32_t n_work = 0;
  PR_CUDA(cudaMemcpyAsync(&n_work, work_off + P, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  PR_CUDA(cudaStreamSynchronize(st));
  PR_CUDA(cudaMalloc(&work, (size_t)(n_work > 0 ? n_work : 1) * sizeof(int4)));
  k_fill_work<<<gridP, 256, 0, st>>>(work_off, canon, ctx->d_edge_off, P, chunk, work);
  ctx->launches += 1;
  PR_CUDA(cudaGetLastError());
  PR_CUDA(cudaStreamSynchronize(st));
  free_tmp();
#undef PR_CUDA
  *out_pairs = canon; *out_perm = perm; *out_tgt_off = tgt_off; *out_src_off = src_off; *out_src_inc = src_inc;
  *out_work = work; *out_work_off = work_off; *out_n_work = n_work;
  return EPO_OK;
}
