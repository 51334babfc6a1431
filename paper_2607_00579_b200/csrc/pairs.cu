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

// work item = {source | target << 16, canonical pair index, first slot of the chunk in the packed point array
// (absolute, a multiple of kLgThreads: EpoPacked), samples of the source's list from there on}: the fused kernel needs no other table before it can start
// loading points (N <= 65535 is checked in epo_create)
__global__ void k_fill_work(const int32_t* __restrict__ work_off, const int2* __restrict__ canon,
                            const int32_t* __restrict__ edge_off, const int32_t* __restrict__ pk_off, int64_t P, int chunk,
                            int4* __restrict__ work) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const int2 st = canon[p];
  const int n = edge_off[st.x + 1] - edge_off[st.x];
  const int e0 = pk_off[st.x] / 2;                   // slots of the packed point array (EpoPacked)
  int lo = work_off[p], hi = work_off[p + 1];
  for (int w = lo; w < hi; ++w) work[w] = make_int4(st.x | (st.y << 16), (int)p, e0 + (w - lo) * (chunk / 2), n - (w - lo) * chunk);
}

// ---------------------------------------------------------------------------------------------------------
// Stochastic viewgraph sub-sampling (Alg. 3 l.3-6): every iteration evaluates a
// fresh uniform random subset S of the pair list, |S| = M.  The draw is a pure function of (seed, step, pair):
// pair p (position in the caller's list) gets key(step, p) = output number step * 2^32 + p + 1 of
// SplitMix64(seed), and S = the M pairs with the smallest (key, p) (include/epo.h).  One launch per iteration, no
// host involvement.  CTA g owns the canonical pairs [g C, (g + 1) C), C = 4096; the CTAs are all resident (at most
// kSelMaxCtas of them, one per SM) and meet at three grid barriers:
//   A  histogram of the keys' leading 11 bits (shared, then global)                              -- barrier 1
//   B  every CTA scans the 2048 bins for the one that holds the M-th smallest key and appends its own members of
//      that bin (P / 2048 expected) to a global candidate list                                     -- barrier 2
//   C  every CTA ranks the candidates by (key, p) and so knows the M-th smallest pair T
//   D  flags of its own pairs ((key, p) <= T), block scan of (selected, their work items)         -- barrier 3
//      then, with the totals of the CTAs before it, its part of the iteration's ordered work list.
// The last CTA out re-zeroes the histogram and the counters for the next launch.
// ---------------------------------------------------------------------------------------------------------
constexpr int kSelUnroll = 4;
constexpr int kSelThreads = 1024, kSelBits = 11, kSelBins = 1 << kSelBits;
constexpr int kSelChunk = kSelUnroll * kSelThreads;       // pairs per CTA
constexpr int kSelStage = 1024;                           // candidates ranked from shared memory

__device__ __forceinline__ unsigned long long subset_key(unsigned long long seed, int step, int p) {
  unsigned long long z = seed + 0x9E3779B97F4A7C15ull * (((unsigned long long)(unsigned)step << 32) + (unsigned long long)p + 1ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// inclusive scan of an int2 over the CTA (kSelThreads threads); *total gets the CTA sum
__device__ int2 block_scan2(int2 v, int2* warp_tot /* [32] shared */, int2* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int a = __shfl_up_sync(0xffffffffu, v.x, o), b = __shfl_up_sync(0xffffffffu, v.y, o);
    if (lane >= o) { v.x += a; v.y += b; }
  }
  __syncthreads();                                  // warp_tot may still be read from the previous call
  if (lane == 31) warp_tot[warp] = v;
  __syncthreads();
  if (warp == 0) {
    int2 w = warp_tot[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int a = __shfl_up_sync(0xffffffffu, w.x, o), b = __shfl_up_sync(0xffffffffu, w.y, o);
      if (lane >= o) { w.x += a; w.y += b; }
    }
    warp_tot[lane] = w;
  }
  __syncthreads();
  if (warp > 0) { v.x += warp_tot[warp - 1].x; v.y += warp_tot[warp - 1].y; }
  *total = warp_tot[31];
  return v;
}

// all CTAs of the grid are resident (the launcher guarantees gridDim.x <= number of SMs): arrive, then spin
__device__ __forceinline__ void grid_barrier(int* counter, int target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(counter, 1);
    while (atomicAdd(counter, 0) < target) __nanosleep(64);
    __threadfence();
  }
  __syncthreads();
}

struct SelParams {
  const int32_t* __restrict__ perm;       // canonical -> caller's pair index
  const int32_t* __restrict__ work_off;   // [P+1] static work items of each canonical pair
  const DevState* state;
  uint8_t* flag;             // [P] canonical order: 1 = in this iteration's subset
  int32_t* sel_work;         // [n_work] static work-item indices of the subset, in order (nullptr: flags only)
  int32_t* info;             // {work items of the subset, pairs of the subset}
  int32_t* scratch;          // EpoSelScratch, zero between launches
  unsigned long long seed;
  int P, M, step_override /* < 0: the device step counter */, gated;
};

__global__ void __launch_bounds__(kSelThreads, 1) k_select_pairs(const SelParams p) {
  __shared__ int hist[kSelBins];
  __shared__ unsigned long long skey[kSelStage];
  __shared__ int sidx[kSelStage];
  __shared__ int2 wtot[32];
  __shared__ int s_bin, s_below;
  __shared__ unsigned long long s_tkey;
  __shared__ int s_tidx, s_last;
  const int tid = threadIdx.x, G = (int)gridDim.x, g = (int)blockIdx.x;
  int* bar = p.scratch + kSelScrBarrier;
  int* ghist = p.scratch + kSelScrHist;
  int* ncand = p.scratch + kSelScrNCand;
  int2* tots = reinterpret_cast<int2*>(p.scratch + kSelScrTotals);
  unsigned long long* ckey = reinterpret_cast<unsigned long long*>(p.scratch + kSelScrCandKey);
  int* cidx = p.scratch + kSelScrCandIdx;
  // this thread's pairs: static loads before the grid-dependency wait
  int u[kSelUnroll], wo[kSelUnroll + 1];
  const int q0 = g * kSelChunk + kSelUnroll * tid;
#pragma unroll
  for (int i = 0; i < kSelUnroll; ++i) {
    u[i] = q0 + i < p.P ? __ldg(p.perm + q0 + i) : -1;
    wo[i] = q0 + i <= p.P ? __ldg(p.work_off + q0 + i) : 0;
  }
  wo[kSelUnroll] = q0 + kSelUnroll <= p.P ? __ldg(p.work_off + q0 + kSelUnroll) : 0;
  for (int i = tid; i < kSelBins; i += kSelThreads) hist[i] = 0;
  cudaTriggerProgrammaticLaunchCompletion();
  cudaGridDependencySynchronize();
  if (p.gated && (p.gated == 2 ? p.state->stopped : p.state->halt)) return;
  const int step = p.step_override >= 0 ? p.step_override : p.state->step;
  unsigned long long key[kSelUnroll];
#pragma unroll
  for (int i = 0; i < kSelUnroll; ++i) key[i] = u[i] >= 0 ? subset_key(p.seed, step, u[i]) : ~0ull;
  // ---- A: histogram of the leading bits
  __syncthreads();
#pragma unroll
  for (int i = 0; i < kSelUnroll; ++i)
    if (u[i] >= 0) atomicAdd(&hist[(int)(key[i] >> (64 - kSelBits))], 1);
  __syncthreads();
  for (int i = tid; i < kSelBins; i += kSelThreads)
    if (hist[i]) atomicAdd(&ghist[i], hist[i]);
  grid_barrier(bar, G);
  // ---- B: the bin of the M-th smallest key (two bins per thread), then this CTA's members of it
  {
    const int h0 = __ldcg(ghist + 2 * tid), h1 = __ldcg(ghist + 2 * tid + 1);
    int2 tot;
    const int2 inc = block_scan2(make_int2(h0 + h1, 0), wtot, &tot);
    const int before = inc.x - h0 - h1;
    if (before < p.M && p.M <= before + h0) { s_bin = 2 * tid; s_below = before; }
    else if (before + h0 < p.M && p.M <= before + h0 + h1) { s_bin = 2 * tid + 1; s_below = before + h0; }
    __syncthreads();
  }
  const int bin = s_bin, k = p.M - s_below;          // rank wanted inside the bin, 1-based
#pragma unroll
  for (int i = 0; i < kSelUnroll; ++i)
    if (u[i] >= 0 && (int)(key[i] >> (64 - kSelBits)) == bin) {
      const int pos = atomicAdd(ncand, 1);
      if (pos < kSelCandCap) { ckey[pos] = key[i]; cidx[pos] = u[i]; }
    }
  grid_barrier(bar, 2 * G);
  // ---- C: the candidate of rank k by (key, caller's index)
  {
    int n = __ldcg(ncand);
    n = n < kSelCandCap ? n : kSelCandCap;           // more only if P > 2048 * kSelCandCap / 4 (refused by the host)
    const bool staged = n <= kSelStage;               // the usual case: rank from shared memory
    if (staged) {
      for (int i = tid; i < n; i += kSelThreads) { skey[i] = __ldcg(ckey + i); sidx[i] = __ldcg(cidx + i); }
      __syncthreads();
    }
    for (int i = tid; i < n; i += kSelThreads) {
      const unsigned long long ki = staged ? skey[i] : __ldcg(ckey + i); const int ui = staged ? sidx[i] : __ldcg(cidx + i);
      int r = 0;
      if (staged) for (int j = 0; j < n; ++j) r += (skey[j] < ki) || (skey[j] == ki && sidx[j] < ui);
      else for (int j = 0; j < n; ++j) { const unsigned long long kj = __ldcg(ckey + j); r += (kj < ki) || (kj == ki && __ldcg(cidx + j) < ui); }
      if (r == k - 1) { s_tkey = ki; s_tidx = ui; }
    }
    __syncthreads();
  }
  const unsigned long long tkey = s_tkey; const int tidx = s_tidx;
  // ---- D: flags, counts, ordered work list
  int f[kSelUnroll], nw[kSelUnroll], fs = 0, ws = 0;
#pragma unroll
  for (int i = 0; i < kSelUnroll; ++i) {
    f[i] = 0; nw[i] = 0;
    if (u[i] >= 0) {
      f[i] = (key[i] < tkey) || (key[i] == tkey && u[i] <= tidx);
      p.flag[q0 + i] = (uint8_t)f[i];
      if (f[i]) nw[i] = wo[i + 1] - wo[i];
    }
    fs += f[i]; ws += nw[i];
  }
  int2 tot;
  const int2 inc = block_scan2(make_int2(fs, ws), wtot, &tot);
  if (tid == 0) { tots[g] = tot; }
  grid_barrier(bar, 3 * G);
  int2 carry = make_int2(0, 0);
  for (int j = 0; j < g; ++j) { const int2 t = __ldcg(tots + j); carry.x += t.x; carry.y += t.y; }
  if (p.sel_work) {
    int off = carry.y + inc.y - ws;
#pragma unroll
    for (int i = 0; i < kSelUnroll; ++i) {
      for (int w = 0; w < nw[i]; ++w) p.sel_work[off + w] = wo[i] + w;
      off += nw[i];
    }
  }
  if (g == G - 1 && tid == 0) { p.info[0] = carry.y + tot.y; p.info[1] = carry.x + tot.x; }
  // ---- the last CTA out cleans up for the next launch
  __syncthreads();
  if (tid == 0) s_last = atomicAdd(bar + 1, 1) == G - 1;
  __syncthreads();
  if (s_last) {
    for (int i = tid; i < kSelBins; i += kSelThreads) ghist[i] = 0;
    if (tid == 0) { *ncand = 0; bar[0] = 0; bar[1] = 0; }
  }
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
    epo_dfree(ctx, canon); epo_dfree(ctx, work); epo_dfree(ctx, perm); epo_dfree(ctx, tgt_off); epo_dfree(ctx, src_off); epo_dfree(ctx, src_inc); epo_dfree(ctx, work_off);
  };
  auto free_tmp = [&]() { epo_dfree(ctx, cnt); epo_dfree(ctx, cursor); epo_dfree(ctx, bucket); epo_dfree(ctx, chunk_cnt); };
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
  PR_CUDA(epo_dmalloc(ctx, &canon, P * sizeof(int2)));
  PR_CUDA(epo_dmalloc(ctx, &perm, P * sizeof(int32_t)));
  PR_CUDA(epo_dmalloc(ctx, &tgt_off, (N + 1) * sizeof(int32_t)));
  PR_CUDA(epo_dmalloc(ctx, &src_off, (N + 1) * sizeof(int32_t)));
  PR_CUDA(epo_dmalloc(ctx, &src_inc, P * sizeof(int32_t)));
  PR_CUDA(epo_dmalloc(ctx, &cnt, (N + 1) * sizeof(int32_t)));
  PR_CUDA(epo_dmalloc(ctx, &cursor, (N + 1) * sizeof(int32_t)));
  PR_CUDA(epo_dmalloc(ctx, &bucket, P * sizeof(int32_t)));
  PR_CUDA(epo_dmalloc(ctx, &chunk_cnt, (P + 1) * sizeof(int32_t)));
  PR_CUDA(epo_dmalloc(ctx, &work_off, (P + 1) * sizeof(int32_t)));
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
  PR_CUDA(epo_dmalloc(ctx, &work, (size_t)(n_work > 0 ? n_work : 1) * sizeof(int4)));
  k_fill_work<<<gridP, 256, 0, st>>>(work_off, canon, ctx->d_edge_off, ctx->packed.d_off, P, chunk, work);
  ctx->launches += 1;
  PR_CUDA(cudaGetLastError());
  free_tmp();
#undef PR_CUDA
  *out_pairs = canon; *out_perm = perm; *out_tgt_off = tgt_off; *out_src_off = src_off; *out_src_inc = src_inc;
  *out_work = work; *out_work_off = work_off; *out_n_work = n_work;
  return EPO_OK;
}

epo_status epo_launch_select_pairs(epo_ctx* ctx, int step_override, bool gated, bool build_work) {
  SelParams p;
  p.perm = ctx->d_perm; p.work_off = ctx->d_work_off; p.state = ctx->d_state; p.flag = ctx->d_sel_flag;
  p.sel_work = build_work ? ctx->d_sel_work : nullptr; p.info = ctx->d_sel_info; p.scratch = ctx->d_sel_scratch;
  p.seed = ctx->cfg.subsample_seed;
  p.P = (int)ctx->P; p.M = ctx->cfg.pair_budget; p.step_override = step_override; p.gated = gated ? (ctx->first_budget > 0 ? 2 : 1) : 0;
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)((ctx->P + kSelChunk - 1) / kSelChunk));   // <= kSelMaxCtas, checked in epo_set_pairs
  lc.blockDim = dim3(kSelThreads); lc.dynamicSmemBytes = 0; lc.stream = ctx->stream;
  cudaLaunchAttribute at[2];
  int na = 0;
  // programmatic dependent launch only inside the loop and only when the static lists are not the work of the
  // kernels just before this one (the same rule as for the fused kernel)
  if (ctx->pdl && gated && !ctx->static_dirty) {
    at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[na].val.programmaticStreamSerializationAllowed = 1; ++na;
  }
  // more than one CTA: they meet at grid_barrier, so the launch is a COOPERATIVE one -- the runtime then checks that the
  // whole grid can be resident at once (cudaErrorCooperativeLaunchTooLarge otherwise) instead of this code assuming it
  if (lc.gridDim.x > 1 && ctx->coop_select) { at[na].id = cudaLaunchAttributeCooperative; at[na].val.cooperative = 1; ++na; }
  lc.attrs = at; lc.numAttrs = na;
  EPO_CUDA(ctx, cudaLaunchKernelEx(&lc, k_select_pairs, p));
  ctx->launches += 1;
  return EPO_OK;
}

int64_t epo_select_max_pairs(void) { return (int64_t)kSelMaxCtas * kSelChunk; }
