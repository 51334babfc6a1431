// Internal declarations of the EPO CUDA library (not part of the C ABI; see include/epo.h).
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <vector>

#include "epo.h"

// One compacted edge pixel: (u | v << 16, Z).  8 bytes, loaded with one LDG.64 (row a-P1 of DESIGN.md).
struct __align__(8) EdgeRec {
  uint32_t uv;
  float z;
};

// Partial sums written by each CTA of the fused kernel (row a-8): S = sum rho, n = valid count,
// A = sum a, M = sum x_t x a (six-accumulator identity I1).  fp64, 64 bytes per work item.
constexpr int kAccStride = 8;
// Joint phase: the record also carries the pair's focal-length sums (slot 8: sum d rho / d ln f_t, slot 9: sum
// d rho / d ln f_s); 16 slots so that k_finish reads it with two chunk classes per warp round.
constexpr int kAccStrideJoint = 16;

// Edge pixels handled by one CTA of the fused kernel: kLgOuter passes of kLgThreads threads x kLgPerThread
// (unrolled) samples.  The point list is padded by kLgChunk entries so that tail lanes may read past a list.
#ifndef EPO_LG_THREADS
#define EPO_LG_THREADS 128
#endif
#ifndef EPO_LG_PER_THREAD
#define EPO_LG_PER_THREAD 2
#endif
#ifndef EPO_LG_OUTER
#define EPO_LG_OUTER 16
#endif
#ifndef EPO_LG_MINBLOCKS
#define EPO_LG_MINBLOCKS 7
#endif
constexpr int kLgThreads = EPO_LG_THREADS;
constexpr int kLgPerThread = EPO_LG_PER_THREAD;
constexpr int kLgOuter = EPO_LG_OUTER;        // most passes per work item (epo_ctx::lg_chunk is what runs)
constexpr int kLgPass = kLgThreads * kLgPerThread;     // samples of one pass of a CTA
constexpr int kLgMaxOuter = 32;
constexpr int kLgPad = kLgPass * kLgMaxOuter;  // zero points appended to the list: tail lanes / prefetches read past a list

// Device-resident control block of the optimisation loop (rows a-10..a-12): lets epo_step enqueue
// n iterations without any host synchronisation; every kernel of an iteration checks `halt`.
struct DevState {
  int32_t step;        // optimiser step counter s (0-based index of the NEXT update)
  int32_t phase;       // 0, 1, 2 (Alg. 2 l.13-17)
  int32_t stopped;     // step >= max_steps, or early_stop && phase == 2
  int32_t iters_done;  // iterations executed since the last epo_step began
  int32_t phase_prev;  // joint loop: phase at the START of the iteration k_finish has just completed
  int32_t joint_pending;   // joint loop: an iteration has completed and its joint pass / variable update are due
  int32_t phase1_step; // joint loop: iteration index at which phase 0 -> 1 happened (depth steps from the next one)
  int32_t ticket;      // CTAs of k_finish that have finished (the last one runs the serial tail and re-zeroes it)
  int32_t budget;      // iterations the epo_step call in flight may still run at most (set by k_begin_step_call)
  int32_t halt;        // stopped || iters_done >= budget: what the kernels of an iteration test
  int32_t graph_limit; // the loop graph runs its body again while !stopped && iters_done < graph_limit (the largest
                       // multiple of its unroll factor within the budget; the host enqueues the remainder)
  double loss;         // loss of the last evaluation
};

// All distance fields in block-linear, gather-enabled 2-D CUDA arrays, views tiled in a grid: view i sits at
// texel offset ((i % cols) W, (i / cols) H).
//   arr / tex    the field itself, fp32 (or fp16 when dtf_format = 1): what epo_get_dtf returns
//   arr8 / tex8  (fp32 format only) the exact integer SQUARED distance, saturated at 255, one byte per texel.
//                The fused kernel samples this one whenever lambda <= kU8LambdaMax and takes the correctly rounded
//                square root from a 256-entry table: the same fp32 tap values from a quarter of the bytes.  A
//                saturated tap (distance >= sqrt(255) = 15.97) can only occur in a footprint whose four taps all
//                exceed 15.97 - sqrt(2) = 14.55 (the exact EDT is 1-Lipschitz), where d > lambda clamps the sample to
//                rho = H(lambda), rho' = 0 whatever the taps are.
struct EpoAtlas {
  cudaArray_t arr, arr8;
  cudaTextureObject_t tex, tex8;
  int cols;
};
constexpr float kU8LambdaMax = 14.5f;

// The camera-frame points as the packed fused kernel reads them.  "Slot" j holds two samples; view i owns the slots
// [off[i] / 2, off[i+1] / 2), off[i+1] - off[i] = its edge count rounded up to a multiple of kLgPass (padding = zero
// points, never counted), and inside a view slot j = 32 g + l holds the samples 64 g + l and 64 g + 32 + l of the
// tile-major list: a warp's load is one contiguous 256-byte row and each of its two gathers covers 32 CONSECUTIVE
// points.  The three coordinates of a block of kLgThreads slots are stored as three consecutive planes,
//   float2 index of (slot j, coordinate c) = (j / kLgThreads) * 3 * kLgThreads + c * kLgThreads + j % kLgThreads,
// so that a CTA's pass is three loads at immediate offsets from ONE running pointer.  kLgPad / 2 zero slots follow the
// last view (the first-pass loads of a short last work item read past its list).
struct EpoPacked {
  float2* xyz;
  int2* pix;                    // [slots] pixel index v W + u of both samples of a slot (-1: padding)
  int32_t* d_off;               // [N+1] device copy of h_off
  std::vector<int32_t> h_off;   // [N+1] in samples, multiples of kLgPass
};

struct epo_ctx {
  epo_config cfg;
  cudaStream_t stream;
  cudaStream_t copy_stream;   // epo_set_views: the depth maps arrive on it while the distance transform runs on `stream`
  cudaMemPool_t pool;         // every device allocation of the context comes from it (stream-ordered)
  bool own_pool;              // created in epo_create (cfg.mem_pool == NULL) and destroyed in epo_destroy
  cudaEvent_t ev_alloc, ev_copied;
  int N, W, H;
  bool have_views, have_pairs;
  bool pdl;            // programmatic dependent launch between the kernels of the loop (EPO_NO_PDL=1 turns it off)
  // The loop as ONE graph launch per epo_step call (epo_api.cu: build_step_graph): k_begin_step_call, then a conditional
  // WHILE node whose body is `unroll` iterations captured with their programmatic dependencies; k_finish sets the
  // condition.  Rebuilt whenever the pair list (and with it the kernels' arguments) changes.  EPO_NO_GRAPH=1: host loop.
  bool use_graph;
  int graph_unroll;
  cudaStream_t capture_stream;
  cudaGraph_t step_graph;
  cudaGraphExec_t step_exec;
  cudaGraphNode_t step_begin_node;
  cudaGraphConditionalHandle step_cond;
  bool coop_select;    // k_select_pairs with more than one CTA is launched cooperatively (EPO_NO_COOP=1 turns it off)
  bool static_dirty;   // work list / points / fields were (re)built since the last fused launch: launch it serialised
  int first_budget;    // > 0 while epo_step enqueues the FIRST iteration of a call that has no k_begin_step_call in front
                       // of it: its kernels gate on DevState.stopped and k_finish opens the call (iters_done, budget)
  int64_t P, E, n_work, reproj_per_eval, launches;
  int lg_chunk;        // samples per work item of the fused kernel (a multiple of kLgPass), chosen in epo_set_pairs

  // views
  float* d_K;             // [N][4]
  double* d_poses;        // [N][12] current (fp64: T_ts is formed without fp32 cancellation)
  double* d_poses_next;   // [N][12] poses after the update in flight (published by the last CTA of k_finish)
  double* d_poses_init;   // [N][12] as given to epo_set_views / epo_reset
  // joint loop (cfg.joint_phase): focal scale gamma per camera, depth affine (alpha, beta) per edge pixel;
  // everything per edge pixel lives in the packed slot order (EpoPacked), two samples per slot
  float* d_K0;            // [N][4] intrinsics as given
  double* d_gamma;        // [3][N] gamma, AdamW m, v
  float2* d_z0;           // [slots] depth as given
  double4* d_ab;          // [slots] (alpha_a, beta_a, alpha_b, beta_b)
  float4* d_abm;          // [slots][2] AdamW moments (m_alpha, v_alpha, m_beta, v_beta) of sample a, then b
  float2* d_dz;           // [n_work][chunk / 2] a . t_ts of both samples of every slot of every work item (the fused
                          // kernel's joint output of the iteration in flight; allocated with the pair list)
  double* d_glogf;        // [N] d L / d ln f (k_finish)
  int32_t* d_depth_stepped;  // [1] 1 once a depth step has been applied since the variables were last at the identity: until
                          // then the packed points are the ones built from (K0, Z0) and the fused kernel rescales them
  int32_t* d_edge_off;    // [N+1]
  EdgeRec* d_edges;       // [E]
  float* d_depth;         // [N][H][W] the depth maps as given (kept for epo_build_viewgraph)
  EpoPacked packed;       // [E] camera-frame points (x_s, y_s, z_s) in the fused kernel's layout: K and Z are fixed outside
                          // the joint phase, so row a-2 is hoisted; + the pixel index of every point
  EpoAtlas atlas;         // the distance fields as the fused kernel samples them (see EpoAtlas)
  std::vector<int32_t> h_edge_off;

  // pairs
  int2* d_pairs;          // [P] canonical (s, t), ascending (t, s)
  int32_t* d_perm;        // [P] user index of canonical pair k
  int32_t* d_tgt_off;     // [N+1] CSR by target over canonical ids
  int32_t* d_src_off;     // [N+1]
  int32_t* d_src_inc;     // [P] canonical ids grouped by source, ascending
  int4* d_work;           // [n_work] {source | target << 16, canonical pair, first point of the chunk (absolute), samples left}, target-major
  int32_t* d_work_off;    // [P+1] first work item of each canonical pair
  std::vector<int32_t> h_pairs;   // user order, for reprojection counting
  // stochastic pair sub-sampling (cfg.pair_budget > 0 and P > budget): rebuilt by k_select_pairs every iteration
  bool subsample;         // epo_step draws a subset each iteration
  uint8_t* d_sel_flag;    // [P] canonical order: in this iteration's subset
  int32_t* d_sel_work;    // [n_work] static work-item indices of the subset's pairs, in order
  int32_t* d_sel_info;    // {work items, pairs} of the subset
  int32_t* d_sel_scratch; // kSelScrInts ints, zero between launches of k_select_pairs (layout below)
  int64_t sel_grid;       // upper bound on the subset's work items (the fused kernel's grid in that mode)

  // per-evaluation buffers
  double* d_part;         // [n_work][8] per-CTA partial sums {S, n, A[3], M[3]} (no atomics: reproducible)
  float* d_pair_loss;     // [P] canonical order
  int32_t* d_pair_valid;  // [P]
  double* d_grad;         // [N][6]
  double* d_loss_part;    // [N] per-target partial sums of pair losses

  // optimiser
  double *d_m, *d_v;      // [N][6]
  double *d_dR, *d_dt;    // [N] per-camera pose change (degrees)
  DevState* d_state;
  double* d_sched;        // [max_steps][4] {lr_s, 1 - beta1^(s+1), 1 - beta2^(s+1), lambda_s}: row a-12, tabulated at create
  double* d_theta;        // [max_steps]
  double* d_loss_trace;   // [max_steps]

  // scratch for outputs in user order / fp32
  float* d_out_f;         // max(P, 12 N, max_steps) floats
  int32_t* d_out_i;       // P ints

  char err[512];
};

// relative pose T_ts = T_t T_s^-1 in fp64 (row a-1): entry k of the 3x4 [R_ts | t_ts], R_ts = R_t R_s^T,
// t_ts = t_t - R_ts t_s  (reading P2: formed in double, rounded once where fp32 is wanted)
#ifdef __CUDACC__
__device__ __forceinline__ double rel_pose_entry(const double* Ts, const double* Tt, int k) {
  int i = k >> 2, j = k & 3;
  if (j < 3) return Tt[4 * i] * Ts[4 * j] + Tt[4 * i + 1] * Ts[4 * j + 1] + Tt[4 * i + 2] * Ts[4 * j + 2];
  double r = Tt[4 * i + 3];
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    double Rim = Tt[4 * i] * Ts[4 * m] + Tt[4 * i + 1] * Ts[4 * m + 1] + Tt[4 * i + 2] * Ts[4 * m + 2];
    r -= Rim * Ts[4 * m + 3];
  }
  return r;
}
#endif

// ---- bounds checks of the hot kernels' indices (compute-sanitizer is closed on the GPU pool, profiles/r2_sanitizer.md):
// a library built with -DEPO_DEBUG_BOUNDS=1 asserts every index below against the size of what it indexes; a failed
// assert traps the kernel and the next API call returns EPO_ERR_CUDA.  Off (and free) in the product build.
#if defined(EPO_DEBUG_BOUNDS) && EPO_DEBUG_BOUNDS
#include <cassert>
#define EPO_CHECK(cond) assert(cond)
#else
#define EPO_CHECK(cond) ((void)0)
#endif

// ---- error plumbing ---------------------------------------------------------------------------
epo_status epo_fail(epo_ctx* ctx, epo_status st, const char* fmt, ...);

#define EPO_CUDA(ctx, call)                                                                         \
  do {                                                                                              \
    cudaError_t e_ = (call);                                                                        \
    if (e_ != cudaSuccess)                                                                          \
      return epo_fail((ctx), e_ == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, \
                      "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__);   \
  } while (0)

#define EPO_TRY(call)              \
  do {                             \
    epo_status s_ = (call);        \
    if (s_ != EPO_OK) return s_;   \
  } while (0)

// ---- device memory: stream-ordered allocation on the context's stream from the context's memory pool -- a private
// pool created in epo_create (release threshold = keep everything until epo_destroy), or the pool the caller passed in
// cfg.mem_pool.  A free costs no device synchronisation and a later allocation of the same size is served from the
// pool, which takes ~2.5 ms of cudaMalloc/cudaFree out of a repeated epo_set_views call.  The device's default pool
// and its attributes are never touched.
template <class T>
inline cudaError_t epo_dmalloc(epo_ctx* ctx, T** p, size_t bytes) {
  return cudaMallocFromPoolAsync(reinterpret_cast<void**>(p), bytes ? bytes : 1, ctx->pool, ctx->stream);
}
inline void epo_dfree(epo_ctx* ctx, void* p) {
  if (p) cudaFreeAsync(p, ctx->stream);
}

// ---- kernel launchers (each .cu file owns its kernels) ----------------------------------------
// preprocess.cu
epo_status epo_build_edge_lists(epo_ctx* ctx, const uint8_t* d_edges_u8, const float* d_depth,
                                int32_t** out_off, EdgeRec** out_rec, int64_t* out_E,
                                std::vector<int32_t>* h_off, bool* out_subsampled);
struct EpoDtfScratch { int32_t* g; cudaSurfaceObject_t surf, surf8; };   // alive until the EDT kernels have run
epo_status epo_build_dtf_atlas(epo_ctx* ctx, const uint8_t* d_edges_u8, EpoAtlas* atlas, EpoDtfScratch* scratch);
void epo_free_dtf_scratch(epo_ctx* ctx, EpoDtfScratch* s);
epo_status epo_build_points(epo_ctx* ctx, const float* d_K, const int32_t* d_off, const EdgeRec* d_rec, int64_t E,
                            const std::vector<int32_t>& h_off, const uint8_t* d_edges_u8, const float* d_depth,
                            bool subsampled, EpoPacked* out);   // tile-major points, packed (EpoPacked) + pixel indices
void epo_free_atlas(EpoAtlas* atlas);
void epo_free_packed(epo_ctx* ctx, EpoPacked* pk);
// pairs.cu
epo_status epo_build_pairs(epo_ctx* ctx, const int32_t* d_user_pairs, int64_t P, int2** out_pairs,
                           int32_t** out_perm, int32_t** out_tgt_off, int32_t** out_src_off,
                           int32_t** out_src_inc, int4** out_work, int32_t** out_work_off, int64_t* out_n_work,
                           int chunk);
// scratch of k_select_pairs (ints): grid-barrier counter + exit ticket, candidate count, global histogram, per-CTA
// totals, candidate keys (64-bit) and indices.  At most kSelMaxCtas CTAs of 4096 pairs (all resident: a spin barrier).
constexpr int kSelMaxCtas = 128, kSelCandCap = 4096;
constexpr int kSelScrBarrier = 0, kSelScrNCand = 2, kSelScrHist = 4, kSelScrTotals = kSelScrHist + 2048,
              kSelScrCandKey = kSelScrTotals + 2 * kSelMaxCtas, kSelScrCandIdx = kSelScrCandKey + 2 * kSelCandCap,
              kSelScrInts = kSelScrCandIdx + kSelCandCap;
int64_t epo_select_max_pairs(void);
epo_status epo_launch_select_pairs(epo_ctx* ctx, int step_override /* < 0: device step */, bool gated, bool build_work);
// canny.cu: edge maps (1 / 0) of [N][H][W] 8-bit images, device pointers
epo_status epo_run_canny(epo_ctx* ctx, const uint8_t* d_img, int low, int high, uint8_t* d_edges);
epo_status epo_run_rgb_to_grey(epo_ctx* ctx, const uint8_t* d_rgb, uint8_t* d_grey);   // [N][H][W][3] -> [N][H][W]
// joint.cu: the joint loop's depth-variable update (AdamW on alpha, beta; new points) and its state
epo_status epo_joint_alloc(epo_ctx* ctx);              // after the points exist (epo_set_views)
void epo_joint_free(epo_ctx* ctx);
epo_status epo_joint_reset(epo_ctx* ctx);              // identity variables, zero moments, K and points as given
epo_status epo_joint_reset_moments(epo_ctx* ctx);      // zero AdamW moments only (epo_set_pairs: the variables stay)
epo_status epo_launch_joint_points(epo_ctx* ctx, bool subset);   // gated by DevState.joint_pending
// d L / d Z of every listed edge pixel from the joint pass's per-slot output (d_dz) and the per-pair valid counts:
// written into the dense [N][H][W] map (zeroed here first)
epo_status epo_joint_gather_gz(epo_ctx* ctx, const float2* d_dz, float* d_map);
epo_status epo_joint_export(epo_ctx* ctx, double* d_gamma_out, double* d_alpha_map, double* d_beta_map);
// viewgraph.cu: cycle counts of all ordered pairs + ordered emission of the valid pairs
epo_status epo_launch_viewgraph(epo_ctx* ctx, int stride, float tau, float min_frac, int2* d_counts, int2* d_pairs,
                                long long* d_n);
// lossgrad.cu
epo_status epo_launch_fused(epo_ctx* ctx, float lambda_override /* < 0: device schedule */, bool gated, bool subset,
                            bool joint /* also the joint-phase derivatives: d_dz, 16-slot partial records */);
epo_status epo_launch_fused_only(epo_ctx* ctx, float lambda);   // the fused kernel alone (measurement hook)
epo_status epo_launch_record_taps(epo_ctx* ctx, float lambda, uint2* d_taps);                  // gather ceiling: the tap stream
epo_status epo_launch_gather_taps(epo_ctx* ctx, float lambda, const uint2* d_taps, unsigned* d_out);   // ... replayed alone
// update.cu: k_finish = per-camera reduction (+ Adam, retraction, pose change, stop test when step_mode)
epo_status epo_launch_finish(epo_ctx* ctx, bool step_mode, bool gated, bool subset, bool joint,
                             cudaGraphConditionalHandle cond /* 0: not inside the loop graph */);
epo_status epo_launch_fill_schedule(epo_ctx* ctx);     // d_sched from the configuration (once, in epo_create)
// first kernel of every epo_step call: iters_done = 0, budget = n_iters, stopped / halt from the current state
epo_status epo_launch_begin_step_call(epo_ctx* ctx, int n_iters);
// the same kernel as a graph node (epo_api.cu builds the node and updates n_iters before every graph launch)
struct EpoBeginArgs { DevState* st; int n_iters, graph_limit, max_steps, early_stop; cudaGraphConditionalHandle cond; void* ptrs[6]; void* func; };
void epo_begin_step_call_args(epo_ctx* ctx, int n_iters, int graph_limit, cudaGraphConditionalHandle cond, EpoBeginArgs* a);
void epo_launch_f64_to_f32(cudaStream_t st, const double* in, float* out, int64_t n);
void epo_launch_f32_to_f64(cudaStream_t st, const float* in, double* out, int64_t n);
void epo_launch_scatter_pair_outputs(cudaStream_t st, const float* pl, const int32_t* pv, const int32_t* perm,
                                     float* out_pl, int32_t* out_pv, int64_t P);
