// Everything of one iteration after the fused kernel (DESIGN.md rows a-9..a-12), one launch, fp64:
//   PAPER.md:485-486   per-direction mean  sum rho / sum valid;  PAPER.md:91 Eq. 6 mean over pairs
//   PAPER.md:121       Adam(W) beta=(0.9, 0.999); linear warm-up 0 -> 3e-3 over 25 steps, cosine decay to 2000
//   PAPER.md:429       OptimizerAndSchedulerStep
//   PAPER.md:104-110   Eq. 9 / Eq. 10 pose change in degrees, 95th percentiles, theta95 = max
//   PAPER.md:112-115, 123, 357, 433-446   windowed two-phase convergence (w1=25, eps1=0.5; w2=50, eps2=0.1)
// The pose parameterisation is a left se(3) increment per camera, T_c <- Exp(eps_c) T_c (north_star;
// DESIGN.md reading S9).  The stop decision is written to the device control block so that the
// following iterations' kernels exit immediately: epo_step never synchronises with the host.
#include <math_constants.h>

#include "epo_internal.h"

namespace {

constexpr double kPi = 3.14159265358979323846;
// k_finish: 512 threads (16 warps share a camera's incident pairs) at two CTAs per SM (<= 64 registers); measured against
// 256 / 1024 threads and 1..6 CTAs per SM: the time between two fused kernels falls from 74 to 49 us at config 4 and from
// 62 to 44 us at config 5
#ifndef EPO_FIN_THREADS
#define EPO_FIN_THREADS 512
#endif
constexpr int kFinThreads = EPO_FIN_THREADS;

struct FinParams {
  // a-9 inputs: pair lists and the fused kernel's per-CTA partial sums
  const int2* pairs;
  const int32_t *tgt_off, *src_off, *src_inc, *work_off;
  const double* part;
  const uint8_t* sel_flag;      // pair sub-sampling: membership of this iteration's subset (canonical order), else nullptr
  float* pair_loss;
  int32_t* pair_valid;
  double *grad, *loss_part;
  // optimiser state
  double *poses, *poses_next;
  // joint phase (kJoint): per-camera focal scale gamma (AdamW, Eq. 4, 121) and the intrinsics it rescales
  double *gamma /* [3][N] gamma, m, v */, *glogf /* [N] d L / d ln f */;
  const float* K0;
  float* K;
  double wd;
  double *m, *v, *dR, *dt, *theta, *loss_trace;
  DevState* state;
  int N;
  int64_t P, n_pairs, n_work;   // P: pairs the mean runs over; n_pairs, n_work: list sizes (EPO_CHECK)
  double beta1, beta2, adam_eps, eps1, eps2;
  const double* sched;          // [max_steps][4] {lr_s, 1 - beta1^(s+1), 1 - beta2^(s+1), lambda_s}
  int max_steps, w1, w2, smooth, early_stop, stop_rule, w_loss;
  double eps_loss;
  int gated, step_mode;      // gated: 1 = by DevState.halt; 2 = first iteration of a call without k_begin_step_call: by
                             // DevState.stopped, and this launch opens the call (iters_done = 0, budget = call_budget)
  int call_budget;
  cudaGraphConditionalHandle cond;   // the loop graph's WHILE condition (0 outside the graph)
};

// sum over the CTA in a fixed order (xor tree inside each warp, then the warps in index order); every thread
// gets the total.  `scratch` holds kFinThreads / 32 doubles.
__device__ double block_sum(double v, double* scratch) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();                                  // scratch may still be in use
  if ((threadIdx.x & 31) == 0) scratch[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
#pragma unroll
  for (int w = 0; w < kFinThreads / 32; ++w) t += scratch[w];
  return t;
}

__device__ double lr_of_step(int s, double lr_max, int warmup, int max_steps) {
  if (s < warmup) return lr_max * (double)(s + 1) / (double)warmup;
  return lr_max * 0.5 * (1.0 + cos(kPi * (double)(s - warmup) / (double)(max_steps - warmup)));
}

// Exp(v, w) = [Exp_SO3(w), V(w) v]; V = I + (1-cos th)/th^2 [w]x + (th - sin th)/th^3 [w]x^2
__device__ void se3_exp(const double* e, double* T) {
  const double v0 = e[0], v1 = e[1], v2 = e[2], w0 = e[3], w1 = e[4], w2 = e[5];
  const double th2 = w0 * w0 + w1 * w1 + w2 * w2;
  double A, B, C;
  if (th2 < 1e-2) {
    // |w| < 0.1 (an Adam step is a few 1e-3): the three series in th^2, seven terms each (next term < 1e-26),
    // by Horner -- no sin / cos / sqrt on the serial path of the iteration
    A = 1.0 + th2 * (-1.0 / 6 + th2 * (1.0 / 120 + th2 * (-1.0 / 5040 + th2 * (1.0 / 362880 + th2 * (-1.0 / 39916800 + th2 * (1.0 / 6227020800.0))))));
    B = 0.5 + th2 * (-1.0 / 24 + th2 * (1.0 / 720 + th2 * (-1.0 / 40320 + th2 * (1.0 / 3628800 + th2 * (-1.0 / 479001600 + th2 * (1.0 / 87178291200.0))))));
    C = 1.0 / 6 + th2 * (-1.0 / 120 + th2 * (1.0 / 5040 + th2 * (-1.0 / 362880 + th2 * (1.0 / 39916800 + th2 * (-1.0 / 6227020800.0 + th2 * (1.0 / 1307674368000.0))))));
  } else { const double th = sqrt(th2); A = sin(th) / th; B = (1.0 - cos(th)) / th2; C = (th - sin(th)) / (th2 * th); }
  const double Wx[9] = {0, -w2, w1, w2, 0, -w0, -w1, w0, 0};
  double W2[9];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      W2[3 * i + j] = Wx[3 * i] * Wx[j] + Wx[3 * i + 1] * Wx[3 + j] + Wx[3 * i + 2] * Wx[6 + j];
  const double vv[3] = {v0, v1, v2};
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double tv = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      const double I = (i == j) ? 1.0 : 0.0;
      T[4 * i + j] = I + A * Wx[3 * i + j] + B * W2[3 * i + j];
      tv += (I + B * Wx[3 * i + j] + C * W2[3 * i + j]) * vv[j];
    }
    T[4 * i + 3] = tv;
  }
}

__device__ __forceinline__ double clip1(double c) { return c > 1.0 ? 1.0 : (c < -1.0 ? -1.0 : c); }

// value of ranks k and k+1 (0-based, ties broken by index) among x[0..n): every thread scans all of x
__device__ void select_two(const double* x, int n, int k, double* lo, double* hi) {
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const double xi = x[i];
    int rank = 0;
    for (int j = 0; j < n; ++j) { const double xj = x[j]; rank += (xj < xi) || (xj == xi && j < i); }
    if (rank == k) *lo = xi;
    if (rank == k + 1 || (k + 1 >= n && rank == k)) *hi = xi;
  }
}

// Converged(theta_{0..s}; w, eps)  (smooth: PAPER.md:357; raw: PAPER.md:114), evaluated by the whole CTA:
// thread k tests the windows ending at steps s - k, s - k - blockDim, ... (k < w; each mean is summed in time order).
__device__ bool converged(const double* theta, double theta_s, int s, int w, double eps, int smooth) {
  const int need = smooth ? 2 * w - 2 : w - 1;
  if (s < need) return false;                       // uniform
  bool ok = true;
  auto th = [&](int j) { return j == s ? theta_s : __ldcg(theta + j); };
  for (int k = threadIdx.x; k < w; k += blockDim.x) {       // any window length: strided over the CTA
    if (smooth) {
      double m = 0.0;
      for (int j = s - k - w + 1; j <= s - k; ++j) m += th(j);
      ok = ok && (m / w < eps);
    } else {
      ok = ok && (th(s - k) < eps);
    }
  }
  return __syncthreads_and(ok) != 0;
}

// ---------------------------------------------------------------------------------------------------------
// k_finish: everything of one iteration after the fused kernel, in ONE launch of N CTAs (one per camera c).
//  a-9   g_c = (1/P) [ sum_{p: t=c} [A; M]_p / n_p  -  sum_{p: s=c} Ad_{T_ts}^T [A; M]_p / n_p ]   (identity I1:
//        G_src = [-R^T A ; -R^T (M - t x A)]), L_p = S_p / n_p, per-target loss sums.  One warp per pair.
//  a-10  (step mode) Adam on the six coordinates (lanes 2..7 of warp 0), SE(3) exponential and T_c <- Exp(eps) T_c
//        by one thread, written to the NEXT pose buffer: other CTAs still read the current poses.
//  a-11  per-camera pose change; then the LAST CTA to finish (atomic ticket) publishes the new poses, takes the
//  a-12  two 95th percentiles, runs the windowed two-phase test and advances the device control block.
// ---------------------------------------------------------------------------------------------------------
// Loss-based rule: relative loss change |L_k - L_{k-1}| / |L_{k-1}| < eps for the w steps k = s-w+1 .. s
// (s >= w); thread j tests step s - j, strided over the window.
__device__ bool converged_loss(const double* trace, double loss_s, int s, int w, double eps) {
  if (w < 1 || s < w) return false;                  // uniform
  bool ok = true;
  auto L = [&](int k) { return k == s ? loss_s : __ldcg(trace + k); };
  for (int j = threadIdx.x; j < w; j += blockDim.x) {
    const double a = L(s - j - 1), d = fabs(L(s - j) - a);
    const double r = a != 0.0 ? d / fabs(a) : (d == 0.0 ? 0.0 : CUDART_INF);
    ok = ok && (r < eps);
  }
  return __syncthreads_and(ok) != 0;
}

#ifndef EPO_FIN_MINBLOCKS
#define EPO_FIN_MINBLOCKS 2
#endif
template <bool kJoint>
__global__ void __launch_bounds__(kFinThreads, EPO_FIN_MINBLOCKS) k_finish(const FinParams p) {
  // partial records: 8 values x 4 chunk classes per warp round, or (joint phase) 16 slots x 2 classes
  constexpr int kVal = kJoint ? kAccStrideJoint : kAccStride, kCls = 32 / kVal;
  DevState* st = p.state;
  extern __shared__ double sdyn[];                 // last CTA: dR[N], dt[N]
  __shared__ double sg[kFinThreads / 32][8];
  __shared__ double sj[kFinThreads / 32];
  __shared__ double sel[4];
  __shared__ int s_last;
  const int c = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, N = p.N;
  constexpr int kWarps = kFinThreads / 32;
  // The pair lists are static: read this camera's ranges, and for every lane one incident pair with its range of
  // work items, before waiting for the fused kernel (programmatic dependent launch: this prologue overlaps the
  // fused kernel's tail).  Incident pairs = first those with target c, then those with source c; warp w takes
  // groups w, w + 8, ... of G consecutive ones (G <= 32 chosen so that all warps share a short list).
  const int t0 = p.tgt_off[c], nt = p.tgt_off[c + 1] - t0, s0 = p.src_off[c], n_inc = nt + p.src_off[c + 1] - s0;
  int G = (n_inc + kWarps - 1) / kWarps;
  G = G < 1 ? 1 : (G > 32 ? 32 : G);
  auto fetch = [&](int j0, int* q, int* w0, int* w1, int* tv) {
    const int j = j0 + lane;
    *q = -1; *w0 = 0; *w1 = 0; *tv = 0;
    if (lane < G && j < n_inc) {
      *q = j < nt ? t0 + j : p.src_inc[s0 + j - nt];
      *w0 = p.work_off[*q]; *w1 = p.work_off[*q + 1];
      *tv = p.pairs[*q].y;                           // the pair's target view (needed when c is its source)
    }
  };
  int j0 = warp * G, q, w0, w1, tv;
  fetch(j0, &q, &w0, &w1, &tv);
  cudaTriggerProgrammaticLaunchCompletion();       // the next fused kernel may start its own static prologue
  cudaGridDependencySynchronize();                 // partial sums, poses and the control block are final now
  const bool first = p.gated == 2;
  if (p.gated && (first ? st->stopped : st->halt)) {
    if (blockIdx.x == 0 && threadIdx.x == 0) {
      st->joint_pending = 0;
      if (first) { st->iters_done = 0; st->budget = p.call_budget; st->halt = 1; }
      if (p.cond) cudaGraphSetConditional(p.cond, 0);
    }
    return;
  }
  const double* Pc = p.poses + 12 * (size_t)c;
  // ---- a-9: one warp per incident pair; lane 0 accumulates the loss sum, lanes 2..7 the six gradient
  // coordinates.  With pair sub-sampling only the pairs of this iteration's subset count.
  double acc = 0.0;
  while (j0 < n_inc) {
    unsigned todo = __ballot_sync(0xffffffffu, q >= 0 && (p.sel_flag == nullptr || p.sel_flag[q] != 0));
    const int jc = j0, qm = q, w0m = w0, w1m = w1, tvm = tv;
    j0 += kWarps * G;
    if (j0 < n_inc) fetch(j0, &q, &w0, &w1, &tv);  // the next group's ranges, in flight
    while (todo) {
      const int b = __ffs(todo) - 1;
      todo &= todo - 1;
      const int qc = __shfl_sync(0xffffffffu, qm, b);
      const int wa = __shfl_sync(0xffffffffu, w0m, b), wb = __shfl_sync(0xffffffffu, w1m, b);
      const int tview = __shfl_sync(0xffffffffu, tvm, b);
      const bool tgt = jc + b < nt;
      EPO_CHECK(qc >= 0 && qc < p.n_pairs && wa >= 0 && wa <= wb && wb <= p.n_work && tview >= 0 && tview < N);
      // per-pair sums: lane l adds value (l & 7) of chunks (l >> 3), (l >> 3) + 4, ... (independent loads), then
      // the four chunk classes are combined by two xor-shuffles: a fixed order
      double v = 0.0;
      for (int w = wa + lane / kVal; w < wb; w += kCls) v += __ldcg(p.part + (size_t)w * kVal + (lane % kVal));
      if (!kJoint) v += __shfl_xor_sync(0xffffffffu, v, 8);
      v += __shfl_xor_sync(0xffffffffu, v, 16);
      const double n = __shfl_sync(0xffffffffu, v, 1);
      // joint phase: lane 8 accumulates d L / d ln f of this camera -- the pair's target sum (slot 8) when the camera
      // is the pair's target, its source sum (slot 9) when it is the source
      const double js = kJoint ? __shfl_sync(0xffffffffu, v, 9) : 0.0;
      if (kJoint && lane == 8 && n > 0.0) acc += (tgt ? v : js) / n;
      if (tgt) {
        const double S = __shfl_sync(0xffffffffu, v, 0);
        const double L = n > 0.0 ? S / n : 0.0;
        if (lane == 0) { p.pair_loss[qc] = (float)L; p.pair_valid[qc] = (int32_t)n; acc += L; }
        else if (lane >= 2 && lane < 8 && n > 0.0) acc += v / n;
      } else {
        const double A0 = __shfl_sync(0xffffffffu, v, 2), A1 = __shfl_sync(0xffffffffu, v, 3), A2 = __shfl_sync(0xffffffffu, v, 4);
        double m0 = __shfl_sync(0xffffffffu, v, 5), m1 = __shfl_sync(0xffffffffu, v, 6), m2 = __shfl_sync(0xffffffffu, v, 7);
        if (lane >= 2 && lane < 8 && n > 0.0) {
          const double* Pt = p.poses + 12 * (size_t)tview;
          const int i = (lane - 2) % 3;
          const double r0 = rel_pose_entry(Pc, Pt, i), r1 = rel_pose_entry(Pc, Pt, 4 + i), r2 = rel_pose_entry(Pc, Pt, 8 + i);
          if (lane < 5) {
            acc -= (r0 * A0 + r1 * A1 + r2 * A2) / n;                      // R^T A
          } else {
            const double t0 = rel_pose_entry(Pc, Pt, 3), t1 = rel_pose_entry(Pc, Pt, 7), t2 = rel_pose_entry(Pc, Pt, 11);
            m0 -= t1 * A2 - t2 * A1; m1 -= t2 * A0 - t0 * A2; m2 -= t0 * A1 - t1 * A0;   // M' = M - t_ts x A
            acc -= (r0 * m0 + r1 * m1 + r2 * m2) / n;                      // R^T M'
          }
        }
      }
    }
  }
  if (lane < 8) sg[warp][lane] = acc;
  if (kJoint && lane == 8) sj[warp] = acc;
  __syncthreads();
  double g = 0.0;                                    // warp 0, lane k < 8: sum over warps in a fixed order
  if (tid < 8) {
#pragma unroll
    for (int w = 0; w < kFinThreads / 32; ++w) g += sg[w][tid];
    if (tid == 0) p.loss_part[c] = g;
    else if (tid >= 2) { g /= (double)p.P; p.grad[6 * (size_t)c + tid - 2] = g; }
  } else if (kJoint && tid == 8) {
#pragma unroll
    for (int w = 0; w < kFinThreads / 32; ++w) g += sj[w];
    g /= (double)p.P;
    p.glogf[c] = g;
  }
  if (!p.step_mode) {
    // evaluation only (epo_loss_grad): the last CTA adds the per-target loss sums
    if (tid == 0) { __threadfence(); s_last = atomicAdd(&st->ticket, 1) == N - 1; }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double lv = 0.0;
    for (int i = tid; i < N; i += kFinThreads) lv += __ldcg(p.loss_part + i);
    const double tot = block_sum(lv, &sg[0][0]);
    if (tid == 0) { st->loss = tot / (double)p.P; st->ticket = 0; }
    return;
  }
  // ---- a-10 Adam (lanes 2..7 of warp 0); the step-dependent scalars come from the schedule table (a-12)
  const int s = st->step;
  __shared__ double sT[24];                          // new pose, old pose
  if (warp == 0) {
    double eps = 0.0;
    if (lane >= 2 && lane < 8) {
      const size_t k = 6 * (size_t)c + lane - 2;
      const double lr = p.sched[4 * (size_t)s], c1 = p.sched[4 * (size_t)s + 1], c2 = p.sched[4 * (size_t)s + 2];
      const double m = p.beta1 * p.m[k] + (1.0 - p.beta1) * g;
      const double v = p.beta2 * p.v[k] + (1.0 - p.beta2) * g * g;
      p.m[k] = m; p.v[k] = v;
      eps = -lr * (m / c1) / (sqrt(v / c2) + p.adam_eps);
    }
    double e[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) e[k] = __shfl_sync(0xffffffffu, eps, 2 + k);
    if (lane == 0) {
      // retraction T_c <- Exp(eps) T_c
      double E[12], T[12], Tn[12];
      se3_exp(e, E);
#pragma unroll
      for (int k = 0; k < 12; ++k) T[k] = Pc[k];
#pragma unroll
      for (int i = 0; i < 3; ++i) {
#pragma unroll
        for (int j = 0; j < 4; ++j) Tn[4 * i + j] = E[4 * i] * T[j] + E[4 * i + 1] * T[4 + j] + E[4 * i + 2] * T[8 + j];
        Tn[4 * i + 3] += E[4 * i + 3];
      }
#pragma unroll
      for (int k = 0; k < 12; ++k) { sT[k] = Tn[k]; sT[12 + k] = T[k]; }
    }
  }
  if (kJoint && tid == 8) {
    // focal scale (Eq. 4): f_c = f0_c (1 + gamma_c), stepped in every iteration ("the first phase ...
    // drives updates to the camera intrinsics K and poses P").  AdamW [PAPER.md:121] with the loop's
    // learning rate, decay towards the identity value 0; d L / d gamma = (d L / d ln f) / (1 + gamma); step number s + 1.
    const int N_ = p.N;
    const double lr = p.sched[4 * (size_t)s], c1 = p.sched[4 * (size_t)s + 1], c2 = p.sched[4 * (size_t)s + 2];
    double gm = p.gamma[c];
    const double gg = g / (1.0 + gm);
    gm -= lr * p.wd * gm;
    const double mm = p.beta1 * p.gamma[N_ + c] + (1.0 - p.beta1) * gg, vv = p.beta2 * p.gamma[2 * N_ + c] + (1.0 - p.beta2) * gg * gg;
    p.gamma[N_ + c] = mm; p.gamma[2 * N_ + c] = vv;
    gm -= lr * (mm / c1) / (sqrt(vv / c2) + p.adam_eps);
    p.gamma[c] = gm;
    p.K[4 * c] = (float)((double)p.K0[4 * c] * (1.0 + gm));
    p.K[4 * c + 1] = (float)((double)p.K0[4 * c + 1] * (1.0 + gm));
  }
  __syncthreads();
  // ---- a-11 pose change of this camera: three warps side by side
  if (tid == 0) {
    double tr = 0.0;   // Eq. 9: tr(R^s (R^{s-1})^T)
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = 0; j < 3; ++j) tr += sT[4 * i + j] * sT[12 + 4 * i + j];
    p.dR[c] = (180.0 / kPi) * acos(clip1((tr - 1.0) / 2.0));
    __threadfence();
  } else if (tid == 32) {
    const double a0 = sT[3], a1 = sT[7], a2 = sT[11], b0 = sT[15], b1 = sT[19], b2 = sT[23];
    const double na = sqrt(a0 * a0 + a1 * a1 + a2 * a2), nb = sqrt(b0 * b0 + b1 * b1 + b2 * b2);
    double dtc = 0.0;  // Eq. 10; 0 if either norm < 1e-12 (reading S13)
    if (na >= 1e-12 && nb >= 1e-12)
      dtc = (180.0 / kPi) * acos(clip1((a0 / na) * (b0 / nb) + (a1 / na) * (b1 / nb) + (a2 / na) * (b2 / nb)));
    p.dt[c] = dtc;
    __threadfence();
  } else if (tid >= 64 && tid < 76) {
    p.poses_next[12 * (size_t)c + tid - 64] = sT[tid - 64];
    __threadfence();
  }
  __syncthreads();
  if (tid == 0) s_last = atomicAdd(&st->ticket, 1) == N - 1;   // this camera's outputs precede its ticket
  __syncthreads();
  if (!s_last) return;
  // ---- last CTA: every camera has been reduced and stepped; nobody reads the current poses any more
  __threadfence();
  double* sdR = sdyn; double* sdt = sdyn + N;
  double lv = 0.0;
  for (int i = tid; i < N; i += kFinThreads) {
    sdR[i] = __ldcg(p.dR + i); sdt[i] = __ldcg(p.dt + i);
    lv += __ldcg(p.loss_part + i);
  }
  for (int i = tid; i < 12 * N; i += kFinThreads) p.poses[i] = __ldcg(p.poses_next + i);
  const double loss = block_sum(lv, &sg[0][0]) / (double)p.P;     // (contains the barrier that publishes sdR / sdt)
  // 95th percentiles, linear interpolation at rank 0.95 (N-1) (reading S12)
  const double rank = 95.0 / 100.0 * (double)(N - 1);
  const int k0 = (int)floor(rank);
  const double fr = rank - (double)k0;
  select_two(sdR, N, k0, &sel[0], &sel[1]);
  select_two(sdt, N, k0, &sel[2], &sel[3]);
  __syncthreads();
  const double r95 = (k0 + 1 < N) ? sel[0] + fr * (sel[1] - sel[0]) : sel[0];
  const double t95 = (k0 + 1 < N) ? sel[2] + fr * (sel[3] - sel[2]) : sel[2];
  const double th = r95 > t95 ? r95 : t95;
  int phase = st->phase;
  const int phase0 = phase;
  if (phase == 0) { if (converged(p.theta, th, s, p.w1, p.eps1, p.smooth)) phase = 1; }
  else if (phase == 1) {
    if (p.stop_rule == 1 ? converged_loss(p.loss_trace, loss, s, p.w_loss, p.eps_loss)
                         : converged(p.theta, th, s, p.w2, p.eps2, p.smooth)) phase = 2;
  }
  if (tid == 0) {
    p.theta[s] = th;
    p.loss_trace[s] = loss;
    st->loss = loss;
    st->phase = phase;
    st->phase_prev = phase0; st->joint_pending = 1;
    if (phase0 == 0 && phase == 1) st->phase1_step = s;
    st->step = s + 1;
    const int done = (first ? 0 : st->iters_done) + 1;
    const int budget = first ? p.call_budget : st->budget;
    const int stopped = (s + 1 >= p.max_steps) || (p.early_stop && phase == 2);
    const int halt = stopped || done >= budget;
    st->iters_done = done; st->budget = budget; st->stopped = stopped; st->halt = halt;
    // the loop graph runs its body again only while the call may go on: nothing is launched after the stop
    if (p.cond) cudaGraphSetConditional(p.cond, (stopped || done >= st->graph_limit) ? 0u : 1u);
    st->ticket = 0;
  }
}

// a-12 schedules, tabulated once per context (the configuration is immutable): row s = {lr_s, 1 - beta1^(s+1),
// 1 - beta2^(s+1), lambda_s}.  lambda_s = clamp_start + (clamp_end - clamp_start) min(s, clamp_steps) / clamp_steps
// (PAPER.md:462), rounded to fp32 as the fused kernel uses it.
__global__ void k_fill_schedule(double* __restrict__ sched, int max_steps, double lr_max, int warmup, double beta1,
                                double beta2, double clamp_start, double clamp_end, int clamp_steps) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= max_steps) return;
  const int m = s < clamp_steps ? s : clamp_steps;
  sched[4 * s] = lr_of_step(s, lr_max, warmup, max_steps);
  sched[4 * s + 1] = 1.0 - pow(beta1, (double)(s + 1));
  sched[4 * s + 2] = 1.0 - pow(beta2, (double)(s + 1));
  sched[4 * s + 3] = (double)(float)(clamp_start + (clamp_end - clamp_start) * (double)m / (double)clamp_steps);
}

__global__ void k_begin_step_call(DevState* st, int n_iters, int graph_limit, int max_steps, int early_stop,
                                  cudaGraphConditionalHandle cond) {
  const int stopped = (st->step >= max_steps) || (early_stop && st->phase == 2);
  const int halt = stopped || n_iters <= 0;
  st->iters_done = 0; st->budget = n_iters; st->graph_limit = graph_limit; st->stopped = stopped; st->halt = halt;
  if (cond) cudaGraphSetConditional(cond, (stopped || graph_limit <= 0) ? 0u : 1u);
}

__global__ void k_f64_to_f32(const double* __restrict__ in, float* __restrict__ out, int64_t n) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (float)in[i];
}
__global__ void k_f32_to_f64(const float* __restrict__ in, double* __restrict__ out, int64_t n) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (double)in[i];
}

}  // namespace

epo_status epo_launch_finish(epo_ctx* ctx, bool step_mode, bool gated, bool subset, bool joint, cudaGraphConditionalHandle cond) {
  FinParams p;
  p.gamma = ctx->d_gamma; p.glogf = ctx->d_glogf; p.K0 = ctx->d_K0; p.K = ctx->d_K; p.wd = ctx->cfg.weight_decay;
  if (joint && !ctx->d_glogf) return epo_fail(ctx, EPO_ERR_BAD_STATE, "joint-phase reduction without joint state");
  p.sel_flag = subset ? ctx->d_sel_flag : nullptr;
  p.pairs = ctx->d_pairs; p.tgt_off = ctx->d_tgt_off; p.src_off = ctx->d_src_off; p.src_inc = ctx->d_src_inc;
  p.work_off = ctx->d_work_off; p.part = ctx->d_part; p.pair_loss = ctx->d_pair_loss; p.pair_valid = ctx->d_pair_valid;
  p.grad = ctx->d_grad; p.loss_part = ctx->d_loss_part;
  p.poses = ctx->d_poses; p.poses_next = ctx->d_poses_next; p.m = ctx->d_m; p.v = ctx->d_v;
  p.dR = ctx->d_dR; p.dt = ctx->d_dt; p.theta = ctx->d_theta; p.loss_trace = ctx->d_loss_trace;
  p.state = ctx->d_state; p.N = ctx->N; p.n_pairs = ctx->P; p.n_work = ctx->n_work;
  p.P = subset ? (int64_t)ctx->cfg.pair_budget : ctx->P;     // the mean runs over the pairs that were evaluated
  p.sched = ctx->d_sched; p.beta1 = ctx->cfg.beta1; p.beta2 = ctx->cfg.beta2; p.adam_eps = ctx->cfg.adam_eps;
  p.eps1 = ctx->cfg.eps1; p.eps2 = ctx->cfg.eps2; p.max_steps = ctx->cfg.max_steps;
  p.w1 = ctx->cfg.w1; p.w2 = ctx->cfg.w2; p.smooth = ctx->cfg.smooth_window; p.early_stop = ctx->cfg.early_stop;
  p.stop_rule = ctx->cfg.stop_rule; p.w_loss = ctx->cfg.w_loss; p.eps_loss = ctx->cfg.eps_loss;
  p.gated = gated ? (ctx->first_budget > 0 ? 2 : 1) : 0; p.call_budget = ctx->first_budget; p.step_mode = step_mode ? 1 : 0; p.cond = cond;
  const size_t smem = (size_t)2 * ctx->N * sizeof(double);   // the last CTA's copy of dR, dt
  if (smem > 200 * 1024) return epo_fail(ctx, EPO_ERR_UNSUPPORTED, "more than %d views", 200 * 1024 / 16);
  if (smem > 48 * 1024) {
    EPO_CUDA(ctx, cudaFuncSetAttribute(k_finish<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    EPO_CUDA(ctx, cudaFuncSetAttribute(k_finish<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  }
  // programmatic dependent launch: the CTAs may become resident while the fused kernel drains; they wait in
  // cudaGridDependencySynchronize() before touching anything it (or an earlier kernel) wrote
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)ctx->N); lc.blockDim = dim3(kFinThreads); lc.dynamicSmemBytes = smem; lc.stream = ctx->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = ctx->pdl ? 1 : 0;
  EPO_CUDA(ctx, joint ? cudaLaunchKernelEx(&lc, k_finish<true>, p) : cudaLaunchKernelEx(&lc, k_finish<false>, p));
  ctx->launches += 1;
  EPO_CUDA(ctx, cudaGetLastError());
  return EPO_OK;
}

epo_status epo_launch_fill_schedule(epo_ctx* ctx) {
  const epo_config& g = ctx->cfg;
  k_fill_schedule<<<(g.max_steps + 127) / 128, 128, 0, ctx->stream>>>(ctx->d_sched, g.max_steps, g.lr_max, g.warmup_steps, g.beta1,
                                                                      g.beta2, g.clamp_start, g.clamp_end, g.clamp_steps);
  ctx->launches += 1;
  EPO_CUDA(ctx, cudaGetLastError());
  return EPO_OK;
}

epo_status epo_launch_begin_step_call(epo_ctx* ctx, int n_iters) {
  k_begin_step_call<<<1, 1, 0, ctx->stream>>>(ctx->d_state, n_iters, 0, ctx->cfg.max_steps, ctx->cfg.early_stop, 0);
  ctx->launches += 1;
  EPO_CUDA(ctx, cudaGetLastError());
  return EPO_OK;
}

void epo_begin_step_call_args(epo_ctx* ctx, int n_iters, int graph_limit, cudaGraphConditionalHandle cond, EpoBeginArgs* a) {
  a->st = ctx->d_state; a->n_iters = n_iters; a->graph_limit = graph_limit; a->max_steps = ctx->cfg.max_steps;
  a->early_stop = ctx->cfg.early_stop; a->cond = cond;
  a->ptrs[0] = &a->st; a->ptrs[1] = &a->n_iters; a->ptrs[2] = &a->graph_limit; a->ptrs[3] = &a->max_steps; a->ptrs[4] = &a->early_stop;
  a->ptrs[5] = &a->cond;
  a->func = (void*)k_begin_step_call;
}

void epo_launch_f64_to_f32(cudaStream_t st, const double* in, float* out, int64_t n) {
  if (n > 0) k_f64_to_f32<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(in, out, n);
}
void epo_launch_f32_to_f64(cudaStream_t st, const float* in, double* out, int64_t n) {
  if (n > 0) k_f32_to_f64<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(in, out, n);
}
