// Optimiser side of one iteration (DESIGN.md rows a-10..a-12), one CTA, fp64 (N is a few hundred):
//   PAPER.md:121       Adam(W) beta=(0.9, 0.999); linear warm-up 0 -> 3e-3 over 25 steps, cosine decay to 2000
//   PAPER.md:429       OptimizerAndSchedulerStep
//   PAPER.md:104-110   Eq. 9 / Eq. 10 pose change in degrees, 95th percentiles, theta95 = max
//   PAPER.md:112-115, 123, 357, 433-446   windowed two-phase convergence (w1=25, eps1=0.5; w2=50, eps2=0.1)
// The pose parameterisation is a left se(3) increment per camera, T_c <- Exp(eps_c) T_c (north_star;
// DESIGN.md reading S9).  The stop decision is written to the device control block so that the
// following iterations' kernels exit immediately: epo_step never synchronises with the host.
#include "epo_internal.h"

namespace {

constexpr double kPi = 3.14159265358979323846;
constexpr int kUpdThreads = 256;

struct UpdParams {
  double* poses;
  const double* grad;
  const double* loss_part;
  double *m, *v, *dR, *dt, *theta, *loss_trace;
  DevState* state;
  int N;
  int64_t P;
  double lr_max, beta1, beta2, adam_eps, eps1, eps2;
  int warmup, max_steps, w1, w2, smooth, early_stop;
};

__device__ double lr_of_step(int s, double lr_max, int warmup, int max_steps) {
  if (s < warmup) return lr_max * (double)(s + 1) / (double)warmup;
  return lr_max * 0.5 * (1.0 + cos(kPi * (double)(s - warmup) / (double)(max_steps - warmup)));
}

// Exp(v, w) = [Exp_SO3(w), V(w) v]; V = I + (1-cos th)/th^2 [w]x + (th - sin th)/th^3 [w]x^2
__device__ void se3_exp(const double* e, double* T) {
  const double v0 = e[0], v1 = e[1], v2 = e[2], w0 = e[3], w1 = e[4], w2 = e[5];
  const double th2 = w0 * w0 + w1 * w1 + w2 * w2, th = sqrt(th2);
  double A, B, C;
  if (th < 1e-4) { A = 1.0 - th2 / 6.0; B = 0.5 - th2 / 24.0; C = 1.0 / 6.0 - th2 / 120.0; }
  else { A = sin(th) / th; B = (1.0 - cos(th)) / th2; C = (th - sin(th)) / (th2 * th); }
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

// value of rank k (0-based, ties broken by index) among x[0..n): every thread scans all of x
__device__ void select_two(const double* x, int n, int k, double* lo, double* hi) {
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const double xi = x[i];
    int rank = 0;
    for (int j = 0; j < n; ++j) { const double xj = x[j]; rank += (xj < xi) || (xj == xi && j < i); }
    if (rank == k) *lo = xi;
    if (rank == k + 1 || (k + 1 >= n && rank == k)) *hi = xi;
  }
}

// Converged(theta_{0..s}; w, eps)  (smooth: PAPER.md:357; raw: PAPER.md:114)
__device__ bool converged(const double* theta, int s, int w, double eps, int smooth) {
  if (smooth) {
    if (s < 2 * w - 2) return false;
    for (int k = s - w + 1; k <= s; ++k) {
      double m = 0.0;
      for (int j = k - w + 1; j <= k; ++j) m += theta[j];
      if (!(m / w < eps)) return false;
    }
    return true;
  }
  if (s < w - 1) return false;
  for (int k = s - w + 1; k <= s; ++k) if (!(theta[k] < eps)) return false;
  return true;
}

__global__ void __launch_bounds__(kUpdThreads) k_update(const UpdParams p) {
  DevState* st = p.state;
  if (st->stopped) return;
  __shared__ double sred[kUpdThreads];
  __shared__ double sel[4];
  const int tid = threadIdx.x, s = st->step, N = p.N;
  // total loss of this evaluation (fixed-order tree)
  double lv = 0.0;
  for (int i = tid; i < N; i += kUpdThreads) lv += p.loss_part[i];
  sred[tid] = lv;
  __syncthreads();
  for (int o = kUpdThreads / 2; o > 0; o >>= 1) { if (tid < o) sred[tid] += sred[tid + o]; __syncthreads(); }
  const double loss = sred[0] / (double)p.P;
  // a-10 Adam + retraction, a-11 per-camera pose change
  const double lr = lr_of_step(s, p.lr_max, p.warmup, p.max_steps);
  const double c1 = 1.0 - pow(p.beta1, (double)(s + 1)), c2 = 1.0 - pow(p.beta2, (double)(s + 1));
  for (int c = tid; c < N; c += kUpdThreads) {
    double eps[6], E[12], T[12], Tn[12];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const double g = p.grad[6 * c + k];
      const double m = p.beta1 * p.m[6 * c + k] + (1.0 - p.beta1) * g;
      const double v = p.beta2 * p.v[6 * c + k] + (1.0 - p.beta2) * g * g;
      p.m[6 * c + k] = m; p.v[6 * c + k] = v;
      eps[k] = -lr * (m / c1) / (sqrt(v / c2) + p.adam_eps);
    }
    se3_exp(eps, E);
#pragma unroll
    for (int k = 0; k < 12; ++k) T[k] = p.poses[12 * c + k];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
#pragma unroll
      for (int j = 0; j < 4; ++j) Tn[4 * i + j] = E[4 * i] * T[j] + E[4 * i + 1] * T[4 + j] + E[4 * i + 2] * T[8 + j];
      Tn[4 * i + 3] += E[4 * i + 3];
    }
    double tr = 0.0;   // Eq. 9: tr(R^s (R^{s-1})^T)
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = 0; j < 3; ++j) tr += Tn[4 * i + j] * T[4 * i + j];
    p.dR[c] = (180.0 / kPi) * acos(clip1((tr - 1.0) / 2.0));
    const double na = sqrt(Tn[3] * Tn[3] + Tn[7] * Tn[7] + Tn[11] * Tn[11]);
    const double nb = sqrt(T[3] * T[3] + T[7] * T[7] + T[11] * T[11]);
    double dtc = 0.0;  // Eq. 10; 0 if either norm < 1e-12 (reading S13)
    if (na >= 1e-12 && nb >= 1e-12)
      dtc = (180.0 / kPi) * acos(clip1((Tn[3] / na) * (T[3] / nb) + (Tn[7] / na) * (T[7] / nb) + (Tn[11] / na) * (T[11] / nb)));
    p.dt[c] = dtc;
#pragma unroll
    for (int k = 0; k < 12; ++k) p.poses[12 * c + k] = Tn[k];
  }
  __syncthreads();   // dR/dt written by this CTA are visible to it after the barrier
  // 95th percentiles, linear interpolation at rank 0.95 (N-1) (reading S12)
  const double rank = 95.0 / 100.0 * (double)(N - 1);
  const int k0 = (int)floor(rank);
  const double fr = rank - (double)k0;
  select_two(p.dR, N, k0, &sel[0], &sel[1]);
  select_two(p.dt, N, k0, &sel[2], &sel[3]);
  __syncthreads();
  if (tid == 0) {
    const double r95 = (k0 + 1 < N) ? sel[0] + fr * (sel[1] - sel[0]) : sel[0];
    const double t95 = (k0 + 1 < N) ? sel[2] + fr * (sel[3] - sel[2]) : sel[2];
    const double th = r95 > t95 ? r95 : t95;
    p.theta[s] = th;
    p.loss_trace[s] = loss;
    st->loss = loss;
    int phase = st->phase;
    if (phase == 0) { if (converged(p.theta, s, p.w1, p.eps1, p.smooth)) phase = 1; }
    else if (phase == 1) { if (converged(p.theta, s, p.w2, p.eps2, p.smooth)) phase = 2; }
    st->phase = phase;
    st->step = s + 1;
    st->iters_done += 1;
    st->stopped = (s + 1 >= p.max_steps) || (p.early_stop && phase == 2);
  }
}

__global__ void k_begin_step_call(DevState* st, int max_steps, int early_stop) {
  st->iters_done = 0;
  st->stopped = (st->step >= max_steps) || (early_stop && st->phase == 2);
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

epo_status epo_launch_update(epo_ctx* ctx) {
  UpdParams p;
  p.poses = ctx->d_poses; p.grad = ctx->d_grad; p.loss_part = ctx->d_loss_part; p.m = ctx->d_m; p.v = ctx->d_v;
  p.dR = ctx->d_dR; p.dt = ctx->d_dt; p.theta = ctx->d_theta; p.loss_trace = ctx->d_loss_trace;
  p.state = ctx->d_state; p.N = ctx->N; p.P = ctx->P;
  p.lr_max = ctx->cfg.lr_max; p.beta1 = ctx->cfg.beta1; p.beta2 = ctx->cfg.beta2; p.adam_eps = ctx->cfg.adam_eps;
  p.eps1 = ctx->cfg.eps1; p.eps2 = ctx->cfg.eps2; p.warmup = ctx->cfg.warmup_steps; p.max_steps = ctx->cfg.max_steps;
  p.w1 = ctx->cfg.w1; p.w2 = ctx->cfg.w2; p.smooth = ctx->cfg.smooth_window; p.early_stop = ctx->cfg.early_stop;
  k_update<<<1, kUpdThreads, 0, ctx->stream>>>(p);
  ctx->launches += 1;
  EPO_CUDA(ctx, cudaGetLastError());
  return EPO_OK;
}

epo_status epo_launch_begin_step_call(epo_ctx* ctx) {
  k_begin_step_call<<<1, 1, 0, ctx->stream>>>(ctx->d_state, ctx->cfg.max_steps, ctx->cfg.early_stop);
  ctx->launches += 1;
  EPO_CUDA(ctx, cudaGetLastError());
  return EPO_OK;
}

void epo_launch_f64_to_f32(cudaStream_t st, const double* in, float* out, int64_t n) {
  if (n > 0) k_f64_to_f32<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(in, out, n);
}
void epo_launch_f32_to_f64(cudaStream_t st, const float* in, double* out, int64_t n) {
  if (n > 0) k_f32_to_f64<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(in, out, n);
}
