// The joint loop's variables (Eq. 4-5, 121, 429-431): a focal scale per
// camera, f_c = f0_c (1 + gamma_c), optimised from the first iteration ("the first phase ... drives updates to the
// camera intrinsics K and poses P"), and an affine depth per listed edge pixel, Z_e = Z0_e alpha_e + beta_e, optimised
// in iterations that start in phase >= 1 ("the depth optimizer steps only once c_pose holds").  AdamW [28] with the
// loop's learning-rate schedule, decay towards the identity values (readings J4-J7).  After the step
// the intrinsics and the hoisted camera-frame points are rebuilt for the next iteration.
#include <algorithm>

#include "epo_internal.h"

namespace {

struct JointParams {
  const DevState* state;
  const double* sched;
  const double* glogf;       // [N]
  const float* gz;           // [E] point order
  const float* K0;           // [N][4]
  float* K;                  // [N][4] current
  double* gamma;             // [3][N]
  double* ab;                // [3][E][2]
  const float* z0;           // [E]
  float4* pts;               // [E]
  const int32_t* off;        // [N+1]
  long long E;
  int N, W, H;
  double beta1, beta2, adam_eps, wd;
  int force;                 // rebuild the points from the current variables without stepping (epo_joint_reset)
};

// c1 = 1 - beta1^t, c2 = 1 - beta2^t of the group's step count t (the same for every variable of a launch)
__device__ __forceinline__ double adamw_step(double p, double g, double* m, double* v, double c1, double c2, double lr,
                                             const JointParams& q, double p_id) {
  p -= lr * q.wd * (p - p_id);
  const double mm = q.beta1 * *m + (1.0 - q.beta1) * g, vv = q.beta2 * *v + (1.0 - q.beta2) * g * g;
  *m = mm; *v = vv;
  return p - lr * (mm / c1) / (sqrt(vv / c2) + q.adam_eps);
}

// gamma_c: step number t = s + 1 of iteration s; d L / d gamma = (d L / d ln f) / (1 + gamma)
__global__ void k_joint_cams(const JointParams q) {
  if (!q.state->joint_pending) return;
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= q.N) return;
  const int s = q.state->step - 1;
  const double lr = q.sched[4 * (size_t)s];
  double g = q.gamma[c];
  const double c1 = 1.0 - pow(q.beta1, (double)(s + 1)), c2 = 1.0 - pow(q.beta2, (double)(s + 1));
  g = adamw_step(g, q.glogf[c] / (1.0 + g), q.gamma + q.N + c, q.gamma + 2 * q.N + c, c1, c2, lr, q, 0.0);
  q.gamma[c] = g;
  q.K[4 * c] = (float)((double)q.K0[4 * c] * (1.0 + g));
  q.K[4 * c + 1] = (float)((double)q.K0[4 * c + 1] * (1.0 + g));
}

// alpha_e, beta_e (iterations that started in phase >= 1), then the point of every listed edge pixel with the new K, Z
__global__ void k_joint_points(const JointParams q) {
  if (!q.force && !q.state->joint_pending) return;
  const int view = blockIdx.y;
  const int lo = q.off[view], n = q.off[view + 1] - lo;
  const int s = q.state->step - 1;
  const bool depth_on = !q.force && q.state->phase_prev >= 1;
  const int t = s - q.state->phase1_step;            // 1 for the first iteration that starts in phase 1
  const double lr = depth_on ? q.sched[4 * (size_t)s] : 0.0;
  const double c1 = depth_on ? 1.0 - pow(q.beta1, (double)t) : 1.0, c2 = depth_on ? 1.0 - pow(q.beta2, (double)t) : 1.0;
  const float ifx = 1.0f / q.K[4 * view], ify = 1.0f / q.K[4 * view + 1], cx = q.K[4 * view + 2], cy = q.K[4 * view + 3];
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const size_t i = (size_t)lo + e;
    float4 pt = q.pts[i];
    const int pix = __float_as_int(pt.w);
    double a = q.ab[2 * i], b = q.ab[2 * i + 1];
    const double Z0 = (double)q.z0[i];
    if (depth_on) {
      const double g = (double)q.gz[i];
      const size_t E2 = 2 * (size_t)q.E;
      a = adamw_step(a, Z0 * g, q.ab + E2 + 2 * i, q.ab + 2 * E2 + 2 * i, c1, c2, lr, q, 1.0);
      b = adamw_step(b, g, q.ab + E2 + 2 * i + 1, q.ab + 2 * E2 + 2 * i + 1, c1, c2, lr, q, 0.0);
      q.ab[2 * i] = a; q.ab[2 * i + 1] = b;
    }
    const float Z = (float)(Z0 * a + b);
    const float u = (float)(pix % q.W), v = (float)(pix / q.W);
    pt.x = Z * ((u - cx) * ifx); pt.y = Z * ((v - cy) * ify); pt.z = Z;     // operation order of reading P1
    q.pts[i] = pt;
  }
}

__global__ void k_joint_init(float4* __restrict__ pts, float* __restrict__ z0, double* __restrict__ ab, long long E, int save_z0) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= E) return;
  if (save_z0) z0[i] = pts[i].z;
  ab[2 * i] = 1.0; ab[2 * i + 1] = 0.0;
  ab[2 * E + 2 * i] = ab[2 * E + 2 * i + 1] = 0.0;
  ab[4 * E + 2 * i] = ab[4 * E + 2 * i + 1] = 0.0;
}

// d L / d Z in point order -> the dense [N][H][W] map of the API (zeroed by the caller)
__global__ void k_joint_scatter_gz(const float4* __restrict__ pts, const float* __restrict__ g, const int32_t* __restrict__ off,
                                   int W, int H, float* __restrict__ map) {
  const int view = blockIdx.y;
  const int lo = off[view], n = off[view + 1] - lo;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x)
    map[(size_t)view * W * H + __float_as_int(pts[(size_t)lo + e].w)] = g[(size_t)lo + e];
}

// dense maps of alpha (1 off the lists) and beta (0 off the lists)
__global__ void k_joint_fill(double* __restrict__ a_map, double* __restrict__ b_map, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { a_map[i] = 1.0; b_map[i] = 0.0; }
}
__global__ void k_joint_scatter(const float4* __restrict__ pts, const double* __restrict__ ab, const int32_t* __restrict__ off,
                                int W, int H, double* __restrict__ a_map, double* __restrict__ b_map) {
  const int view = blockIdx.y;
  const int lo = off[view], n = off[view + 1] - lo;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const size_t i = (size_t)lo + e, o = (size_t)view * W * H + __float_as_int(pts[i].w);
    a_map[o] = ab[2 * i]; b_map[o] = ab[2 * i + 1];
  }
}

JointParams make_params(epo_ctx* c) {
  JointParams q;
  q.state = c->d_state; q.sched = c->d_sched; q.glogf = c->d_glogf; q.gz = c->d_gz; q.K0 = c->d_K0; q.K = c->d_K;
  q.gamma = c->d_gamma; q.ab = c->d_ab; q.z0 = c->d_z0; q.pts = c->d_pts; q.off = c->d_edge_off; q.E = c->E;
  q.N = c->N; q.W = c->W; q.H = c->H;
  q.beta1 = c->cfg.beta1; q.beta2 = c->cfg.beta2; q.adam_eps = c->cfg.adam_eps; q.wd = c->cfg.weight_decay;
  q.force = 0;
  return q;
}

int max_list(const epo_ctx* c) {
  int m = 1;
  for (int i = 0; i < c->N; ++i) m = std::max(m, c->h_edge_off[i + 1] - c->h_edge_off[i]);
  return m;
}

}  // namespace

void epo_joint_free(epo_ctx* c) {
  epo_dfree(c, c->d_poses_prev); epo_dfree(c, c->d_K0); epo_dfree(c, c->d_gamma); epo_dfree(c, c->d_ab);
  epo_dfree(c, c->d_z0); epo_dfree(c, c->d_gz); epo_dfree(c, c->d_glogf);
  c->d_poses_prev = nullptr; c->d_K0 = nullptr; c->d_gamma = nullptr; c->d_ab = nullptr; c->d_z0 = nullptr;
  c->d_gz = nullptr; c->d_glogf = nullptr;
}

epo_status epo_joint_alloc(epo_ctx* c) {
  epo_joint_free(c);
  if (!c->cfg.joint_phase) return EPO_OK;
  const size_t N = (size_t)c->N, E = (size_t)(c->E > 0 ? c->E : 1);
  cudaError_t e = epo_dmalloc(c, &c->d_poses_prev, N * 12 * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_K0, N * 4 * sizeof(float));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_gamma, 3 * N * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_ab, 6 * E * sizeof(double));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_z0, E * sizeof(float));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_gz, E * sizeof(float));
  if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_glogf, N * sizeof(double));
  if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_K0, c->d_K, N * 4 * sizeof(float), cudaMemcpyDeviceToDevice, c->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->d_gamma, 0, 3 * N * sizeof(double), c->stream);
  if (e == cudaSuccess && c->E > 0) {
    k_joint_init<<<(unsigned)((c->E + 255) / 256), 256, 0, c->stream>>>(c->d_pts, c->d_z0, c->d_ab, c->E, 1);
    c->launches += 1;
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    epo_joint_free(c);
    return epo_fail(c, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, "joint phase: %s", cudaGetErrorString(e));
  }
  return EPO_OK;
}

// back to the identity: gamma = 0, alpha = 1, beta = 0, zero moments, K and points as given
epo_status epo_joint_reset(epo_ctx* c) {
  if (!c->cfg.joint_phase || !c->d_gamma) return EPO_OK;
  EPO_CUDA(c, cudaMemsetAsync(c->d_gamma, 0, 3 * (size_t)c->N * sizeof(double), c->stream));
  EPO_CUDA(c, cudaMemcpyAsync(c->d_K, c->d_K0, (size_t)c->N * 4 * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
  if (c->E > 0) {
    k_joint_init<<<(unsigned)((c->E + 255) / 256), 256, 0, c->stream>>>(c->d_pts, c->d_z0, c->d_ab, c->E, 0);
    JointParams q = make_params(c);
    q.force = 1;                                   // the points again from (K0, Z0)
    const int m = max_list(c);
    dim3 grid((unsigned)std::min((m + 255) / 256, 64), (unsigned)c->N);
    k_joint_points<<<grid, 256, 0, c->stream>>>(q);
    c->launches += 2;
    EPO_TRY(epo_launch_pack_points(c, c->d_pts, c->d_edge_off, c->packed));
  }
  EPO_CUDA(c, cudaGetLastError());
  return EPO_OK;
}

epo_status epo_joint_reset_moments(epo_ctx* c) {
  if (!c->cfg.joint_phase || !c->d_gamma) return EPO_OK;
  EPO_CUDA(c, cudaMemsetAsync(c->d_gamma + c->N, 0, 2 * (size_t)c->N * sizeof(double), c->stream));
  if (c->E > 0) EPO_CUDA(c, cudaMemsetAsync(c->d_ab + 2 * (size_t)c->E, 0, 4 * (size_t)c->E * sizeof(double), c->stream));
  return EPO_OK;
}

epo_status epo_launch_joint_update(epo_ctx* c) {
  const JointParams q = make_params(c);
  k_joint_cams<<<(c->N + 127) / 128, 128, 0, c->stream>>>(q);
  const int m = max_list(c);
  dim3 grid((unsigned)std::min((m + 255) / 256, 64), (unsigned)c->N);
  k_joint_points<<<grid, 256, 0, c->stream>>>(q);
  c->launches += 2;
  EPO_TRY(epo_launch_pack_points(c, c->d_pts, c->d_edge_off, c->packed));    // the fused kernel's copy of the points
  EPO_CUDA(c, cudaGetLastError());
  return EPO_OK;
}

epo_status epo_joint_scatter_gz(epo_ctx* c, const float* d_g_points, float* d_map) {
  const int m = max_list(c);
  dim3 grid((unsigned)std::min((m + 255) / 256, 64), (unsigned)c->N);
  k_joint_scatter_gz<<<grid, 256, 0, c->stream>>>(c->d_pts, d_g_points, c->d_edge_off, c->W, c->H, d_map);
  c->launches += 1;
  EPO_CUDA(c, cudaGetLastError());
  return EPO_OK;
}

epo_status epo_joint_export(epo_ctx* c, double* d_gamma_out, double* d_alpha_map, double* d_beta_map) {
  const long long n = (long long)c->N * c->W * c->H;
  if (d_gamma_out) EPO_CUDA(c, cudaMemcpyAsync(d_gamma_out, c->d_gamma, (size_t)c->N * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  if (d_alpha_map && d_beta_map) {
    k_joint_fill<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(d_alpha_map, d_beta_map, n);
    const int m = max_list(c);
    dim3 grid((unsigned)std::min((m + 255) / 256, 64), (unsigned)c->N);
    k_joint_scatter<<<grid, 256, 0, c->stream>>>(c->d_pts, c->d_ab, c->d_edge_off, c->W, c->H, d_alpha_map, d_beta_map);
    c->launches += 2;
  }
  EPO_CUDA(c, cudaGetLastError());
  return EPO_OK;
}
