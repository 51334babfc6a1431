// The joint loop's depth variables (Eq. 5, 121, 429-431): an affine depth per
// listed edge pixel, Z_e = Z0_e alpha_e + beta_e, optimised in iterations that START in phase >= 1 ("the depth optimizer
// steps only once c_pose holds"), AdamW [28] with the loop's learning-rate schedule and decay towards the identity
// (readings J4-J7).  The focal scale gamma_c (Eq. 4) is stepped per camera in k_finish (update.cu).
//
// One kernel per iteration, k_joint_points, thread = one slot (two edge pixels) of the packed point layout (EpoPacked):
//   d L / d Z_e = -(1 / z_e) sum over the pairs p with source(e) = s, in ascending canonical order, of
//                 (a . t_ts)_{e,p} / (P n_p)          [(a . t_ts) is what the fused kernel's joint mode stored per slot
//                                                       and work item; n_p is k_finish's valid count of the pair]
//   AdamW on (alpha_e, beta_e) with d L / d alpha = Z0 d L / d Z, d L / d beta = d L / d Z
//   the hoisted point of the pixel again from the new intrinsics and Z = fp32(Z0 alpha + beta)
// A point's pairs are summed by ONE thread in a fixed order: no atomics, bit-reproducible (the pass this replaces
// added 15 M float atomics per iteration).  All joint state lives in slot order, two pixels per slot.
#include <algorithm>

#include "epo_internal.h"

namespace {

struct JointParams {
  const DevState* state;
  const double* sched;
  const float* K;            // [N][4] current intrinsics (k_finish has stepped gamma already)
  const float2* dz;          // [n_work][chunk / 2]
  const int32_t *pair_valid, *src_off, *src_inc, *work_off;
  const uint8_t* sel_flag;   // pair sub-sampling: this iteration's subset (canonical order), else nullptr
  const int32_t* pk_off;     // [N+1] samples
  const int2* pix;           // [slots]
  const float2* z0;          // [slots]
  double4* ab;               // [slots]
  float4* abm;               // [slots][2]
  float2* xyz;               // packed points
  double inv_P;              // 1 / (pairs the mean runs over)
  int W, chunk;
  double beta1, beta2, adam_eps, wd;
  int force;                 // rebuild the points from the current variables without stepping (epo_joint_reset)
  int32_t* depth_stepped;    // [1] see epo_ctx::d_depth_stepped
  long long n_slots, n_work; // sizes EPO_CHECK tests indices against
};

// one AdamW step of a scalar; c1 = 1 - beta1^t, c2 = 1 - beta2^t of the group's step count t; moments in fp32 (a
// relative 6e-8 on a step of ~lr: far below the variables' own resolution)
__device__ __forceinline__ double adamw_step(double p, double g, float* m, float* v, double c1, double c2, double lr,
                                             const JointParams& q, double p_id) {
  p -= lr * q.wd * (p - p_id);
  const double mm = q.beta1 * (double)*m + (1.0 - q.beta1) * g, vv = q.beta2 * (double)*v + (1.0 - q.beta2) * g * g;
  *m = (float)mm; *v = (float)vv;
  return p - lr * (mm / c1) / (sqrt(vv / c2) + q.adam_eps);
}

// sum over the pairs whose source is `view` of (stored value of slot `j` of the view) / (P n_p), both samples
__device__ __forceinline__ double2 gather_dz(const float2* __restrict__ dz, const int32_t* __restrict__ pair_valid,
                                             const int32_t* __restrict__ src_off, const int32_t* __restrict__ src_inc,
                                             const int32_t* __restrict__ work_off, const uint8_t* __restrict__ sel_flag,
                                             int view, int j, int chunk, double inv_P) {
  double ga = 0.0, gb = 0.0;
  const int half = chunk / 2, it = j / half, so = j % half;
  for (int k = src_off[view]; k < src_off[view + 1]; ++k) {
    const int p = src_inc[k];
    if (sel_flag != nullptr && sel_flag[p] == 0) continue;
    const int n = __ldcg(pair_valid + p);
    if (n <= 0) continue;
    const float2 v = __ldcg(dz + (size_t)(work_off[p] + it) * half + so);
    const double w = inv_P / (double)n;
    ga += w * (double)v.x; gb += w * (double)v.y;
  }
  return make_double2(ga, gb);
}

constexpr int kJointPairsSmem = 512;   // pairs per source view whose weights k_joint_points keeps in shared memory

__global__ void k_joint_points(const JointParams q) {
  const int view = blockIdx.y;
  const int slots = (q.pk_off[view + 1] - q.pk_off[view]) / 2;
  const size_t base = (size_t)q.pk_off[view] / 2;
  cudaTriggerProgrammaticLaunchCompletion();
  cudaGridDependencySynchronize();                   // k_finish: valid counts, gamma -> K, phase, joint_pending
  if (!q.force && !q.state->joint_pending) return;
  const int s = q.state->step - 1;
  const bool depth_on = !q.force && q.state->phase_prev >= 1;
  const int t = s - q.state->phase1_step;            // 1 for the first iteration that starts in phase 1
  const double lr = depth_on ? q.sched[4 * (size_t)s] : 0.0;
  const double c1 = depth_on ? 1.0 - pow(q.beta1, (double)t) : 1.0, c2 = depth_on ? 1.0 - pow(q.beta2, (double)t) : 1.0;
  const float ifx = 1.0f / __ldcg(q.K + 4 * view), ify = 1.0f / __ldcg(q.K + 4 * view + 1);
  const float cx = __ldcg(q.K + 4 * view + 2), cy = __ldcg(q.K + 4 * view + 3);
  // until the first depth step alpha = 1, beta = 0 everywhere and Z = Z0 exactly: the stored points are the ones built
  // from (K0, Z0), and the focal step is a per-camera scaling of x_s and y_s that the fused kernel folds into the first
  // two columns of R_ts (lossgrad.cu) -- nothing to rewrite, this launch returns.  From the first depth step on the
  // points are rebuilt here in every iteration.
  const bool identity = __ldcg(q.depth_stepped) == 0 && !depth_on;
  if (identity && !q.force) return;
  if (depth_on && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) *q.depth_stepped = 1;
  // the pairs this view is the source of, once per CTA: weight 1 / (P n_p) (0: not in this iteration's subset, or no
  // valid sample) and first work item -- the per-pixel sums below then issue independent loads only (the same terms
  // in the same ascending order as gather_dz: identical results)
  __shared__ double s_w[kJointPairsSmem];
  __shared__ int s_wo[kJointPairsSmem];
  // (the pair tables are read only when the depth steps: a forced rebuild may run before any pair list exists, with
  // src_off == nullptr -- epo_set_views -> epo_reset)
  const int k0 = depth_on ? q.src_off[view] : 0, np = depth_on ? q.src_off[view + 1] - k0 : 0;
  const bool pairs_in_smem = depth_on && np <= kJointPairsSmem;
  if (pairs_in_smem) {
    for (int i = threadIdx.x; i < np; i += blockDim.x) {
      const int p = q.src_inc[k0 + i];
      const int n = __ldcg(q.pair_valid + p);
      const bool skip = (q.sel_flag != nullptr && q.sel_flag[p] == 0) || n <= 0;
      s_w[i] = skip ? 0.0 : q.inv_P / (double)n;
      s_wo[i] = q.work_off[p];
    }
    __syncthreads();
  }
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < slots; j += gridDim.x * blockDim.x) {
    const size_t sl = base + j, o = sl / kLgThreads * (3 * kLgThreads) + sl % kLgThreads;
    EPO_CHECK((long long)sl < q.n_slots);
    const int2 px = q.pix[sl];
    const float2 Z0 = q.z0[sl];
    double4 ab = identity ? make_double4(1.0, 0.0, 1.0, 0.0) : q.ab[sl];
    if (depth_on) {
      const float2 zc = q.xyz[o + 2 * kLgThreads];  // the depth the loss of this iteration was evaluated at
      double2 g;
      if (pairs_in_smem) {
        const int half = q.chunk / 2, it = j / half, so = j % half;
        double ga = 0.0, gb = 0.0;
        for (int i = 0; i < np; ++i) {
          const double w = s_w[i];
          if (w == 0.0) continue;
          EPO_CHECK(s_wo[i] + it < q.n_work);
          const float2 v = __ldcg(q.dz + (size_t)(s_wo[i] + it) * half + so);
          ga += w * (double)v.x; gb += w * (double)v.y;
        }
        g = make_double2(ga, gb);
      } else {
        g = gather_dz(q.dz, q.pair_valid, q.src_off, q.src_inc, q.work_off, q.sel_flag, view, j, q.chunk, q.inv_P);
      }
      float4 ma = q.abm[2 * sl], mb = q.abm[2 * sl + 1];
      if (px.x >= 0) {
        const double gz = -g.x / (double)zc.x;
        ab.x = adamw_step(ab.x, (double)Z0.x * gz, &ma.x, &ma.y, c1, c2, lr, q, 1.0);
        ab.y = adamw_step(ab.y, gz, &ma.z, &ma.w, c1, c2, lr, q, 0.0);
      }
      if (px.y >= 0) {
        const double gz = -g.y / (double)zc.y;
        ab.z = adamw_step(ab.z, (double)Z0.y * gz, &mb.x, &mb.y, c1, c2, lr, q, 1.0);
        ab.w = adamw_step(ab.w, gz, &mb.z, &mb.w, c1, c2, lr, q, 0.0);
      }
      q.ab[sl] = ab; q.abm[2 * sl] = ma; q.abm[2 * sl + 1] = mb;
    }
    // the hoisted points again: x_s = Z ((u - cx) (1 / fx)), y_s likewise (the operation order of k_tile_points)
    float2 X = make_float2(0.f, 0.f), Y = X, Zn = X;
    if (px.x >= 0) {
      const float Z = (float)((double)Z0.x * ab.x + ab.y), u = (float)(px.x % q.W), v = (float)(px.x / q.W);
      X.x = Z * ((u - cx) * ifx); Y.x = Z * ((v - cy) * ify); Zn.x = Z;
    }
    if (px.y >= 0) {
      const float Z = (float)((double)Z0.y * ab.z + ab.w), u = (float)(px.y % q.W), v = (float)(px.y / q.W);
      X.y = Z * ((u - cx) * ifx); Y.y = Z * ((v - cy) * ify); Zn.y = Z;
    }
    q.xyz[o] = X; q.xyz[o + kLgThreads] = Y; q.xyz[o + 2 * kLgThreads] = Zn;
  }
}

// identity variables, zero moments; Z0 saved from the packed points (first call after epo_set_views)
__global__ void k_joint_init(const float2* __restrict__ xyz, float2* __restrict__ z0, double4* __restrict__ ab,
                             float4* __restrict__ abm, long long slots, int save_z0) {
  const long long sl = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (sl >= slots) return;
  if (save_z0) z0[sl] = xyz[sl / kLgThreads * (3 * kLgThreads) + sl % kLgThreads + 2 * kLgThreads];
  ab[sl] = make_double4(1.0, 0.0, 1.0, 0.0);
  abm[2 * sl] = make_float4(0.f, 0.f, 0.f, 0.f); abm[2 * sl + 1] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// d L / d Z of every listed edge pixel into the dense [N][H][W] map (zeroed by the caller), from one joint evaluation
__global__ void k_joint_gather_gz(const float2* __restrict__ dz, const int32_t* __restrict__ pair_valid,
                                  const int32_t* __restrict__ src_off, const int32_t* __restrict__ src_inc,
                                  const int32_t* __restrict__ work_off, const int32_t* __restrict__ pk_off,
                                  const int2* __restrict__ pix, const float2* __restrict__ xyz, int chunk, double inv_P,
                                  size_t px_per_view, float* __restrict__ map) {
  const int view = blockIdx.y;
  const int slots = (pk_off[view + 1] - pk_off[view]) / 2;
  const size_t base = (size_t)pk_off[view] / 2;
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < slots; j += gridDim.x * blockDim.x) {
    const size_t sl = base + j;
    const int2 px = pix[sl];
    if (px.x < 0 && px.y < 0) continue;
    const float2 z = xyz[sl / kLgThreads * (3 * kLgThreads) + sl % kLgThreads + 2 * kLgThreads];
    const double2 g = gather_dz(dz, pair_valid, src_off, src_inc, work_off, nullptr, view, j, chunk, inv_P);
    if (px.x >= 0) map[(size_t)view * px_per_view + px.x] = (float)(-g.x / (double)z.x);
    if (px.y >= 0) map[(size_t)view * px_per_view + px.y] = (float)(-g.y / (double)z.y);
  }
}

// dense maps of alpha (1 off the lists) and beta (0 off the lists)
__global__ void k_joint_fill(double* __restrict__ a_map, double* __restrict__ b_map, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { a_map[i] = 1.0; b_map[i] = 0.0; }
}
__global__ void k_joint_scatter(const int2* __restrict__ pix, const double4* __restrict__ ab, const int32_t* __restrict__ pk_off,
                                size_t px_per_view, double* __restrict__ a_map, double* __restrict__ b_map) {
  const int view = blockIdx.y;
  const int slots = (pk_off[view + 1] - pk_off[view]) / 2;
  const size_t base = (size_t)pk_off[view] / 2;
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < slots; j += gridDim.x * blockDim.x) {
    const int2 px = pix[base + j];
    const double4 v = ab[base + j];
    if (px.x >= 0) { a_map[(size_t)view * px_per_view + px.x] = v.x; b_map[(size_t)view * px_per_view + px.x] = v.y; }
    if (px.y >= 0) { a_map[(size_t)view * px_per_view + px.y] = v.z; b_map[(size_t)view * px_per_view + px.y] = v.w; }
  }
}

size_t n_slots(const epo_ctx* c) { return c->packed.h_off.empty() ? 0 : (size_t)c->packed.h_off[c->N] / 2; }

dim3 view_grid(const epo_ctx* c) {
  int m = 1;
  for (int i = 0; i < c->N; ++i) m = std::max(m, (c->packed.h_off[i + 1] - c->packed.h_off[i]) / 2);
  return dim3((unsigned)std::min((m + 255) / 256, 64), (unsigned)c->N);
}

JointParams make_params(epo_ctx* c, bool subset) {
  JointParams q;
  q.state = c->d_state; q.sched = c->d_sched; q.K = c->d_K; q.dz = c->d_dz; q.pair_valid = c->d_pair_valid;
  q.src_off = c->d_src_off; q.src_inc = c->d_src_inc; q.work_off = c->d_work_off; q.sel_flag = subset ? c->d_sel_flag : nullptr;
  q.pk_off = c->packed.d_off; q.pix = c->packed.pix; q.z0 = c->d_z0; q.ab = c->d_ab; q.abm = c->d_abm; q.xyz = c->packed.xyz;
  q.inv_P = 1.0 / (double)(subset ? (int64_t)c->cfg.pair_budget : (c->P > 0 ? c->P : 1));
  q.W = c->W; q.chunk = c->lg_chunk;
  q.beta1 = c->cfg.beta1; q.beta2 = c->cfg.beta2; q.adam_eps = c->cfg.adam_eps; q.wd = c->cfg.weight_decay;
  q.force = 0; q.depth_stepped = c->d_depth_stepped; q.n_slots = (long long)n_slots(c); q.n_work = (long long)c->n_work;
  return q;
}

}  // namespace

void epo_joint_free(epo_ctx* c) {
  epo_dfree(c, c->d_K0); epo_dfree(c, c->d_gamma); epo_dfree(c, c->d_ab); epo_dfree(c, c->d_abm);
  epo_dfree(c, c->d_z0); epo_dfree(c, c->d_glogf); epo_dfree(c, c->d_depth_stepped);
  c->d_depth_stepped = nullptr; c->d_K0 = nullptr; c->d_gamma = nullptr; c->d_ab = nullptr; c->d_abm = nullptr; c->d_z0 = nullptr; c->d_glogf = nullptr;
}

// d_glogf exists in every context (epo_loss_grad_joint works without cfg.joint_phase); the variables only with it
epo_status epo_joint_alloc(epo_ctx* c) {
  epo_joint_free(c);
  const size_t N = (size_t)c->N, S = std::max<size_t>(n_slots(c), 1);
  cudaError_t e = epo_dmalloc(c, &c->d_glogf, N * sizeof(double));
  if (e == cudaSuccess && c->cfg.joint_phase) {
    e = epo_dmalloc(c, &c->d_K0, N * 4 * sizeof(float));
    if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_gamma, 3 * N * sizeof(double));
    if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_ab, S * sizeof(double4));
    if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_abm, 2 * S * sizeof(float4));
    if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_z0, S * sizeof(float2));
    if (e == cudaSuccess) e = epo_dmalloc(c, &c->d_depth_stepped, sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemsetAsync(c->d_depth_stepped, 0, sizeof(int32_t), c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_K0, c->d_K, N * 4 * sizeof(float), cudaMemcpyDeviceToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->d_gamma, 0, 3 * N * sizeof(double), c->stream);
    if (e == cudaSuccess && n_slots(c) > 0) {
      k_joint_init<<<(unsigned)((n_slots(c) + 255) / 256), 256, 0, c->stream>>>(c->packed.xyz, c->d_z0, c->d_ab, c->d_abm,
                                                                                 (long long)n_slots(c), 1);
      c->launches += 1;
      e = cudaGetLastError();
    }
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
  EPO_CUDA(c, cudaMemsetAsync(c->d_depth_stepped, 0, sizeof(int32_t), c->stream));
  if (n_slots(c) > 0) {
    k_joint_init<<<(unsigned)((n_slots(c) + 255) / 256), 256, 0, c->stream>>>(c->packed.xyz, c->d_z0, c->d_ab, c->d_abm,
                                                                               (long long)n_slots(c), 0);
    JointParams q = make_params(c, false);
    q.force = 1;                                   // the points again from (K0, Z0)
    k_joint_points<<<view_grid(c), 256, 0, c->stream>>>(q);
    c->launches += 2;
  }
  c->static_dirty = true;
  EPO_CUDA(c, cudaGetLastError());
  return EPO_OK;
}

epo_status epo_joint_reset_moments(epo_ctx* c) {
  if (!c->cfg.joint_phase || !c->d_gamma) return EPO_OK;
  EPO_CUDA(c, cudaMemsetAsync(c->d_gamma + c->N, 0, 2 * (size_t)c->N * sizeof(double), c->stream));
  if (n_slots(c) > 0) EPO_CUDA(c, cudaMemsetAsync(c->d_abm, 0, 2 * n_slots(c) * sizeof(float4), c->stream));
  return EPO_OK;
}

epo_status epo_launch_joint_points(epo_ctx* c, bool subset) {
  if (n_slots(c) == 0) return EPO_OK;
  const JointParams q = make_params(c, subset);
  cudaLaunchConfig_t lc = {};
  lc.gridDim = view_grid(c); lc.blockDim = dim3(256); lc.dynamicSmemBytes = 0; lc.stream = c->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at; lc.numAttrs = c->pdl ? 1 : 0;
  EPO_CUDA(c, cudaLaunchKernelEx(&lc, k_joint_points, q));
  c->launches += 1;
  return EPO_OK;
}

epo_status epo_joint_gather_gz(epo_ctx* c, const float2* d_dz, float* d_map) {
  const size_t px = (size_t)c->W * c->H;
  EPO_CUDA(c, cudaMemsetAsync(d_map, 0, (size_t)c->N * px * sizeof(float), c->stream));
  if (n_slots(c) == 0) return EPO_OK;
  k_joint_gather_gz<<<view_grid(c), 256, 0, c->stream>>>(d_dz, c->d_pair_valid, c->d_src_off, c->d_src_inc, c->d_work_off,
                                                          c->packed.d_off, c->packed.pix, c->packed.xyz, c->lg_chunk,
                                                          1.0 / (double)(c->P > 0 ? c->P : 1), px, d_map);
  c->launches += 1;
  EPO_CUDA(c, cudaGetLastError());
  return EPO_OK;
}

epo_status epo_joint_export(epo_ctx* c, double* d_gamma_out, double* d_alpha_map, double* d_beta_map) {
  const long long n = (long long)c->N * c->W * c->H;
  if (d_gamma_out) EPO_CUDA(c, cudaMemcpyAsync(d_gamma_out, c->d_gamma, (size_t)c->N * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  if (d_alpha_map && d_beta_map) {
    k_joint_fill<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(d_alpha_map, d_beta_map, n);
    c->launches += 1;
    if (n_slots(c) > 0) {
      k_joint_scatter<<<view_grid(c), 256, 0, c->stream>>>(c->packed.pix, c->d_ab, c->packed.d_off, (size_t)c->W * c->H,
                                                            d_alpha_map, d_beta_map);
      c->launches += 1;
    }
  }
  EPO_CUDA(c, cudaGetLastError());
  return EPO_OK;
}
