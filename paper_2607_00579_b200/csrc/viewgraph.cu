// Viewgraph estimation by exhaustive cycle-consistent reprojection, once per problem:
//   PAPER.md:66-70 Eq. 2   p_{i->j} = pi(K_i, K_j, P_i, P_j, Z_i; p), projected back to p_{i->j->i}; a pair is valid
//                          if sufficiently many pixels have || p - p_{i->j->i} ||_2 < tau
//   PAPER.md:117           at least 12.5 % of the reprojected points below tau = 3.0 px
//   PAPER.md:380-384, 396  BuildViewgraph: for every candidate pair a kernel projects a grid of source pixels into
//                          the target view and back
// Readings V1-V8: grid u = stride/2 + a stride; usable = finite depth > z_min; landing must be in front
// of and inside view j; view j's depth at the NEAREST pixel; back-projection from the sub-pixel landing position;
// strict threshold on the squared error; a pair needs min_frac in BOTH directions; positions in binary32 with the
// operation order of the loss path (reading P1), relative poses formed in double.
#include "epo_internal.h"

namespace {

constexpr int kVgThreads = 128;

struct VgParams {
  const float* K;
  const double* poses;
  const float* depth;      // [N][H][W]
  int2* counts;            // [N][N] {consistent, usable} of the cycle i -> j -> i
  int N, W, H, stride;
  float tau2, z_min;
};

// one CTA per ordered pair (i, j): threads stride over the grid points of view i
__global__ void __launch_bounds__(kVgThreads) k_vg_counts(const VgParams p) {
  __shared__ float sA[12], sB[12];
  __shared__ int sred[kVgThreads / 32][2];
  const int i = blockIdx.x / p.N, j = blockIdx.x % p.N, tid = threadIdx.x;
  if (i == j) { if (tid == 0) p.counts[blockIdx.x] = make_int2(0, 0); return; }
  if (tid < 12) sA[tid] = (float)rel_pose_entry(p.poses + 12 * (size_t)i, p.poses + 12 * (size_t)j, tid);          // i -> j
  else if (tid >= 32 && tid < 44) sB[tid - 32] = (float)rel_pose_entry(p.poses + 12 * (size_t)j, p.poses + 12 * (size_t)i, tid - 32);
  __syncthreads();
  const float fxi = p.K[4 * i], fyi = p.K[4 * i + 1], cxi = p.K[4 * i + 2], cyi = p.K[4 * i + 3];
  const float fxj = p.K[4 * j], fyj = p.K[4 * j + 1], cxj = p.K[4 * j + 2], cyj = p.K[4 * j + 3];
  const float ifxi = __fdiv_rn(1.0f, fxi), ifyi = __fdiv_rn(1.0f, fyi), ifxj = __fdiv_rn(1.0f, fxj), ifyj = __fdiv_rn(1.0f, fyj);
  const float xmax = (float)(p.W - 1), ymax = (float)(p.H - 1);
  const float* __restrict__ Zi_map = p.depth + (size_t)i * p.W * p.H;
  const float* __restrict__ Zj_map = p.depth + (size_t)j * p.W * p.H;
  const int h0 = p.stride / 2;
  const int gx = p.W > h0 ? (p.W - h0 + p.stride - 1) / p.stride : 0, gy = p.H > h0 ? (p.H - h0 + p.stride - 1) / p.stride : 0;
  int cons = 0, usable = 0;
  for (int g = tid; g < gx * gy; g += kVgThreads) {
    const int ui = h0 + (g % gx) * p.stride, vi = h0 + (g / gx) * p.stride;
    const float Zi = __ldg(Zi_map + (size_t)vi * p.W + ui);
    if (!(isfinite(Zi) && Zi > p.z_min)) continue;
    ++usable;
    const float u = (float)ui, v = (float)vi;
    const float xs = __fmul_rn(Zi, __fmul_rn(u - cxi, ifxi)), ys = __fmul_rn(Zi, __fmul_rn(v - cyi, ifyi));
    const float X = fmaf(sA[0], xs, fmaf(sA[1], ys, fmaf(sA[2], Zi, sA[3])));
    const float Y = fmaf(sA[4], xs, fmaf(sA[5], ys, fmaf(sA[6], Zi, sA[7])));
    const float Z = fmaf(sA[8], xs, fmaf(sA[9], ys, fmaf(sA[10], Zi, sA[11])));
    if (!(Z > p.z_min)) continue;
    const float iz = __fdiv_rn(1.0f, Z);
    const float x = fmaf(__fmul_rn(fxj, X), iz, cxj), y = fmaf(__fmul_rn(fyj, Y), iz, cyj);
    if (!(x >= 0.0f && x <= xmax && y >= 0.0f && y <= ymax)) continue;
    const int xn = (int)floorf(__fadd_rn(x, 0.5f)), yn = (int)floorf(__fadd_rn(y, 0.5f));
    const float Zj = __ldg(Zj_map + (size_t)yn * p.W + xn);
    if (!(isfinite(Zj) && Zj > p.z_min)) continue;
    const float xb = __fmul_rn(Zj, __fmul_rn(x - cxj, ifxj)), yb = __fmul_rn(Zj, __fmul_rn(y - cyj, ifyj));
    const float X2 = fmaf(sB[0], xb, fmaf(sB[1], yb, fmaf(sB[2], Zj, sB[3])));
    const float Y2 = fmaf(sB[4], xb, fmaf(sB[5], yb, fmaf(sB[6], Zj, sB[7])));
    const float Z2 = fmaf(sB[8], xb, fmaf(sB[9], yb, fmaf(sB[10], Zj, sB[11])));
    if (!(Z2 > p.z_min)) continue;
    const float iz2 = __fdiv_rn(1.0f, Z2);
    const float x2 = fmaf(__fmul_rn(fxi, X2), iz2, cxi), y2 = fmaf(__fmul_rn(fyi, Y2), iz2, cyi);
    const float dx = x2 - u, dy = y2 - v;
    cons += fmaf(dx, dx, __fmul_rn(dy, dy)) < p.tau2;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    cons += __shfl_xor_sync(0xffffffffu, cons, o);
    usable += __shfl_xor_sync(0xffffffffu, usable, o);
  }
  if ((tid & 31) == 0) { sred[tid >> 5][0] = cons; sred[tid >> 5][1] = usable; }
  __syncthreads();
  if (tid == 0) {
    int c = 0, n = 0;
#pragma unroll
    for (int w = 0; w < kVgThreads / 32; ++w) { c += sred[w][0]; n += sred[w][1]; }
    p.counts[blockIdx.x] = make_int2(c, n);
  }
}

// ordered emission: unordered pair {i, j}, i < j, is valid iff both directions keep >= min_frac of their usable
// points; valid pairs are written as (i, j), (j, i) in ascending (i, j) order (one CTA, block scans of 1024 cells)
constexpr int kEmitThreads = 1024;
__global__ void __launch_bounds__(kEmitThreads) k_vg_emit(const int2* __restrict__ counts, int N, double min_frac,
                                                          int2* __restrict__ pairs, long long* __restrict__ n_out) {
  __shared__ int wtot[32];
  __shared__ long long s_carry;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) s_carry = 0;
  __syncthreads();
  const long long cells = (long long)N * N;
  for (long long base = 0; base < cells; base += kEmitThreads) {
    const long long c = base + tid;
    int ok = 0, i = 0, j = 0;
    if (c < cells) {
      i = (int)(c / N); j = (int)(c % N);
      if (i < j) {
        const int2 a = counts[c], b = counts[(long long)j * N + i];
        ok = a.y > 0 && b.y > 0 && (double)a.x >= min_frac * (double)a.y && (double)b.x >= min_frac * (double)b.y;
      }
    }
    int x = ok;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) wtot[warp] = x;
    __syncthreads();
    if (warp == 0) {
      int w = wtot[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += y; }
      wtot[lane] = w;
    }
    __syncthreads();
    const long long before = s_carry + (warp > 0 ? wtot[warp - 1] : 0) + x - ok;
    if (ok && pairs) { pairs[2 * before] = make_int2(i, j); pairs[2 * before + 1] = make_int2(j, i); }
    __syncthreads();
    if (tid == 0) s_carry += wtot[31];
    __syncthreads();
  }
  if (tid == 0) *n_out = 2 * s_carry;
}

}  // namespace

epo_status epo_launch_viewgraph(epo_ctx* ctx, int stride, float tau, float min_frac, int2* d_counts, int2* d_pairs,
                                long long* d_n) {
  VgParams p;
  p.K = ctx->d_K; p.poses = ctx->d_poses; p.depth = ctx->d_depth; p.counts = d_counts;
  p.N = ctx->N; p.W = ctx->W; p.H = ctx->H; p.stride = stride; p.tau2 = tau * tau; p.z_min = ctx->cfg.z_min;
  k_vg_counts<<<(unsigned)(ctx->N * ctx->N), kVgThreads, 0, ctx->stream>>>(p);
  k_vg_emit<<<1, kEmitThreads, 0, ctx->stream>>>(d_counts, ctx->N, (double)min_frac, d_pairs, d_n);
  ctx->launches += 2;
  EPO_CUDA(ctx, cudaGetLastError());
  return EPO_OK;
}
