// Edge extraction: "the edge map E_i via the Canny edge detector [4]" (Alg. 1
// l.6), in integer arithmetic on 8-bit images -- readings C1-C6 of DESIGN.md:
//   C1 binomial 5x5 smoothing, replicate border, (sum + 128) >> 8      C2 Sobel 3x3 on the smoothed image
//   C3 squared L2 magnitude                                            C4 four direction sectors, tan 22.5 ~ 13573/32768
//   C5 non-maximum suppression (m2 > low^2, > first neighbour, >= second; border pixels never)
//   C6 hysteresis: candidates 8-connected through candidates to a strong one (m2 > high^2)
// Three kernels: k_canny_gradient (smoothing + Sobel fused through shared memory, gradient packed as two int16),
// k_canny_suppress, and k_canny_grow, which spreads "edge" from strong pixels through candidates inside 32x32 tiles
// until the tile is stable; it is relaunched until no tile changed (a device flag read by the host: this is
// one-time preprocessing, not the loop).
#include "epo_internal.h"

namespace {

constexpr int kCT = 32;                 // tile edge

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

// one CTA (32 x 8 threads) per 32x32 tile: stage the tile with a halo of 3, smooth to a halo of 1, Sobel
__global__ void __launch_bounds__(256) k_canny_gradient(const uint8_t* __restrict__ img, int W, int H, int* __restrict__ grad) {
  __shared__ uint8_t sraw[kCT + 6][kCT + 6];
  __shared__ uint8_t sblur[kCT + 2][kCT + 2];
  const int n = blockIdx.z, x0 = blockIdx.x * kCT, y0 = blockIdx.y * kCT, tid = threadIdx.y * 32 + threadIdx.x;
  const uint8_t* im = img + (size_t)n * W * H;
  for (int i = tid; i < (kCT + 6) * (kCT + 6); i += 256) {
    const int ly = i / (kCT + 6), lx = i % (kCT + 6);
    sraw[ly][lx] = im[(size_t)clampi(y0 + ly - 3, 0, H - 1) * W + clampi(x0 + lx - 3, 0, W - 1)];
  }
  __syncthreads();
  // the smoothed value at an out-of-image halo position is the smoothed value of the clamped position (replicate
  // border applies to the smoothed image in the Sobel stage): compute it from the clamped centre
  for (int i = tid; i < (kCT + 2) * (kCT + 2); i += 256) {
    const int ly = i / (kCT + 2), lx = i % (kCT + 2);
    const int gy = clampi(y0 + ly - 1, 0, H - 1), gx = clampi(x0 + lx - 1, 0, W - 1);
    int acc = 0;
#pragma unroll
    for (int dy = -2; dy <= 2; ++dy) {
      const int wy = dy == 0 ? 6 : (dy == -1 || dy == 1 ? 4 : 1);
      const int sy = clampi(gy + dy, 0, H - 1) - y0 + 3;
#pragma unroll
      for (int dx = -2; dx <= 2; ++dx) {
        const int wx = dx == 0 ? 6 : (dx == -1 || dx == 1 ? 4 : 1);
        acc += wy * wx * (int)sraw[sy][clampi(gx + dx, 0, W - 1) - x0 + 3];
      }
    }
    sblur[ly][lx] = (uint8_t)((acc + 128) >> 8);
  }
  __syncthreads();
  for (int ly = threadIdx.y; ly < kCT; ly += 8) {
    const int x = x0 + threadIdx.x, y = y0 + ly, lx = threadIdx.x;
    if (x >= W || y >= H) continue;
    const int p00 = sblur[ly][lx], p01 = sblur[ly][lx + 1], p02 = sblur[ly][lx + 2];
    const int p10 = sblur[ly + 1][lx], p12 = sblur[ly + 1][lx + 2];
    const int p20 = sblur[ly + 2][lx], p21 = sblur[ly + 2][lx + 1], p22 = sblur[ly + 2][lx + 2];
    const int gx = (p02 - p00) + 2 * (p12 - p10) + (p22 - p20);
    const int gy = (p20 - p00) + 2 * (p21 - p01) + (p22 - p02);
    grad[((size_t)n * H + y) * W + x] = (int)((unsigned)(gx & 0xffff) | ((unsigned)gy << 16));      // |g| <= 1020: two int16
  }
}

__device__ __forceinline__ int mag2(int g) { const int gx = (short)(g & 0xffff), gy = g >> 16; return gx * gx + gy * gy; }

// cand: 0 no, 1 candidate, 2 strong
__global__ void k_canny_suppress(const int* __restrict__ grad, int W, int H, int lo2, int hi2, uint8_t* __restrict__ cand,
                                 uint8_t* __restrict__ edges) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y, n = blockIdx.z;
  if (x >= W) return;
  const size_t base = (size_t)n * W * H, i = base + (size_t)y * W + x;
  uint8_t c = 0;
  if (x > 0 && y > 0 && x < W - 1 && y < H - 1) {
    const int g = grad[i];
    const int gx = (short)(g & 0xffff), gy = g >> 16, ax = abs(gx), ay = abs(gy), m2 = gx * gx + gy * gy;
    if (m2 > lo2) {
      int dx1, dy1;
      if (ay * 32768 < ax * 13573) { dx1 = -1; dy1 = 0; }
      else if (ay * 13573 > ax * 32768) { dx1 = 0; dy1 = -1; }
      else if ((gx < 0) == (gy < 0)) { dx1 = -1; dy1 = -1; }
      else { dx1 = 1; dy1 = -1; }
      const int ma = mag2(grad[base + (size_t)(y + dy1) * W + (x + dx1)]), mb = mag2(grad[base + (size_t)(y - dy1) * W + (x - dx1)]);
      if (m2 > ma && m2 >= mb) c = m2 > hi2 ? 2 : 1;
    }
  }
  cand[i] = c;
  edges[i] = c == 2;
}

// grow "edge" through candidates inside a 32x32 tile (plus a read-only halo of 1) until the tile is stable
__global__ void __launch_bounds__(256) k_canny_grow(const uint8_t* __restrict__ cand, uint8_t* __restrict__ edges, int W, int H,
                                                    int* __restrict__ changed) {
  __shared__ uint8_t se[kCT + 2][kCT + 2];
  __shared__ uint8_t sc[kCT][kCT];
  __shared__ int s_changed, s_any;
  const int n = blockIdx.z, x0 = blockIdx.x * kCT, y0 = blockIdx.y * kCT, tid = threadIdx.y * 32 + threadIdx.x;
  const size_t base = (size_t)n * W * H;
  for (int i = tid; i < (kCT + 2) * (kCT + 2); i += 256) {
    const int ly = i / (kCT + 2), lx = i % (kCT + 2), y = y0 + ly - 1, x = x0 + lx - 1;
    se[ly][lx] = (x >= 0 && y >= 0 && x < W && y < H) ? edges[base + (size_t)y * W + x] : 0;
  }
  for (int i = tid; i < kCT * kCT; i += 256) {
    const int ly = i / kCT, lx = i % kCT, y = y0 + ly, x = x0 + lx;
    sc[ly][lx] = (x < W && y < H) ? cand[base + (size_t)y * W + x] : 0;
  }
  if (tid == 0) s_any = 0;
  __syncthreads();
  while (true) {
    if (tid == 0) s_changed = 0;
    __syncthreads();
    for (int ly = threadIdx.y; ly < kCT; ly += 8) {
      const int lx = threadIdx.x;
      if (sc[ly][lx] && !se[ly + 1][lx + 1]) {
        const int near = se[ly][lx] | se[ly][lx + 1] | se[ly][lx + 2] | se[ly + 1][lx] | se[ly + 1][lx + 2] |
                         se[ly + 2][lx] | se[ly + 2][lx + 1] | se[ly + 2][lx + 2];
        if (near) { se[ly + 1][lx + 1] = 1; s_changed = 1; }     // monotone: racing reads only delay a pixel by a sweep
      }
    }
    __syncthreads();
    if (!s_changed) break;
    if (tid == 0) s_any = 1;
    __syncthreads();
  }
  if (s_any) {
    for (int ly = threadIdx.y; ly < kCT; ly += 8) {
      const int x = x0 + threadIdx.x, y = y0 + ly;
      if (x < W && y < H && se[ly + 1][threadIdx.x + 1]) edges[base + (size_t)y * W + x] = 1;
    }
    if (tid == 0) *changed = 1;
  }
}

}  // namespace

// colour -> grey (reading C7): BT.601 luma in 8-bit fixed point, interleaved RGB in, one thread per pixel
__global__ void k_rgb_to_grey(const uint8_t* __restrict__ rgb, uint8_t* __restrict__ grey, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) grey[i] = (uint8_t)((77 * (int)rgb[3 * i] + 150 * (int)rgb[3 * i + 1] + 29 * (int)rgb[3 * i + 2] + 128) >> 8);
}

epo_status epo_run_rgb_to_grey(epo_ctx* ctx, const uint8_t* d_rgb, uint8_t* d_grey) {
  const long long n = (long long)ctx->N * ctx->W * ctx->H;
  k_rgb_to_grey<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(d_rgb, d_grey, n);
  ctx->launches += 1;
  EPO_CUDA(ctx, cudaGetLastError());
  return EPO_OK;
}

epo_status epo_run_canny(epo_ctx* ctx, const uint8_t* d_img, int low, int high, uint8_t* d_edges) {
  const int N = ctx->N, W = ctx->W, H = ctx->H;
  cudaStream_t st = ctx->stream;
  const size_t px = (size_t)N * W * H;
  int* grad = nullptr; uint8_t* cand = nullptr; int* changed = nullptr;
  cudaError_t e = epo_dmalloc(ctx, &grad, px * sizeof(int));
  if (e == cudaSuccess) e = epo_dmalloc(ctx, &cand, px);
  if (e == cudaSuccess) e = epo_dmalloc(ctx, &changed, sizeof(int));
  if (e == cudaSuccess) {
    const dim3 tiles((W + kCT - 1) / kCT, (H + kCT - 1) / kCT, N);
    k_canny_gradient<<<tiles, dim3(32, 8), 0, st>>>(d_img, W, H, grad);
    k_canny_suppress<<<dim3((W + 127) / 128, H, N), 128, 0, st>>>(grad, W, H, low * low, high * high, cand, d_edges);
    ctx->launches += 2;
    for (int it = 0; it < W + H && e == cudaSuccess; ++it) {     // at most the longest possible chain of tiles
      int h_changed = 0;
      e = cudaMemsetAsync(changed, 0, sizeof(int), st);
      if (e == cudaSuccess) { k_canny_grow<<<tiles, dim3(32, 8), 0, st>>>(cand, d_edges, W, H, changed); ctx->launches += 1; }
      if (e == cudaSuccess) e = cudaMemcpyAsync(&h_changed, changed, sizeof(int), cudaMemcpyDeviceToHost, st);
      if (e == cudaSuccess) e = cudaStreamSynchronize(st);
      if (!h_changed) break;
    }
    if (e == cudaSuccess) e = cudaGetLastError();
  }
  epo_dfree(ctx, grad); epo_dfree(ctx, cand); epo_dfree(ctx, changed);
  if (e != cudaSuccess)
    return epo_fail(ctx, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, "edge extraction: %s", cudaGetErrorString(e));
  return EPO_OK;
}
