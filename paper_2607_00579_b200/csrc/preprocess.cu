// One-time preprocessing kernels (DESIGN.md rows a-P1..a-P3): edge-pixel compaction and the exact
// Euclidean distance transform.  Integer work; results are bit-reproducible.
//   PAPER.md:374-376 (Alg. 1 l.6)  "Canny edges, sub-sampled to <= E_max points / image"
//   PAPER.md:378-379 (Alg. 1 l.7), 396  "exact L2 distance transform [14]" kept on the GPU
#include <climits>
#include <cstring>

#include "epo_internal.h"

namespace {

constexpr int kWarpsPerBlock = 8;

// ---------------------------------------------------------------------------------------------
// generic single-CTA exclusive scan with carry (n up to a few million; one-time use)
// ---------------------------------------------------------------------------------------------
__global__ void k_exclusive_scan(const int32_t* __restrict__ in, int32_t* __restrict__ out, int64_t n,
                                 int32_t clamp_max /* <=0: none */) {
  __shared__ int32_t warp_sums[32];
  __shared__ int32_t carry_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) carry_s = 0;
  __syncthreads();
  for (int64_t base = 0; base < n; base += blockDim.x) {
    int64_t i = base + tid;
    int32_t v = (i < n) ? in[i] : 0;
    if (clamp_max > 0 && v > clamp_max) v = clamp_max;
    int32_t x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int32_t y = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= o) x += y;
    }
    if (lane == 31) warp_sums[warp] = x;
    __syncthreads();
    if (warp == 0) {
      int32_t w = (lane < (blockDim.x >> 5)) ? warp_sums[lane] : 0;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        int32_t y = __shfl_up_sync(0xffffffffu, w, o);
        if (lane >= o) w += y;
      }
      warp_sums[lane] = w;   // inclusive over warps
    }
    __syncthreads();
    int32_t carry = carry_s;
    int32_t prefix = carry + (warp > 0 ? warp_sums[warp - 1] : 0) + x - v;
    if (i < n) out[i] = prefix;
    __syncthreads();
    if (tid == blockDim.x - 1) carry_s = prefix + v;
    __syncthreads();
  }
  if (tid == 0) out[n] = carry_s;
}

// ---------------------------------------------------------------------------------------------
// a-P1  compaction: count per row -> scan -> ordered scatter (raster order: v ascending, then u)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ bool edge_kept(const uint8_t* e, const float* d, int64_t idx, float z_min) {
  float z = d[idx];
  return e[idx] != 0 && isfinite(z) && z > z_min;
}

__global__ void k_row_count(const uint8_t* __restrict__ edges, const float* __restrict__ depth, int64_t rows,
                            int W, float z_min, int32_t* __restrict__ row_cnt) {
  const int lane = threadIdx.x & 31;
  int64_t row = (int64_t)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  if (row >= rows) return;
  int cnt = 0;
  for (int x0 = 0; x0 < W; x0 += 32) {
    int x = x0 + lane;
    bool f = x < W && edge_kept(edges, depth, row * W + x, z_min);
    cnt += __popc(__ballot_sync(0xffffffffu, f));
  }
  if (lane == 0) row_cnt[row] = cnt;
}

__global__ void k_row_scatter(const uint8_t* __restrict__ edges, const float* __restrict__ depth, int64_t rows,
                              int W, int H, float z_min, const int32_t* __restrict__ row_off,
                              EdgeRec* __restrict__ rec) {
  const int lane = threadIdx.x & 31;
  int64_t row = (int64_t)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  if (row >= rows) return;
  int v = (int)(row % H);
  int32_t pos = row_off[row];
  for (int x0 = 0; x0 < W; x0 += 32) {
    int x = x0 + lane;
    bool f = x < W && edge_kept(edges, depth, row * W + x, z_min);
    unsigned m = __ballot_sync(0xffffffffu, f);
    if (f) {
      EdgeRec r;
      r.uv = (uint32_t)x | ((uint32_t)v << 16);
      r.z = depth[row * W + x];
      rec[pos + __popc(m & ((1u << lane) - 1u))] = r;
    }
    pos += __popc(m);
  }
}

// per-view totals from the row-level offsets: view_cnt[i] = row_off[(i+1)H] - row_off[iH]
__global__ void k_view_counts(const int32_t* __restrict__ row_off, int N, int H, int32_t* __restrict__ view_cnt) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < N) view_cnt[i] = row_off[(int64_t)(i + 1) * H] - row_off[(int64_t)i * H];
}
__global__ void k_view_offsets_from_rows(const int32_t* __restrict__ row_off, int N, int H, int32_t* __restrict__ off) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i <= N) off[i] = row_off[(int64_t)i * H];
}

// E_max sub-sampling (reading S6): keep entries floor(j n / e_max), j = 0..e_max-1, when n > e_max
__global__ void k_subsample(const EdgeRec* __restrict__ full, const int32_t* __restrict__ full_off,
                            const int32_t* __restrict__ out_off, int e_max, EdgeRec* __restrict__ out) {
  int view = blockIdx.y;
  int n = full_off[view + 1] - full_off[view];
  int m = out_off[view + 1] - out_off[view];
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < m; j += gridDim.x * blockDim.x) {
    int64_t k = (n > e_max) ? ((int64_t)j * n) / e_max : j;
    out[out_off[view] + j] = full[full_off[view] + k];
  }
}

// ---------------------------------------------------------------------------------------------
// a-P2  EDT pass 1: g[y][x] = min_{x' edge in row y} |x - x'|, sentinel W+H if the row has none.
// One warp per row: a forward max-scan of "last edge position" and a backward min-scan of "next".
// ---------------------------------------------------------------------------------------------
__global__ void k_edt_rows(const uint8_t* __restrict__ edges, int64_t rows, int W, int sentinel,
                           int32_t* __restrict__ g) {
  const int lane = threadIdx.x & 31;
  int64_t row = (int64_t)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  if (row >= rows) return;
  const uint8_t* e = edges + row * W;
  int32_t* out = g + row * W;
  const int NONE_L = INT_MIN / 2, NONE_R = INT_MAX / 2;
  int carry = NONE_L;
  for (int x0 = 0; x0 < W; x0 += 32) {
    int x = x0 + lane;
    int p = (x < W && e[x] != 0) ? x : NONE_L;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int q = __shfl_up_sync(0xffffffffu, p, o);
      if (lane >= o) p = max(p, q);
    }
    p = max(p, carry);
    carry = __shfl_sync(0xffffffffu, p, 31);
    if (x < W) out[x] = (p == NONE_L) ? sentinel : x - p;
  }
  carry = NONE_R;
  for (int x0 = ((W - 1) / 32) * 32; x0 >= 0; x0 -= 32) {
    int x = x0 + lane;
    int p = (x < W && e[x] != 0) ? x : NONE_R;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int q = __shfl_down_sync(0xffffffffu, p, o);
      if (lane + o < 32) p = min(p, q);
    }
    p = min(p, carry);
    carry = __shfl_sync(0xffffffffu, p, 0);
    if (x < W) {
      int dr = (p == NONE_R) ? sentinel : p - x;
      out[x] = min(out[x], dr);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// a-P3  EDT pass 2: d2[y][x] = min_{y'} g[y'][x]^2 + (y - y')^2 by the lower envelope of parabolas,
// with the integer-only separator of Meijster, Roerdink & Hesselink (2000): every comparison is an
// exact integer comparison, so d2 is the exact minimum.  One thread per column; its two stacks
// (s: parabola apex rows, t: first row where that parabola is the minimum) live in shared memory,
// laid out [stack index][column] so that threads never collide on a bank.
// DTF = correctly rounded fp32 sqrt of d2 (d2 < 2^24 exactly representable; else via fp64 sqrt).
// ---------------------------------------------------------------------------------------------
template <typename I>
__device__ __forceinline__ I parab(I x, I i, I gi) { return (x - i) * (x - i) + gi * gi; }

template <typename I>
__global__ void k_edt_cols(const int32_t* __restrict__ g, int W, int H, float* __restrict__ dtf,
                           __half* __restrict__ dtf_h) {
  extern __shared__ uint16_t stacks[];
  const int C = blockDim.x;
  uint16_t* s = stacks;                       // [H][C]
  uint16_t* t = stacks + (size_t)H * C;       // [H][C]
  const int col = blockIdx.x * C + threadIdx.x;
  const int view = blockIdx.y;
  if (col >= W) return;
  const int c = threadIdx.x;
  const int32_t* gv = g + (size_t)view * W * H + col;
  int q = 0;
  s[c] = 0; t[c] = 0;
  for (int u = 1; u < H; ++u) {
    I gu = (I)gv[(size_t)u * W];
    while (q >= 0) {
      I tq = (I)t[q * C + c], sq = (I)s[q * C + c];
      if (parab<I>(tq, sq, (I)gv[(size_t)sq * W]) > parab<I>(tq, (I)u, gu)) --q; else break;
    }
    if (q < 0) { q = 0; s[c] = (uint16_t)u; }
    else {
      I i = (I)s[q * C + c], gi = (I)gv[(size_t)i * W];
      I sep = ((I)u * u - i * i + gu * gu - gi * gi) / (2 * ((I)u - i));   // >= t[q] >= 0: floor == trunc
      I w = sep + 1;
      if (w < (I)H) { ++q; s[q * C + c] = (uint16_t)u; t[q * C + c] = (uint16_t)w; }
    }
  }
  for (int u = H - 1; u >= 0; --u) {
    I i = (I)s[q * C + c];
    I d2 = parab<I>((I)u, i, (I)gv[(size_t)i * W]);
    float r = (d2 < (I)(1 << 24)) ? __fsqrt_rn((float)d2) : (float)sqrt((double)d2);
    size_t o = ((size_t)view * H + u) * W + col;
    dtf[o] = r;
    if (dtf_h) dtf_h[o] = __float2half_rn(r);
    if (u == (int)t[q * C + c]) --q;
  }
}

// ---------------------------------------------------------------------------------------------
// a-2 hoisted: camera-frame point of every edge pixel, x_s = Z ((u - cx) (1/fx)), y_s likewise, z_s = Z
// (K and Z are not optimised on this path, so the point is iteration-invariant).
// The operation order is the one the fp32-position reading (P1) states.
// ---------------------------------------------------------------------------------------------
__global__ void k_make_points(const EdgeRec* __restrict__ rec, const int32_t* __restrict__ off,
                              const float* __restrict__ K, float4* __restrict__ pts) {
  const int view = blockIdx.y;
  const int lo = off[view], n = off[view + 1] - lo;
  const float ifx = 1.0f / K[4 * view], ify = 1.0f / K[4 * view + 1], cx = K[4 * view + 2], cy = K[4 * view + 3];
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const EdgeRec r = rec[lo + e];
    const float u = (float)(r.uv & 0xffffu), v = (float)(r.uv >> 16);
    pts[lo + e] = make_float4(r.z * ((u - cx) * ifx), r.z * ((v - cy) * ify), r.z, 0.f);
  }
}


}  // namespace

epo_status epo_build_edge_lists(epo_ctx* ctx, const uint8_t* d_edges_u8, const float* d_depth,
                                int32_t** out_off, EdgeRec** out_rec, int64_t* out_E,
                                std::vector<int32_t>* h_off) {
  const int N = ctx->N, W = ctx->W, H = ctx->H;
  const int64_t rows = (int64_t)N * H;
  cudaStream_t st = ctx->stream;
  int32_t *row_cnt = nullptr, *row_off = nullptr, *full_off = nullptr, *view_cnt = nullptr, *fin_off = nullptr;
  EdgeRec *full = nullptr, *fin = nullptr;
  epo_status rc = EPO_OK;
  auto cleanup = [&]() {
    cudaFree(row_cnt); cudaFree(row_off); cudaFree(view_cnt);
  };
#define PP_CUDA(call)                                                                                \
  do {                                                                                               \
    cudaError_t e_ = (call);                                                                         \
    if (e_ != cudaSuccess) {                                                                         \
      rc = epo_fail(ctx, e_ == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA,     \
                    "%s failed: %s", #call, cudaGetErrorString(e_));                                 \
      cleanup(); cudaFree(full_off); cudaFree(full); cudaFree(fin_off); cudaFree(fin);               \
      return rc;                                                                                     \
    }                                                                                                \
  } while (0)
  PP_CUDA(cudaMalloc(&row_cnt, (rows + 1) * sizeof(int32_t)));
  PP_CUDA(cudaMalloc(&row_off, (rows + 1) * sizeof(int32_t)));
  PP_CUDA(cudaMalloc(&view_cnt, (N + 1) * sizeof(int32_t)));
  PP_CUDA(cudaMalloc(&full_off, (N + 1) * sizeof(int32_t)));
  const int grid_rows = (int)((rows + kWarpsPerBlock - 1) / kWarpsPerBlock);
  k_row_count<<<grid_rows, kWarpsPerBlock * 32, 0, st>>>(d_edges_u8, d_depth, rows, W, ctx->cfg.z_min, row_cnt);
  k_exclusive_scan<<<1, 1024, 0, st>>>(row_cnt, row_off, rows, 0);
  k_view_offsets_from_rows<<<(N + 256) / 256, 256, 0, st>>>(row_off, N, H, full_off);
  ctx->launches += 3;
  std::vector<int32_t> hfull(N + 1);
  PP_CUDA(cudaMemcpyAsync(hfull.data(), full_off, (N + 1) * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  PP_CUDA(cudaStreamSynchronize(st));
  const int64_t Efull = hfull[N];
  PP_CUDA(cudaMalloc(&full, (size_t)(Efull > 0 ? Efull : 1) * sizeof(EdgeRec)));
  k_row_scatter<<<grid_rows, kWarpsPerBlock * 32, 0, st>>>(d_edges_u8, d_depth, rows, W, H, ctx->cfg.z_min, row_off, full);
  ctx->launches += 1;
  const int e_max = ctx->cfg.e_max;
  bool need_sub = false;
  if (e_max > 0)
    for (int i = 0; i < N; ++i) need_sub |= (hfull[i + 1] - hfull[i]) > e_max;
  if (!need_sub) {
    *out_off = full_off; *out_rec = full; *out_E = Efull; *h_off = hfull;
    full_off = nullptr; full = nullptr;
  } else {
    PP_CUDA(cudaMalloc(&fin_off, (N + 1) * sizeof(int32_t)));
    k_view_counts<<<(N + 255) / 256, 256, 0, st>>>(row_off, N, H, view_cnt);
    k_exclusive_scan<<<1, 1024, 0, st>>>(view_cnt, fin_off, N, e_max);
    std::vector<int32_t> hfin(N + 1);
    PP_CUDA(cudaMemcpyAsync(hfin.data(), fin_off, (N + 1) * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    PP_CUDA(cudaStreamSynchronize(st));
    PP_CUDA(cudaMalloc(&fin, (size_t)(hfin[N] > 0 ? hfin[N] : 1) * sizeof(EdgeRec)));
    dim3 grid((e_max + 255) / 256 > 64 ? 64 : (e_max + 255) / 256, N);
    k_subsample<<<grid, 256, 0, st>>>(full, full_off, fin_off, e_max, fin);
    ctx->launches += 3;
    PP_CUDA(cudaStreamSynchronize(st));
    cudaFree(full_off); cudaFree(full); full_off = nullptr; full = nullptr;
    *out_off = fin_off; *out_rec = fin; *out_E = hfin[N]; *h_off = hfin;
  }
  PP_CUDA(cudaGetLastError());
  cleanup();
#undef PP_CUDA
  return EPO_OK;
}

epo_status epo_build_dtf(epo_ctx* ctx, const uint8_t* d_edges_u8, float* d_dtf, __half* d_dtf_h) {
  const int N = ctx->N, W = ctx->W, H = ctx->H;
  const int64_t rows = (int64_t)N * H;
  cudaStream_t st = ctx->stream;
  int32_t* g = nullptr;
  EPO_CUDA(ctx, cudaMalloc(&g, (size_t)rows * W * sizeof(int32_t)));
  const int grid_rows = (int)((rows + kWarpsPerBlock - 1) / kWarpsPerBlock);
  k_edt_rows<<<grid_rows, kWarpsPerBlock * 32, 0, st>>>(d_edges_u8, rows, W, W + H, g);
  // columns per CTA: as many as fit the two uint16 stacks [H][C] in shared memory
  int C = 128;
  const size_t budget = 200 * 1024;
  while (C > 1 && (size_t)H * C * 2 * sizeof(uint16_t) > budget) C >>= 1;
  const size_t smem = (size_t)H * C * 2 * sizeof(uint16_t);
  if (smem > 227 * 1024) { cudaFree(g); return epo_fail(ctx, EPO_ERR_UNSUPPORTED, "height %d too large for the EDT column pass", H); }
  const bool wide = (int64_t)(W + H) * (W + H) + (int64_t)H * H >= (int64_t)INT32_MAX / 2;
  dim3 grid((W + C - 1) / C, N);
  cudaError_t e;
  if (wide) {
    e = cudaFuncSetAttribute(k_edt_cols<long long>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) k_edt_cols<long long><<<grid, C, smem, st>>>(g, W, H, d_dtf, d_dtf_h);
  } else {
    e = cudaFuncSetAttribute(k_edt_cols<int>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) k_edt_cols<int><<<grid, C, smem, st>>>(g, W, H, d_dtf, d_dtf_h);
  }
  ctx->launches += 2;
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(g);
  if (e != cudaSuccess) return epo_fail(ctx, EPO_ERR_CUDA, "EDT kernels failed: %s", cudaGetErrorString(e));
  return EPO_OK;
}

epo_status epo_build_points(epo_ctx* ctx, const float* d_K, const int32_t* d_off, const EdgeRec* d_rec, int64_t E,
                            const std::vector<int32_t>& h_off, float4** out_pts) {
  float4* pts = nullptr;
  // padded by one chunk of zeros: the fused kernel's tail lanes read past the end of a list and discard
  EPO_CUDA(ctx, cudaMalloc(&pts, (size_t)(E + kLgChunk) * sizeof(float4)));
  EPO_CUDA(ctx, cudaMemsetAsync(pts + E, 0, (size_t)kLgChunk * sizeof(float4), ctx->stream));
  int max_n = 1;
  for (int i = 0; i < ctx->N; ++i) max_n = h_off[i + 1] - h_off[i] > max_n ? h_off[i + 1] - h_off[i] : max_n;
  dim3 grid((max_n + 255) / 256, ctx->N);
  k_make_points<<<grid, 256, 0, ctx->stream>>>(d_rec, d_off, d_K, pts);
  ctx->launches += 1;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { cudaFree(pts); return epo_fail(ctx, EPO_ERR_CUDA, "k_make_points: %s", cudaGetErrorString(e)); }
  *out_pts = pts;
  return EPO_OK;
}

void epo_free_atlas(cudaArray_t atlas, cudaTextureObject_t tex) {
  if (tex) cudaDestroyTextureObject(tex);
  if (atlas) cudaFreeArray(atlas);
}

// Block-linear, gather-enabled copy of the distance fields: ONE 2-D CUDA array holding all views tiled in a
// grid (view i at texel offset ((i % cols) W, (i / cols) H)) behind one texture object.  The fused kernel
// fetches the 2x2 bilinear footprint with ONE tld4 (tex2Dgather) and applies the exact fp32 weights itself;
// the hardware's 8-bit-fraction filtering is never used.  A footprint never leaves its view (x0 <= W-2).
epo_status epo_build_atlas(epo_ctx* ctx, const float* d_dtf, const __half* d_dtf_h, cudaArray_t* atlas_out,
                           cudaTextureObject_t* tex_out, int* cols_out) {
  const int N = ctx->N, W = ctx->W, H = ctx->H;
  const bool half = d_dtf_h != nullptr;
  int cols = 32768 / W; if (cols < 1) cols = 1; if (cols > N) cols = N;
  const int rows = (N + cols - 1) / cols;
  if ((int64_t)rows * H > 65536 || (int64_t)cols * W > 131072)
    return epo_fail(ctx, EPO_ERR_UNSUPPORTED, "%d views of %dx%d do not fit one 2-D texture atlas", N, W, H);
  cudaChannelFormatDesc desc = half ? cudaCreateChannelDescHalf() : cudaCreateChannelDesc<float>();
  const size_t esz = half ? sizeof(__half) : sizeof(float);
  cudaArray_t arr = nullptr; cudaTextureObject_t t = 0;
  cudaError_t e = cudaMallocArray(&arr, &desc, (size_t)cols * W, (size_t)rows * H, cudaArrayTextureGather);
  for (int i = 0; i < N && e == cudaSuccess; ++i) {
    const void* src = half ? (const void*)(d_dtf_h + (size_t)i * W * H) : (const void*)(d_dtf + (size_t)i * W * H);
    e = cudaMemcpy2DToArrayAsync(arr, (size_t)(i % cols) * W * esz, (size_t)(i / cols) * H, src, W * esz, W * esz, H,
                                 cudaMemcpyDeviceToDevice, ctx->stream);
  }
  if (e == cudaSuccess) {
    cudaResourceDesc rd; memset(&rd, 0, sizeof(rd));
    rd.resType = cudaResourceTypeArray; rd.res.array.array = arr;
    cudaTextureDesc td; memset(&td, 0, sizeof(td));
    td.addressMode[0] = td.addressMode[1] = cudaAddressModeClamp;
    td.filterMode = cudaFilterModePoint; td.readMode = cudaReadModeElementType; td.normalizedCoords = 0;
    e = cudaCreateTextureObject(&t, &rd, &td, nullptr);
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) {
    epo_free_atlas(arr, t);
    return epo_fail(ctx, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, "distance-field atlas: %s",
                    cudaGetErrorString(e));
  }
  *atlas_out = arr; *tex_out = t; *cols_out = cols;
  return EPO_OK;
}
