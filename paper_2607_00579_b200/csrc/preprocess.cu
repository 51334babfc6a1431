// One-time preprocessing kernels (DESIGN.md rows a-P1..a-P3): edge-pixel compaction and the exact
// Euclidean distance transform.  Integer work; results are bit-reproducible.
//   PAPER.md:374-376 (Alg. 1 l.6)  "Canny edges, sub-sampled to <= E_max points / image"
//   PAPER.md:378-379 (Alg. 1 l.7), 396  "exact L2 distance transform [14]" kept on the GPU
#include <climits>
#include <cstdarg>
#include <cstring>

#include <algorithm>
#include <mutex>

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
// a-P3  EDT pass 2: d2[y][x] = min_{y'} g[y'][x]^2 + (y - y')^2, exactly, in integers.
// One thread per PIXEL (not per column): a CTA stages the g values of a strip of 32 columns x H rows in
// shared memory (coalesced 128-byte rows), then every pixel searches outwards dy = 1, 2, ... in both
// directions and stops as soon as dy^2 >= the best value so far -- no farther row can improve it, so the
// minimum is exact.  The search length is the distance itself (a few to a few tens of rows at the paper's
// edge densities, at most H), all H x W pixels of a view run in parallel, and lanes of a warp are
// neighbouring columns of one row, whose distances differ by at most 31 (the field is 1-Lipschitz), so a warp
// stays converged.  An out-of-range row is clamped to the border row: its candidate only over-estimates
// that row's true candidate, so the minimum is unchanged and the loop is branch-free.
// DTF = correctly rounded fp32 sqrt of d2 (d2 < 2^24 is exact in fp32; else via fp64 sqrt), written
// straight into the block-linear atlas (surface store; fp16 = RNE of the fp32), and -- fp32 format -- d2 itself,
// saturated at 255, into the one-byte atlas the fused kernel samples (see EpoAtlas).
// ---------------------------------------------------------------------------------------------
constexpr int kEdtStrip = 32, kEdtWarps = 8;

template <typename I, bool kStage>
__global__ void __launch_bounds__(kEdtStrip * kEdtWarps)
k_edt_cols(const int32_t* __restrict__ g, int W, int H, cudaSurfaceObject_t atlas, cudaSurfaceObject_t atlas8,
           int atlas_cols, int half) {
  extern __shared__ int32_t sg[];             // [H][32] when kStage
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int view = blockIdx.y, x = blockIdx.x * kEdtStrip + lane;
  const bool in = x < W;
  const int32_t* gv = g + (size_t)view * W * H + (in ? x : W - 1);
  if (kStage) {
    for (int y = warp; y < H; y += kEdtWarps) sg[y * kEdtStrip + lane] = gv[(size_t)y * W];
    __syncthreads();
  }
  auto G = [&](int y) -> I { return kStage ? (I)sg[y * kEdtStrip + lane] : (I)__ldg(gv + (size_t)y * W); };
  const int ox = (view % atlas_cols) * W + x, oy = (view / atlas_cols) * H;
  for (int y = warp; y < H; y += kEdtWarps) {
    const I g0 = G(y);
    I best = g0 * g0;
    const int dmax = max(y, H - 1 - y);
    for (int dy = 1; dy <= dmax; ++dy) {
      const I dd = (I)dy * dy;
      if (dd >= best) break;
      const I a = G(max(y - dy, 0)), b = G(min(y + dy, H - 1));
      const I m = a < b ? a : b;
      const I c = m * m + dd;
      best = c < best ? c : best;
    }
    if (in) {
      const float r = (best < (I)(1 << 24)) ? __fsqrt_rn((float)best) : (float)sqrt((double)best);
      if (half) surf2Dwrite(__half_as_ushort(__float2half_rn(r)), atlas, ox * 2, oy + y);
      else {
        surf2Dwrite(r, atlas, ox * 4, oy + y);
        surf2Dwrite((unsigned char)(best < (I)255 ? best : (I)255), atlas8, ox, oy + y);   // exact d^2, saturated
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// a-2 hoisted: camera-frame point of every edge pixel, x_s = Z ((u - cx) (1/fx)), y_s likewise, z_s = Z
// (K and Z are not optimised on this path, so the point is iteration-invariant).
// The operation order is the one the fp32-position reading (P1) states.
// ---------------------------------------------------------------------------------------------
__global__ void k_make_points(const EdgeRec* __restrict__ rec, const int32_t* __restrict__ off,
                              const float* __restrict__ K, int W, float4* __restrict__ pts) {
  const int view = blockIdx.y;
  const int lo = off[view], n = off[view + 1] - lo;
  const float ifx = 1.0f / K[4 * view], ify = 1.0f / K[4 * view + 1], cx = K[4 * view + 2], cy = K[4 * view + 3];
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const EdgeRec r = rec[lo + e];
    const float u = (float)(r.uv & 0xffffu), v = (float)(r.uv >> 16);
    pts[lo + e] = make_float4(r.z * ((u - cx) * ifx), r.z * ((v - cy) * ify), r.z,
                              __int_as_float((int)(r.uv >> 16) * W + (int)(r.uv & 0xffffu)));   // .w: pixel index (joint phase)
  }
}

// The same points in TILE-MAJOR order (the order the fused kernel consumes; the canonical raster list above is
// what the API exposes).  Each view is cut into kTile x kTile pixel tiles, tiles in raster order, pixels in
// raster order inside a tile: 32 consecutive points then follow one or two edge curves through a compact patch
// of the source image, so the lanes of a warp gather from neighbouring texels of the target field (shared
// sectors inside one tld4, a compact L1 working set) instead of from 32 unrelated places along an image row.
// Only the summation order changes.  One warp per (view, tile): two tile rows (32 pixels) per step.
#ifndef EPO_TILE
#define EPO_TILE 16
#endif
constexpr int kTile = EPO_TILE;   // power of two, 4..32

__device__ __forceinline__ bool tile_pixel(int W, int H, int tx, int ty, int step, int lane, int* u, int* v) {
  *u = tx * kTile + (lane & (kTile - 1));
  *v = ty * kTile + step * (32 / kTile) + lane / kTile;
  return *u < W && *v < H;
}

__global__ void k_tile_count(const uint8_t* __restrict__ edges, const float* __restrict__ depth, int N, int W, int H,
                             int tiles_x, int tiles_y, float z_min, int32_t* __restrict__ tile_cnt) {
  const int lane = threadIdx.x & 31;
  const int64_t wid = (int64_t)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  const int64_t per_view = (int64_t)tiles_x * tiles_y;
  if (wid >= per_view * N) return;
  const int view = (int)(wid / per_view), t = (int)(wid % per_view), tx = t % tiles_x, ty = t / tiles_x;
  int cnt = 0;
  for (int step = 0; step < kTile * kTile / 32; ++step) {
    int u, v;
    const bool f = tile_pixel(W, H, tx, ty, step, lane, &u, &v) &&
                   edge_kept(edges, depth, ((int64_t)view * H + v) * W + u, z_min);
    cnt += __popc(__ballot_sync(0xffffffffu, f));
  }
  if (lane == 0) tile_cnt[wid] = cnt;
}

__global__ void k_tile_points(const uint8_t* __restrict__ edges, const float* __restrict__ depth, int N, int W, int H,
                              int tiles_x, int tiles_y, float z_min, const int32_t* __restrict__ tile_off,
                              const float* __restrict__ K, float4* __restrict__ pts) {
  const int lane = threadIdx.x & 31;
  const int64_t wid = (int64_t)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  const int64_t per_view = (int64_t)tiles_x * tiles_y;
  if (wid >= per_view * N) return;
  const int view = (int)(wid / per_view), t = (int)(wid % per_view), tx = t % tiles_x, ty = t / tiles_x;
  const float ifx = 1.0f / K[4 * view], ify = 1.0f / K[4 * view + 1], cx = K[4 * view + 2], cy = K[4 * view + 3];
  int32_t pos = tile_off[wid];
  for (int step = 0; step < kTile * kTile / 32; ++step) {
    int u, v;
    const bool in = tile_pixel(W, H, tx, ty, step, lane, &u, &v);
    const int64_t idx = ((int64_t)view * H + v) * W + u;
    const bool f = in && edge_kept(edges, depth, idx, z_min);
    const unsigned m = __ballot_sync(0xffffffffu, f);
    if (f) {
      const float z = depth[idx];
      pts[pos + __popc(m & ((1u << lane) - 1u))] =
          make_float4(z * (((float)u - cx) * ifx), z * (((float)v - cy) * ify), z, __int_as_float(v * W + u));   // .w: pixel index
    }
    pos += __popc(m);
  }
}


// tile-major float4 points (.w = pixel index) -> the packed layout (EpoPacked): thread = one slot (two samples) of a view
__global__ void k_pack_points(const float4* __restrict__ pts, const int32_t* __restrict__ edge_off,
                              const int32_t* __restrict__ pk_off, float2* __restrict__ xyz, int2* __restrict__ pix) {
  const int view = blockIdx.y;
  const int lo = edge_off[view], n = edge_off[view + 1] - lo;
  const int slots = (pk_off[view + 1] - pk_off[view]) / 2;
  const size_t base = (size_t)pk_off[view] / 2;
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < slots; j += gridDim.x * blockDim.x) {
    const int a = 64 * (j >> 5) + (j & 31), b = a + 32;
    const float4 none = make_float4(0.f, 0.f, 0.f, __int_as_float(-1));
    const float4 pa = a < n ? pts[(size_t)lo + a] : none, pb = b < n ? pts[(size_t)lo + b] : none;
    const size_t s = base + j, o = s / kLgThreads * (3 * kLgThreads) + s % kLgThreads;
    xyz[o] = make_float2(pa.x, pb.x); xyz[o + kLgThreads] = make_float2(pa.y, pb.y); xyz[o + 2 * kLgThreads] = make_float2(pa.z, pb.z);
    pix[s] = make_int2(__float_as_int(pa.w), __float_as_int(pb.w));
  }
}

}  // namespace

static epo_status alloc_packed(epo_ctx* ctx, const std::vector<int32_t>& h_edge_off, EpoPacked* out) {
  EpoPacked pk = {nullptr, nullptr, nullptr, {}};
  const int N = ctx->N;
  pk.h_off.assign((size_t)N + 1, 0);
  for (int i = 0; i < N; ++i) pk.h_off[i + 1] = pk.h_off[i] + (h_edge_off[i + 1] - h_edge_off[i] + kLgPass - 1) / kLgPass * kLgPass;
  const size_t slots = (size_t)pk.h_off[N] / 2, used = slots * 3, all = used + (size_t)kLgPad / 2 * 3;     // float2 entries
  cudaError_t e = epo_dmalloc(ctx, &pk.xyz, all * sizeof(float2));
  if (e == cudaSuccess) e = epo_dmalloc(ctx, &pk.pix, (slots ? slots : 1) * sizeof(int2));
  if (e == cudaSuccess) e = epo_dmalloc(ctx, &pk.d_off, ((size_t)N + 1) * sizeof(int32_t));
  if (e == cudaSuccess) e = cudaMemsetAsync(pk.xyz + used, 0, (all - used) * sizeof(float2), ctx->stream);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(pk.d_off, pk.h_off.data(), ((size_t)N + 1) * sizeof(int32_t), cudaMemcpyHostToDevice, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);      // h_off is copied from this frame
  if (e != cudaSuccess) {
    epo_free_packed(ctx, &pk);
    return epo_fail(ctx, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, "packed points: %s", cudaGetErrorString(e));
  }
  *out = pk;
  return EPO_OK;
}

void epo_free_packed(epo_ctx* ctx, EpoPacked* pk) {
  epo_dfree(ctx, pk->xyz); epo_dfree(ctx, pk->pix); epo_dfree(ctx, pk->d_off);
  pk->xyz = nullptr; pk->pix = nullptr; pk->d_off = nullptr; pk->h_off.clear();
}

epo_status epo_build_edge_lists(epo_ctx* ctx, const uint8_t* d_edges_u8, const float* d_depth,
                                int32_t** out_off, EdgeRec** out_rec, int64_t* out_E,
                                std::vector<int32_t>* h_off, bool* out_subsampled) {
  const int N = ctx->N, W = ctx->W, H = ctx->H;
  const int64_t rows = (int64_t)N * H;
  cudaStream_t st = ctx->stream;
  int32_t *row_cnt = nullptr, *row_off = nullptr, *full_off = nullptr, *view_cnt = nullptr, *fin_off = nullptr;
  EdgeRec *full = nullptr, *fin = nullptr;
  epo_status rc = EPO_OK;
  auto cleanup = [&]() {
    epo_dfree(ctx, row_cnt); epo_dfree(ctx, row_off); epo_dfree(ctx, view_cnt);
  };
#define PP_CUDA(call)                                                                                \
  do {                                                                                               \
    cudaError_t e_ = (call);                                                                         \
    if (e_ != cudaSuccess) {                                                                         \
      rc = epo_fail(ctx, e_ == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA,     \
                    "%s failed: %s", #call, cudaGetErrorString(e_));                                 \
      cleanup(); epo_dfree(ctx, full_off); epo_dfree(ctx, full); epo_dfree(ctx, fin_off); epo_dfree(ctx, fin);               \
      return rc;                                                                                     \
    }                                                                                                \
  } while (0)
  PP_CUDA(epo_dmalloc(ctx, &row_cnt, (rows + 1) * sizeof(int32_t)));
  PP_CUDA(epo_dmalloc(ctx, &row_off, (rows + 1) * sizeof(int32_t)));
  PP_CUDA(epo_dmalloc(ctx, &view_cnt, (N + 1) * sizeof(int32_t)));
  PP_CUDA(epo_dmalloc(ctx, &full_off, (N + 1) * sizeof(int32_t)));
  const int grid_rows = (int)((rows + kWarpsPerBlock - 1) / kWarpsPerBlock);
  k_row_count<<<grid_rows, kWarpsPerBlock * 32, 0, st>>>(d_edges_u8, d_depth, rows, W, ctx->cfg.z_min, row_cnt);
  k_exclusive_scan<<<1, 1024, 0, st>>>(row_cnt, row_off, rows, 0);
  k_view_offsets_from_rows<<<(N + 256) / 256, 256, 0, st>>>(row_off, N, H, full_off);
  ctx->launches += 3;
  std::vector<int32_t> hfull(N + 1);
  PP_CUDA(cudaMemcpyAsync(hfull.data(), full_off, (N + 1) * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  PP_CUDA(cudaStreamSynchronize(st));
  const int64_t Efull = hfull[N];
  PP_CUDA(epo_dmalloc(ctx, &full, (size_t)(Efull > 0 ? Efull : 1) * sizeof(EdgeRec)));
  k_row_scatter<<<grid_rows, kWarpsPerBlock * 32, 0, st>>>(d_edges_u8, d_depth, rows, W, H, ctx->cfg.z_min, row_off, full);
  ctx->launches += 1;
  const int e_max = ctx->cfg.e_max;
  bool need_sub = false;
  if (e_max > 0)
    for (int i = 0; i < N; ++i) need_sub |= (hfull[i + 1] - hfull[i]) > e_max;
  *out_subsampled = need_sub;
  if (!need_sub) {
    *out_off = full_off; *out_rec = full; *out_E = Efull; *h_off = hfull;
    full_off = nullptr; full = nullptr;
  } else {
    PP_CUDA(epo_dmalloc(ctx, &fin_off, (N + 1) * sizeof(int32_t)));
    k_view_counts<<<(N + 255) / 256, 256, 0, st>>>(row_off, N, H, view_cnt);
    k_exclusive_scan<<<1, 1024, 0, st>>>(view_cnt, fin_off, N, e_max);
    std::vector<int32_t> hfin(N + 1);
    PP_CUDA(cudaMemcpyAsync(hfin.data(), fin_off, (N + 1) * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    PP_CUDA(cudaStreamSynchronize(st));
    PP_CUDA(epo_dmalloc(ctx, &fin, (size_t)(hfin[N] > 0 ? hfin[N] : 1) * sizeof(EdgeRec)));
    dim3 grid((e_max + 255) / 256 > 64 ? 64 : (e_max + 255) / 256, N);
    k_subsample<<<grid, 256, 0, st>>>(full, full_off, fin_off, e_max, fin);
    ctx->launches += 3;
    epo_dfree(ctx, full_off); epo_dfree(ctx, full); full_off = nullptr; full = nullptr;
    *out_off = fin_off; *out_rec = fin; *out_E = hfin[N]; *h_off = hfin;
  }
  PP_CUDA(cudaGetLastError());
  cleanup();
#undef PP_CUDA
  return EPO_OK;
}

void epo_free_atlas(EpoAtlas* a) {
  if (a->tex) cudaDestroyTextureObject(a->tex);
  if (a->tex8) cudaDestroyTextureObject(a->tex8);
  if (a->arr) cudaFreeArray(a->arr);
  if (a->arr8) cudaFreeArray(a->arr8);
  a->tex = a->tex8 = 0; a->arr = a->arr8 = nullptr;
}

// Distance fields of all views (rows a-P2, a-P3), written straight into ONE block-linear, gather-enabled 2-D
// CUDA array (view i at texel offset ((i % cols) W, (i / cols) H)) behind one texture object.  The fused kernel
// fetches the 2x2 bilinear footprint with ONE tld4 (tex2Dgather) and applies the exact fp32 weights itself;
// the hardware's 8-bit-fraction filtering is never used.  A footprint never leaves its view (x0 <= W-2).
// Enqueues on the context's stream and does NOT synchronise; the caller releases *scratch_out (row-pass
// buffer + the surface handle the column kernel writes through) with epo_free_dtf_scratch once the stream
// has drained.
void epo_free_dtf_scratch(epo_ctx* ctx, EpoDtfScratch* s) {
  if (s->surf) cudaDestroySurfaceObject(s->surf);
  if (s->surf8) cudaDestroySurfaceObject(s->surf8);
  epo_dfree(ctx, s->g);
  s->surf = s->surf8 = 0; s->g = nullptr;
}

epo_status epo_build_dtf_atlas(epo_ctx* ctx, const uint8_t* d_edges_u8, EpoAtlas* out, EpoDtfScratch* scratch_out) {
  const int N = ctx->N, W = ctx->W, H = ctx->H;
  const int64_t rows = (int64_t)N * H;
  cudaStream_t st = ctx->stream;
  const bool half = ctx->cfg.dtf_format == 1;
  int cols = 32768 / W; if (cols < 1) cols = 1; if (cols > N) cols = N;
  const int arows = (N + cols - 1) / cols;
  if ((int64_t)arows * H > 65536 || (int64_t)cols * W > 131072)
    return epo_fail(ctx, EPO_ERR_UNSUPPORTED, "%d views of %dx%d do not fit one 2-D texture atlas", N, W, H);
  EpoAtlas a = {nullptr, nullptr, 0, 0, cols};
  cudaSurfaceObject_t surf = 0, surf8 = 0; int32_t* g = nullptr;
  cudaChannelFormatDesc desc = half ? cudaCreateChannelDescHalf() : cudaCreateChannelDesc<float>();
  cudaChannelFormatDesc desc8 = cudaCreateChannelDesc<unsigned char>();
  const unsigned flags = cudaArrayTextureGather | cudaArraySurfaceLoadStore;
  cudaError_t e = cudaMallocArray(&a.arr, &desc, (size_t)cols * W, (size_t)arows * H, flags);
  if (e == cudaSuccess && !half) e = cudaMallocArray(&a.arr8, &desc8, (size_t)cols * W, (size_t)arows * H, flags);
  cudaResourceDesc rd; memset(&rd, 0, sizeof(rd));
  rd.resType = cudaResourceTypeArray; rd.res.array.array = a.arr;
  cudaResourceDesc rd8 = rd; rd8.res.array.array = a.arr8;
  if (e == cudaSuccess) e = cudaCreateSurfaceObject(&surf, &rd);
  if (e == cudaSuccess && !half) e = cudaCreateSurfaceObject(&surf8, &rd8);
  if (e == cudaSuccess) e = epo_dmalloc(ctx, &g, (size_t)rows * W * sizeof(int32_t));
  if (e == cudaSuccess) {
    const int grid_rows = (int)((rows + kWarpsPerBlock - 1) / kWarpsPerBlock);
    k_edt_rows<<<grid_rows, kWarpsPerBlock * 32, 0, st>>>(d_edges_u8, rows, W, W + H, g);
    // 64-bit arithmetic only when (W+H)^2 + H^2 could overflow int32
    const bool wide = (int64_t)(W + H) * (W + H) + (int64_t)H * H >= (int64_t)INT32_MAX / 2;
    const size_t smem = (size_t)H * kEdtStrip * sizeof(int32_t);
    const bool stage = smem <= 200 * 1024;   // taller images read g through L1/L2 instead of a staged strip
    dim3 grid((W + kEdtStrip - 1) / kEdtStrip, N);
    const int thr = kEdtStrip * kEdtWarps;
#define EDT_LAUNCH(I, S)                                                                                       \
    do {                                                                                                        \
      if (S) e = cudaFuncSetAttribute(k_edt_cols<I, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
      if (e == cudaSuccess) k_edt_cols<I, S><<<grid, thr, (S) ? smem : 0, st>>>(g, W, H, surf, surf8, cols, half ? 1 : 0); \
    } while (0)
    if (wide) { if (stage) EDT_LAUNCH(long long, true); else EDT_LAUNCH(long long, false); }
    else      { if (stage) EDT_LAUNCH(int, true);       else EDT_LAUNCH(int, false); }
#undef EDT_LAUNCH
    ctx->launches += 2;
    if (e == cudaSuccess) e = cudaGetLastError();
  }
  if (e == cudaSuccess) {
    cudaTextureDesc td; memset(&td, 0, sizeof(td));
    td.addressMode[0] = td.addressMode[1] = cudaAddressModeClamp;
    td.filterMode = cudaFilterModePoint; td.readMode = cudaReadModeElementType; td.normalizedCoords = 0;
    e = cudaCreateTextureObject(&a.tex, &rd, &td, nullptr);
    if (e == cudaSuccess && !half) e = cudaCreateTextureObject(&a.tex8, &rd8, &td, nullptr);
  }
  if (e != cudaSuccess) {
    cudaStreamSynchronize(st);
    if (surf) cudaDestroySurfaceObject(surf);
    if (surf8) cudaDestroySurfaceObject(surf8);
    epo_dfree(ctx, g);
    epo_free_atlas(&a);
    return epo_fail(ctx, e == cudaErrorMemoryAllocation ? EPO_ERR_OUT_OF_MEMORY : EPO_ERR_CUDA, "distance fields: %s",
                    cudaGetErrorString(e));
  }
  *out = a; scratch_out->g = g; scratch_out->surf = surf; scratch_out->surf8 = surf8;
  return EPO_OK;
}

epo_status epo_build_points(epo_ctx* ctx, const float* d_K, const int32_t* d_off, const EdgeRec* d_rec, int64_t E,
                            const std::vector<int32_t>& h_off, const uint8_t* d_edges_u8, const float* d_depth,
                            bool subsampled, EpoPacked* out) {
  float4* pts = nullptr;                             // tile-major (x_s, y_s, z_s, pixel index), packed at the end
  cudaStream_t st = ctx->stream;
  EPO_CUDA(ctx, epo_dmalloc(ctx, &pts, (size_t)(E > 0 ? E : 1) * sizeof(float4)));
  cudaError_t e = cudaSuccess;
  if (subsampled) {
    // an E_max sub-sample is defined on the raster list (reading S6): keep its order
    int max_n = 1;
    for (int i = 0; i < ctx->N; ++i) max_n = h_off[i + 1] - h_off[i] > max_n ? h_off[i + 1] - h_off[i] : max_n;
    dim3 grid((max_n + 255) / 256, ctx->N);
    k_make_points<<<grid, 256, 0, st>>>(d_rec, d_off, d_K, ctx->W, pts);
    ctx->launches += 1;
    e = cudaGetLastError();
  } else {
    // tile-major: per-(view, tile) counts -> scan -> ordered scatter.  The per-view totals equal the raster
    // list's (same keep rule), so view i's points occupy [off[i], off[i+1]) in both orders.
    const int N = ctx->N, W = ctx->W, H = ctx->H;
    const int tiles_x = (W + kTile - 1) / kTile, tiles_y = (H + kTile - 1) / kTile;
    const int64_t n_tiles = (int64_t)N * tiles_x * tiles_y;
    int32_t *tile_cnt = nullptr, *tile_off = nullptr;
    e = epo_dmalloc(ctx, &tile_cnt, (size_t)(n_tiles + 1) * sizeof(int32_t));
    if (e == cudaSuccess) e = epo_dmalloc(ctx, &tile_off, (size_t)(n_tiles + 1) * sizeof(int32_t));
    if (e == cudaSuccess) {
      const int grid = (int)((n_tiles + kWarpsPerBlock - 1) / kWarpsPerBlock);
      k_tile_count<<<grid, kWarpsPerBlock * 32, 0, st>>>(d_edges_u8, d_depth, N, W, H, tiles_x, tiles_y, ctx->cfg.z_min, tile_cnt);
      k_exclusive_scan<<<1, 1024, 0, st>>>(tile_cnt, tile_off, n_tiles, 0);
      k_tile_points<<<grid, kWarpsPerBlock * 32, 0, st>>>(d_edges_u8, d_depth, N, W, H, tiles_x, tiles_y, ctx->cfg.z_min,
                                                          tile_off, d_K, pts);
      ctx->launches += 3;
      e = cudaGetLastError();
    }
    epo_dfree(ctx, tile_cnt); epo_dfree(ctx, tile_off);
  }
  if (e != cudaSuccess) { epo_dfree(ctx, pts); return epo_fail(ctx, EPO_ERR_CUDA, "point list: %s", cudaGetErrorString(e)); }
  EpoPacked pk = {nullptr, nullptr, nullptr, {}};
  epo_status rc = alloc_packed(ctx, h_off, &pk);
  if (rc == EPO_OK) {
    int max_slots = 1;
    for (int i = 0; i < ctx->N; ++i) max_slots = std::max(max_slots, (pk.h_off[i + 1] - pk.h_off[i]) / 2);
    dim3 grid((unsigned)std::min((max_slots + 255) / 256, 64), (unsigned)ctx->N);
    k_pack_points<<<grid, 256, 0, st>>>(pts, d_off, pk.d_off, pk.xyz, pk.pix);
    ctx->launches += 1;
    if (cudaGetLastError() != cudaSuccess) { epo_free_packed(ctx, &pk); rc = epo_fail(ctx, EPO_ERR_CUDA, "packed points: launch failed"); }
  }
  epo_dfree(ctx, pts);                               // stream-ordered: after the packing kernel
  if (rc == EPO_OK) *out = pk;
  return rc;
}

// =============================================================================================
// epo_edt_no_alloc (include/epo.h): the distance transform of ONE edge map for callers that must not allocate.
//
// The ordinary path (epo_set_views -> epo_build_dtf_atlas above) takes its row-pass buffer g[H][W] from the context's
// memory pool.  Some programs cannot let a library do that: a serving or training process that has already given all of
// HBM to its own caching allocator (a cudaMalloc made behind its back fails, or succeeds and later makes ITS next
// allocation fail), and a per-frame loop with a latency budget, where cudaMalloc / cudaFree stall the whole device.
// For them the row-pass buffer lives in the library image instead: a file-scope __device__ array, present on every GPU
// that loads libepo.so from the moment the module is loaded until the process exits.  The entry point below makes no
// cudaMalloc / cudaFree / pool / array / texture / surface / event call, in its first call or in any later one.
//
// k_edt_cols_linear is k_edt_cols with a plain row-major fp32 output instead of the surface stores into the atlas, and
// without the staged strip (no opt-in shared memory): same outward integer search, same square root, so the field is
// bit-identical to epo_get_dtf's.
// =============================================================================================
namespace {

// the scratch: EPO_EDT_NO_ALLOC_MAX_PIXELS int32 = 2 MiB per GPU
static __device__ __align__(256) int32_t g_edt_na_scratch[EPO_EDT_NO_ALLOC_MAX_PIXELS];

// In host code `g_edt_na_scratch` is only the host-side shadow of the symbol, not an address the GPU can use: the real
// address differs per device and comes from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int kNaMaxDevices = 64;
std::mutex g_edt_na_mu;
int32_t* g_edt_na_ptr[kNaMaxDevices] = {};

template <typename I>
__global__ void __launch_bounds__(kEdtStrip * kEdtWarps)
k_edt_cols_linear(const int32_t* __restrict__ g, int W, int H, float* __restrict__ dtf) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int x = blockIdx.x * kEdtStrip + lane;
  const bool in = x < W;
  const int32_t* gv = g + (in ? x : W - 1);
  auto G = [&](int y) -> I { return (I)__ldg(gv + (size_t)y * W); };
  for (int y = blockIdx.y * kEdtWarps + warp; y < H; y += gridDim.y * kEdtWarps) {
    const I g0 = G(y);
    I best = g0 * g0;
    const int dmax = max(y, H - 1 - y);
    for (int dy = 1; dy <= dmax; ++dy) {
      const I dd = (I)dy * dy;
      if (dd >= best) break;
      const I a = G(max(y - dy, 0)), b = G(min(y + dy, H - 1));
      const I m = a < b ? a : b;
      const I c = m * m + dd;
      best = c < best ? c : best;
    }
    if (in) dtf[(size_t)y * W + x] = (best < (I)(1 << 24)) ? __fsqrt_rn((float)best) : (float)sqrt((double)best);
  }
}

epo_status na_fail(char* err, int32_t err_len, epo_status st, const char* fmt, ...) {
  if (err && err_len > 0) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(err, (size_t)err_len, fmt, ap);
    va_end(ap);
  }
  return st;
}

bool na_on_device(const void* p, int dev) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return (a.type == cudaMemoryTypeDevice && a.device == dev) || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" epo_status epo_edt_no_alloc(const uint8_t* d_edges, int32_t width, int32_t height, float* d_dtf, void* stream,
                                       char* err, int32_t err_len) {
  if (err && err_len > 0) err[0] = 0;
  if (!d_edges || !d_dtf) return na_fail(err, err_len, EPO_ERR_INVALID_ARG, "epo_edt_no_alloc: d_edges and d_dtf are required");
  if (width < 2 || height < 2 || width > 65535 || height > 65535)
    return na_fail(err, err_len, EPO_ERR_INVALID_ARG, "epo_edt_no_alloc: need 2 <= width, height <= 65535 (got %d x %d)", width, height);
  const int64_t px = (int64_t)width * height;
  if (px > (int64_t)EPO_EDT_NO_ALLOC_MAX_PIXELS)
    return na_fail(err, err_len, EPO_ERR_UNSUPPORTED,
                   "epo_edt_no_alloc: %d x %d = %lld pixels exceed the built-in scratch of %d pixels "
                   "(EPO_EDT_NO_ALLOC_MAX_PIXELS); use epo_set_views / epo_get_dtf, which allocate",
                   width, height, (long long)px, (int)EPO_EDT_NO_ALLOC_MAX_PIXELS);
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return na_fail(err, err_len, EPO_ERR_CUDA, "epo_edt_no_alloc: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kNaMaxDevices)
    return na_fail(err, err_len, EPO_ERR_UNSUPPORTED, "epo_edt_no_alloc: device ordinal %d (at most %d devices)", dev, kNaMaxDevices);
  if (!na_on_device(d_edges, dev) || !na_on_device(d_dtf, dev))
    return na_fail(err, err_len, EPO_ERR_INVALID_ARG, "epo_edt_no_alloc: d_edges and d_dtf must be device pointers of the current device (%d)", dev);

  // set-up, once per device and with that device current (it is: `dev` is what cudaGetDevice just returned)
  int32_t* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_edt_na_mu);
    if (!g_edt_na_ptr[dev]) {
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_edt_na_scratch);
      if (e != cudaSuccess || !p)
        return na_fail(err, err_len, EPO_ERR_CUDA, "epo_edt_no_alloc: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
      g_edt_na_ptr[dev] = static_cast<int32_t*>(p);
    }
    scratch = g_edt_na_ptr[dev];
  }

  // Nothing in the scratch has to start at zero: the row pass writes all width x height entries before the column pass
  // reads any of them (same stream), and entries beyond them -- left by an earlier, larger call -- are never read.
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int grid_rows = (height + kWarpsPerBlock - 1) / kWarpsPerBlock;
  k_edt_rows<<<grid_rows, kWarpsPerBlock * 32, 0, st>>>(d_edges, (int64_t)height, width, width + height, scratch);
  const bool wide = (int64_t)(width + height) * (width + height) + (int64_t)height * height >= (int64_t)INT32_MAX / 2;
  const int strips = (width + kEdtStrip - 1) / kEdtStrip;
  int bands = (height + kEdtWarps - 1) / kEdtWarps;          // row bands per strip: enough CTAs to fill the machine
  if (bands > 65535) bands = 65535;
  const dim3 grid((unsigned)strips, (unsigned)bands);
  if (wide) k_edt_cols_linear<long long><<<grid, kEdtStrip * kEdtWarps, 0, st>>>(scratch, width, height, d_dtf);
  else      k_edt_cols_linear<int><<<grid, kEdtStrip * kEdtWarps, 0, st>>>(scratch, width, height, d_dtf);
  e = cudaGetLastError();
  if (e != cudaSuccess) return na_fail(err, err_len, EPO_ERR_CUDA, "epo_edt_no_alloc: launch: %s", cudaGetErrorString(e));
  return EPO_OK;
}
