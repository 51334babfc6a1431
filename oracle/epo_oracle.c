/*
 * epo_oracle.c -- plain, slow, obviously-correct CPU oracle for the EPO hot path.
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  It shares no code, header, table or helper with the CUDA
 * library under paper_2607_00579_b200/ and neither includes the other.
 *
 * Everything is double precision on the caller's fp32 inputs (the paper fixes FP32 for the geometry,
 * PAPER.md:121; double here makes the oracle the "exact" side of every tolerance in BASELINE.json).
 * There is no blocking, fusion or re-ordering beyond what the cited passage states.  OpenMP is used
 * over PAIRS only (each pair is an independent unit, Eq. 6); per-pair results are stored
 * and then reduced serially in ascending pair order, so results do not depend on the thread count.
 *
 * Conventions:
 *   - poses are world-to-camera T = [R|t], x_cam = R X_w + t   ("P=[R|t]")
 *   - K = (fx, fy, cx, cy); Z is z-depth (the homogeneous pixel is scaled by Z)
 *   - pixel (u,v) is the sample position; DTF[v][u] is the field value AT (u,v)        (reading S2)
 *   - pose perturbation: T <- Exp(eps) T, eps = (v, w), translation part first          (reading S9)
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): Z0..Z11 of SURVEY.md §8(c) for the loop; S0..S3 (pair
 * sub-sampling), V1..V5 (viewgraph estimation), K1..K5 (Canny), J1..J3 (joint-phase gradients): DESIGN.md §5.
 * Numerical VALUES of the loss/gradient on realistic scenes are "parity unpinned" beyond those checks (nothing in
 * the paper prints one).
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC -o liboracle.so epo_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* =================================================================================================
 * O1  Edge list  ("p in E_i"; "sub-sampled to <= E_max points / image")
 * Raster order (v ascending, then u ascending).  A pixel is kept iff edges != 0 and its depth is
 * finite and > z_min (reading S7).  If e_max > 0 and n > e_max keep entries floor(j*n/e_max) (S6).
 * Returns the count; uv = [count][2] (u, v), z = [count].
 * ================================================================================================= */
int orc_edge_list(int W, int H, const uint8_t* edges, const float* depth, double z_min, int e_max,
                  uint16_t* uv, float* z) {
  int n = 0;
  for (int v = 0; v < H; ++v)
    for (int u = 0; u < W; ++u) {
      float d = depth[(size_t)v * W + u];
      if (edges[(size_t)v * W + u] != 0 && isfinite(d) && (double)d > z_min) {
        uv[2 * n] = (uint16_t)u; uv[2 * n + 1] = (uint16_t)v; z[n] = d; ++n;
      }
    }
  if (e_max > 0 && n > e_max) {
    for (int j = 0; j < e_max; ++j) {
      int k = (int)(((int64_t)j * n) / e_max);
      uv[2 * j] = uv[2 * k]; uv[2 * j + 1] = uv[2 * k + 1]; z[j] = z[k];
    }
    n = e_max;
  }
  return n;
}

/* =================================================================================================
 * O2  Exact Euclidean distance transform  ("each pixel encodes the Euclidean distance to
 * the nearest edge"; "exact L2 distance transform [14]").
 * Distances between pixel centres, in pixels; an edge pixel has DTF 0; an image without edge pixels
 * has DTF = W+H everywhere (reading S8).  d2 is an exact integer; DTF = (float)sqrt((double)d2), which
 * is the correctly rounded fp32 square root because d2 < 2^24 is exact in both formats and rounding
 * the double root to float cannot double-round here: for a non-square integer n < 2^24 the root is at
 * least 2^-50 (relative) away from every fp32 rounding midpoint m (n - m^2 is a non-zero multiple of
 * 2^(2e-48)), far more than the 2^-53 error of the double root.
 * ================================================================================================= */
void orc_edt_brute(int W, int H, const uint8_t* edges, float* dtf) { /* the definition, O(n^2) */
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      int64_t best = (int64_t)(W + H) * (W + H);
      for (int yy = 0; yy < H; ++yy)
        for (int xx = 0; xx < W; ++xx)
          if (edges[(size_t)yy * W + xx]) {
            int64_t d2 = (int64_t)(x - xx) * (x - xx) + (int64_t)(y - yy) * (y - yy);
            if (d2 < best) best = d2;
          }
      dtf[(size_t)y * W + x] = (float)sqrt((double)best);
    }
}

/* Separable form: g[y][x] = min_{x' edge in row y} |x-x'| (W+H if the row has none);
 * d2[y][x] = min_{y'} g[y'][x]^2 + (y-y')^2, every minimum taken by exhaustive search in integers. */
void orc_edt_separable(int W, int H, const uint8_t* edges, float* dtf) {
  int32_t* g = (int32_t*)malloc((size_t)W * H * sizeof(int32_t));
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      int best = W + H;
      for (int xx = 0; xx < W; ++xx)
        if (edges[(size_t)y * W + xx]) { int d = abs(x - xx); if (d < best) best = d; }
      g[(size_t)y * W + x] = best;
    }
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      int64_t best = INT64_MAX;
      for (int yy = 0; yy < H; ++yy) {
        int64_t gg = g[(size_t)yy * W + x];
        int64_t d2 = gg * gg + (int64_t)(y - yy) * (y - yy);
        if (d2 < best) best = d2;
      }
      dtf[(size_t)y * W + x] = (float)sqrt((double)best);
    }
  free(g);
}

void orc_edt_batch(int N, int W, int H, const uint8_t* edges, float* dtf) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int i = 0; i < N; ++i)
    orc_edt_separable(W, H, edges + (size_t)i * W * H, dtf + (size_t)i * W * H);
}

/* fp16 variant of the field (BASELINE.json config 4): round-to-nearest-even of the fp32 value to IEEE
 * binary16, returned widened back to float.  Written out on the bits. */
float orc_round_to_half(float f) {
  uint32_t x; memcpy(&x, &f, 4);
  uint32_t sign = x & 0x80000000u, mag = x & 0x7fffffffu;
  float out;
  if (mag >= 0x7f800000u) return f;                       /* inf / nan unchanged */
  if (mag >= 0x477ff000u) { mag = 0x7f800000u; }          /* >= 65520 rounds to inf */
  else if (mag < 0x38800000u) {                           /* below 2^-14: half subnormal, spacing 2^-24 */
    float a; memcpy(&a, &mag, 4);
    double q = nearbyint((double)a * 16777216.0);         /* ties-to-even in the default rounding mode */
    a = (float)(q / 16777216.0); memcpy(&mag, &a, 4);
  } else {                                                /* normal: keep 10 mantissa bits */
    uint32_t rem = mag & 0x1fffu, base = mag & ~0x1fffu;
    if (rem > 0x1000u || (rem == 0x1000u && (base & 0x2000u))) base += 0x2000u;
    mag = base;
  }
  mag |= sign; memcpy(&out, &mag, 4);
  return out;
}
void orc_round_field_to_half(int64_t n, const float* in, float* out) {
  for (int64_t i = 0; i < n; ++i) out[i] = orc_round_to_half(in[i]);
}

/* =================================================================================================
 * O3  Canonical pair order  (PAPER.md:70 the viewgraph is the pair set; PAPER.md:478-483 batching)
 * ascending (target, source), stable; duplicates kept.  perm[k] = index in the user list of the
 * k-th canonical pair.  Plain bottom-up stable merge sort on the 64-bit key (t, s).
 * ================================================================================================= */
void orc_canonical_pairs(int64_t P, const int32_t* pairs, int32_t* sorted, int32_t* perm) {
  for (int64_t k = 0; k < P; ++k) perm[k] = (int32_t)k;
  int32_t* tmp = (int32_t*)malloc((size_t)P * sizeof(int32_t));
  for (int64_t width = 1; width < P; width *= 2) {
    for (int64_t lo = 0; lo < P; lo += 2 * width) {
      int64_t mid = lo + width < P ? lo + width : P, hi = lo + 2 * width < P ? lo + 2 * width : P;
      int64_t i = lo, j = mid, o = lo;
      while (i < mid && j < hi) {
        int32_t a = perm[i], b = perm[j];
        int64_t ka = ((int64_t)pairs[2 * a + 1] << 32) | (uint32_t)pairs[2 * a];
        int64_t kb = ((int64_t)pairs[2 * b + 1] << 32) | (uint32_t)pairs[2 * b];
        if (kb < ka) tmp[o++] = perm[j++]; else tmp[o++] = perm[i++];   /* ties take the left: stable */
      }
      while (i < mid) tmp[o++] = perm[i++];
      while (j < hi) tmp[o++] = perm[j++];
    }
    memcpy(perm, tmp, (size_t)P * sizeof(int32_t));
  }
  free(tmp);
  for (int64_t k = 0; k < P; ++k) { sorted[2 * k] = pairs[2 * perm[k]]; sorted[2 * k + 1] = pairs[2 * perm[k] + 1]; }
}

/* =================================================================================================
 * Projective function pi, split as the paper splits it (Eq. 2 / Eq. 8)
 * ================================================================================================= */
/* camera-frame point of pixel (u,v) with z-depth Z:  K^-1 [u,v,1]^T Z */
void orc_backproject_cam(const double K[4], double u, double v, double Z, double x[3]) {
  x[0] = Z * ((u - K[2]) / K[0]); x[1] = Z * ((v - K[3]) / K[1]); x[2] = Z;
}
/* world point X = P^-1 x_cam = R^T (x_cam - t) */
void orc_cam_to_world(const double T[12], const double x[3], double X[3]) {
  double d[3] = { x[0] - T[3], x[1] - T[7], x[2] - T[11] };
  for (int i = 0; i < 3; ++i) X[i] = T[i] * d[0] + T[4 + i] * d[1] + T[8 + i] * d[2];
}
/* x_cam = R X + t */
void orc_world_to_cam(const double T[12], const double X[3], double x[3]) {
  for (int i = 0; i < 3; ++i) x[i] = T[4 * i] * X[0] + T[4 * i + 1] * X[1] + T[4 * i + 2] * X[2] + T[4 * i + 3];
}
/* pixel = (fx X/Z + cx, fy Y/Z + cy) */
void orc_project_px(const double K[4], const double x[3], double px[2]) {
  px[0] = K[0] * x[0] / x[2] + K[2]; px[1] = K[1] * x[1] / x[2] + K[3];
}
/* relative pose T_ts = T_t T_s^-1:  R_ts = R_t R_s^T,  t_ts = t_t - R_ts t_s */
void orc_relative_pose(const double Ts[12], const double Tt[12], double Tts[12]) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      Tts[4 * i + j] = Tt[4 * i] * Ts[4 * j] + Tt[4 * i + 1] * Ts[4 * j + 1] + Tt[4 * i + 2] * Ts[4 * j + 2];
  for (int i = 0; i < 3; ++i)
    Tts[4 * i + 3] = Tt[4 * i + 3] - (Tts[4 * i] * Ts[3] + Tts[4 * i + 1] * Ts[7] + Tts[4 * i + 2] * Ts[11]);
}

/* =================================================================================================
 * O4-O6  One directed pair s -> t: loss sum, valid count and the 12 gradient sums.
 *
 * Per source edge pixel p = (u, v, Z)                                    (Eq. 8; 97; 483)
 *   x_s = K_s^-1 [u,v,1]^T Z ;  x_t = R_ts x_s + t_ts ;  reject if x_t.z <= z_min
 *   (x, y) = K_t-projection of x_t ; reject unless 0 <= x <= W-1 and 0 <= y <= H-1      (reading S3)
 *   x0 = min(floor x, W-2), y0 = min(floor y, H-2), wx = x - x0, wy = y - y0
 *   d  = (1-wy)((1-wx) D00 + wx D01) + wy((1-wx) D10 + wx D11)      "bilinearly samples DTF_j"
 *   dhat = min(d, lambda) ;  rho = Huber_delta(dhat) = dhat^2/2 if dhat <= delta else delta (dhat - delta/2)
 *   rho' = [d <= lambda] * min(d, delta)                                              (reading S5)
 * Gradient w.r.t. left perturbations of both poses (reading S9):
 *   a = rho' * (dd/dx, dd/dy) * d(x,y)/d x_t
 *   g_tgt += [ a ; x_t x a ] ;  b = R_ts^T a ;  g_src += [ -b ; -x_s x b ]
 * All 12 numbers are accumulated independently (identity I1 is NOT used here).
 * near[0] counts samples within 1e-3 px (or 1e-3 in z) of the validity border, near[1] those with
 * |d - lambda| < 1e-3 or |d - delta| < 1e-3 -- the discrete events of "Tolerance realism".
 * ================================================================================================= */
/* Variant "coord_fp32" (reading P1).  The paper computes the geometry in FP32, and
 * the projected position decides three integers per sample -- valid or not, and the bilinear cell (x0, y0) --
 * at which the gradient is discontinuous.  Deciding them in double here and in fp32 on the GPU flips a few
 * samples per 10^5 (those within ~3e-5 px of a cell or image border), each worth ~1/n_valid of a pair's
 * gradient.  In this variant steps a-2..a-4 (back-project, transform, project) are therefore evaluated in
 * IEEE binary32 with the operation order stated below (every operation individually rounded; fmaf is the
 * correctly rounded fused multiply-add), and everything after the position (weights, interpolation, robust
 * loss, Jacobian, sums) continues in double exactly as in the default path -- except the one remaining discrete
 * decision, the clamp test d <= lambda (rho' jumps there), taken on the binary32 value of d stated at that line.
 *   T_ts, K rounded once to float;  ifx = 1/fx_s, ify = 1/fy_s
 *   x_s = Z ((u - cx_s) ifx), y_s = Z ((v - cy_s) ify), z_s = Z
 *   X = fma(r00, x_s, fma(r01, y_s, fma(r02, z_s, t_x)))   (same for Y, Z)
 *   iz = 1/Z ;  x = fma(fx_t X, iz, cx_t) ;  y = fma(fy_t Y, iz, cy_t)
 */
static void orc_pair_loss_grad_f32coords(int W, int H, int n_edges, const uint16_t* uv, const float* z,
                                         const double Ks[4], const double Kt[4], const double Tts[12],
                                         const float* dtf_t, double lambda, double delta, double z_min,
                                         double* sum_rho, int32_t* n_valid, double G[12], int32_t near[2],
                                         double* J /* nullable [2] */, double* dZ /* nullable [n_edges] */) {
  float T[12];
  for (int k = 0; k < 12; ++k) T[k] = (float)Tts[k];
  const float ifx = 1.0f / (float)Ks[0], ify = 1.0f / (float)Ks[1], cxs = (float)Ks[2], cys = (float)Ks[3];
  const float fxt = (float)Kt[0], fyt = (float)Kt[1], cxt = (float)Kt[2], cyt = (float)Kt[3];
  const float zmin = (float)z_min, xmax = (float)(W - 1), ymax = (float)(H - 1);
  double S = 0.0; int32_t nv = 0;
  for (int k = 0; k < 12; ++k) G[k] = 0.0;
  near[0] = near[1] = 0;
  if (J) J[0] = J[1] = 0.0;
  if (dZ) for (int e = 0; e < n_edges; ++e) dZ[e] = 0.0;
  for (int e = 0; e < n_edges; ++e) {
    const float u = (float)uv[2 * e], v = (float)uv[2 * e + 1], Zs = z[e];
    const float a_ = (u - cxs) * ifx, b_ = (v - cys) * ify;
    const float xsf = Zs * a_, ysf = Zs * b_, zsf = Zs;
    const float Xf = fmaf(T[0], xsf, fmaf(T[1], ysf, fmaf(T[2], zsf, T[3])));
    const float Yf = fmaf(T[4], xsf, fmaf(T[5], ysf, fmaf(T[6], zsf, T[7])));
    const float Zf = fmaf(T[8], xsf, fmaf(T[9], ysf, fmaf(T[10], zsf, T[11])));
    if (!(Zf > zmin)) continue;
    const float izf = 1.0f / Zf;
    const float fxX = fxt * Xf, fyY = fyt * Yf;
    const float xf = fmaf(fxX, izf, cxt), yf = fmaf(fyY, izf, cyt);
    if (!(xf >= 0.0f && xf <= xmax && yf >= 0.0f && yf <= ymax)) continue;
    /* from here on: the default path, in double, on the fp32 position */
    const double xs[3] = { xsf, ysf, zsf }, xt[3] = { Xf, Yf, Zf };
    const double x = xf, y = yf;
    int x0 = (int)floor(x), y0 = (int)floor(y);
    if (x0 > W - 2) x0 = W - 2;
    if (y0 > H - 2) y0 = H - 2;
    double wx = x - x0, wy = y - y0;
    double D00 = dtf_t[(size_t)y0 * W + x0], D01 = dtf_t[(size_t)y0 * W + x0 + 1];
    double D10 = dtf_t[(size_t)(y0 + 1) * W + x0], D11 = dtf_t[(size_t)(y0 + 1) * W + x0 + 1];
    double d = (1.0 - wy) * ((1.0 - wx) * D00 + wx * D01) + wy * ((1.0 - wx) * D10 + wx * D11);
    double ddx = (1.0 - wy) * (D01 - D00) + wy * (D11 - D10);
    double ddy = (1.0 - wx) * (D10 - D00) + wx * (D11 - D01);
    if (fabs(d - lambda) < 1e-3 || fabs(d - delta) < 1e-3) near[1]++;
    double dhat = d < lambda ? d : lambda;
    double rho = dhat <= delta ? 0.5 * dhat * dhat : delta * (dhat - 0.5 * delta);
    /* reading P1 (clamp decision): rho' jumps from delta to 0 at d = lambda, so "d <= lambda" is a discrete
     * decision like the cell index; in this variant it is taken on the binary32 value of d, evaluated as
     *   dx0 = D01 - D00, dy0 = D10 - D00, c = (D11 - D10) - dx0, d32 = fma(wy, fma(wx, c, dy0), fma(wx, dx0, D00))
     * (wx, wy are exact in binary32: x - x0 with x0 <= x < x0 + 1).  Values (rho, rho', gradient) stay double. */
    const float wxf = (float)wx, wyf = (float)wy;
    const float D00f = dtf_t[(size_t)y0 * W + x0], D01f = dtf_t[(size_t)y0 * W + x0 + 1];
    const float D10f = dtf_t[(size_t)(y0 + 1) * W + x0], D11f = dtf_t[(size_t)(y0 + 1) * W + x0 + 1];
    const float dx0f = D01f - D00f, dy0f = D10f - D00f, cf = (D11f - D10f) - dx0f;
    const float d32 = fmaf(wyf, fmaf(wxf, cf, dy0f), fmaf(wxf, dx0f, D00f));
    double drho = (d32 <= (float)lambda) ? (d < delta ? d : delta) : 0.0;
    S += rho; nv++;
    double iz = 1.0 / xt[2];
    double a[3], b[3];
    a[0] = drho * ddx * Kt[0] * iz;
    a[1] = drho * ddy * Kt[1] * iz;
    a[2] = -drho * (ddx * Kt[0] * xt[0] + ddy * Kt[1] * xt[1]) * iz * iz;
    G[0] += a[0]; G[1] += a[1]; G[2] += a[2];
    G[3] += xt[1] * a[2] - xt[2] * a[1];
    G[4] += xt[2] * a[0] - xt[0] * a[2];
    G[5] += xt[0] * a[1] - xt[1] * a[0];
    for (int i = 0; i < 3; ++i) b[i] = Tts[i] * a[0] + Tts[4 + i] * a[1] + Tts[8 + i] * a[2];
    /* joint phase (Eq. 4-5): d rho / d ln f_t, d rho / d ln f_s (both focal lengths of a camera scale
     * together, f = f0 (1 + gamma)) and d rho / d Z_s of this edge pixel:
     *   (x, y) - c_t = f_t (X, Y)/Z            ->  d rho / d ln f_t = rho' (dd/dx (x - cx_t) + dd/dy (y - cy_t))
     *   x_s = Z ((u - cx)/fx, (v - cy)/fy, 1)  ->  d x_s / d ln f_s = (-x_s.x, -x_s.y, 0),  d x_s / d Z = x_s / Z
     *   and d rho / d x_s = R_ts^T a = b                                                                           */
    if (J) { J[0] += drho * (ddx * (x - Kt[2]) + ddy * (y - Kt[3])); J[1] -= b[0] * xs[0] + b[1] * xs[1]; }
    if (dZ) dZ[e] = (b[0] * xs[0] + b[1] * xs[1] + b[2] * xs[2]) / (double)z[e];
    G[6] -= b[0]; G[7] -= b[1]; G[8] -= b[2];
    G[9]  -= xs[1] * b[2] - xs[2] * b[1];
    G[10] -= xs[2] * b[0] - xs[0] * b[2];
    G[11] -= xs[0] * b[1] - xs[1] * b[0];
  }
  *sum_rho = S; *n_valid = nv;
}

void orc_pair_loss_grad_joint(int W, int H, int n_edges, const uint16_t* uv, const float* z,
                              const double Ks[4], const double Kt[4], const double Ts[12], const double Tt[12],
                              const float* dtf_t, double lambda, double delta, double z_min, int coord_fp32,
                              double* sum_rho, int32_t* n_valid, double G[12], int32_t near[2],
                              double* J /* nullable [2]: sum d rho / d ln f_t, sum d rho / d ln f_s */,
                              double* dZ /* nullable [n_edges]: d rho / d Z_s per edge pixel (0 if not valid) */) {
  double Tts[12];
  orc_relative_pose(Ts, Tt, Tts);
  if (coord_fp32) {
    orc_pair_loss_grad_f32coords(W, H, n_edges, uv, z, Ks, Kt, Tts, dtf_t, lambda, delta, z_min, sum_rho, n_valid, G, near, J, dZ);
    return;
  }
  double S = 0.0; int32_t nv = 0;
  for (int k = 0; k < 12; ++k) G[k] = 0.0;
  near[0] = near[1] = 0;
  if (J) J[0] = J[1] = 0.0;
  if (dZ) for (int e = 0; e < n_edges; ++e) dZ[e] = 0.0;
  for (int e = 0; e < n_edges; ++e) {
    double xs[3], xt[3], px[2];
    orc_backproject_cam(Ks, (double)uv[2 * e], (double)uv[2 * e + 1], (double)z[e], xs);
    for (int i = 0; i < 3; ++i)
      xt[i] = Tts[4 * i] * xs[0] + Tts[4 * i + 1] * xs[1] + Tts[4 * i + 2] * xs[2] + Tts[4 * i + 3];
    if (fabs(xt[2] - z_min) < 1e-3 * fabs(z_min)) near[0]++;
    if (!(xt[2] > z_min)) continue;
    orc_project_px(Kt, xt, px);
    double x = px[0], y = px[1];
    if (fabs(x) < 1e-3 || fabs(x - (W - 1)) < 1e-3 || fabs(y) < 1e-3 || fabs(y - (H - 1)) < 1e-3) near[0]++;
    if (!(x >= 0.0 && x <= (double)(W - 1) && y >= 0.0 && y <= (double)(H - 1))) continue;
    int x0 = (int)floor(x), y0 = (int)floor(y);
    if (x0 > W - 2) x0 = W - 2;
    if (y0 > H - 2) y0 = H - 2;
    double wx = x - x0, wy = y - y0;
    double D00 = dtf_t[(size_t)y0 * W + x0], D01 = dtf_t[(size_t)y0 * W + x0 + 1];
    double D10 = dtf_t[(size_t)(y0 + 1) * W + x0], D11 = dtf_t[(size_t)(y0 + 1) * W + x0 + 1];
    double d = (1.0 - wy) * ((1.0 - wx) * D00 + wx * D01) + wy * ((1.0 - wx) * D10 + wx * D11);
    double ddx = (1.0 - wy) * (D01 - D00) + wy * (D11 - D10);
    double ddy = (1.0 - wx) * (D10 - D00) + wx * (D11 - D01);
    if (fabs(d - lambda) < 1e-3 || fabs(d - delta) < 1e-3) near[1]++;
    double dhat = d < lambda ? d : lambda;
    double rho = dhat <= delta ? 0.5 * dhat * dhat : delta * (dhat - 0.5 * delta);
    double drho = (d <= lambda) ? (d < delta ? d : delta) : 0.0;
    S += rho; nv++;
    /* d(x,y)/d x_t = [ fx/Z, 0, -fx X/Z^2 ; 0, fy/Z, -fy Y/Z^2 ] */
    double iz = 1.0 / xt[2];
    double a[3], b[3];
    a[0] = drho * ddx * Kt[0] * iz;
    a[1] = drho * ddy * Kt[1] * iz;
    a[2] = -drho * (ddx * Kt[0] * xt[0] + ddy * Kt[1] * xt[1]) * iz * iz;
    G[0] += a[0]; G[1] += a[1]; G[2] += a[2];
    G[3] += xt[1] * a[2] - xt[2] * a[1];
    G[4] += xt[2] * a[0] - xt[0] * a[2];
    G[5] += xt[0] * a[1] - xt[1] * a[0];
    for (int i = 0; i < 3; ++i) b[i] = Tts[i] * a[0] + Tts[4 + i] * a[1] + Tts[8 + i] * a[2];
    /* joint phase (Eq. 4-5): d rho / d ln f_t, d rho / d ln f_s (both focal lengths of a camera scale
     * together, f = f0 (1 + gamma)) and d rho / d Z_s of this edge pixel:
     *   (x, y) - c_t = f_t (X, Y)/Z            ->  d rho / d ln f_t = rho' (dd/dx (x - cx_t) + dd/dy (y - cy_t))
     *   x_s = Z ((u - cx)/fx, (v - cy)/fy, 1)  ->  d x_s / d ln f_s = (-x_s.x, -x_s.y, 0),  d x_s / d Z = x_s / Z
     *   and d rho / d x_s = R_ts^T a = b                                                                           */
    if (J) { J[0] += drho * (ddx * (x - Kt[2]) + ddy * (y - Kt[3])); J[1] -= b[0] * xs[0] + b[1] * xs[1]; }
    if (dZ) dZ[e] = (b[0] * xs[0] + b[1] * xs[1] + b[2] * xs[2]) / (double)z[e];
    G[6] -= b[0]; G[7] -= b[1]; G[8] -= b[2];
    G[9]  -= xs[1] * b[2] - xs[2] * b[1];
    G[10] -= xs[2] * b[0] - xs[0] * b[2];
    G[11] -= xs[0] * b[1] - xs[1] * b[0];
  }
  *sum_rho = S; *n_valid = nv;
}

/* =================================================================================================
 * O5 + row a-9: whole loss and per-camera gradient over a pair list (any order; reduced in list order)
 *   L_{s->t} = sum_valid rho / n_valid (0 if none)     (Alg. 3, reading A1)
 *   L = (1/P) sum_D L_{s->t}                           (Eq. 6, reading A3)
 *   g_c = (1/P) [ sum_{t=c} G^tgt_p / n_p + sum_{s=c} G^src_p / n_p ]
 * edge_off [N+1], uv [E][2], z [E] hold all views' lists; dtf [N][H][W]; K float [N][4]; poses double [N][12].
 * Nullable outputs: pair_G [P][12] (un-normalised sums), near [P][2].
 * ================================================================================================= */
void orc_pair_loss_grad(int W, int H, int n_edges, const uint16_t* uv, const float* z,
                        const double Ks[4], const double Kt[4], const double Ts[12], const double Tt[12],
                        const float* dtf_t, double lambda, double delta, double z_min, int coord_fp32,
                        double* sum_rho, int32_t* n_valid, double G[12], int32_t near[2]) {
  orc_pair_loss_grad_joint(W, H, n_edges, uv, z, Ks, Kt, Ts, Tt, dtf_t, lambda, delta, z_min, coord_fp32, sum_rho, n_valid,
                           G, near, NULL, NULL);
}

/* Joint-phase gradients of the loss (Eq. 4-5; 64: "in the subsequent joint phase, optimization is extended
 * to include the depth maps"): with L = (1/P) sum_pairs (1/n_p) sum rho and n_p held fixed as for the poses,
 *   g_logf[c]  = d L / d ln f_c   (as target and as source; d L / d gamma_c = g_logf[c] / (1 + gamma_c))
 *   g_depth[e] = d L / d Z of edge-list entry e (all pairs whose source owns e); with Z = Z0 alpha + beta (Eq. 5):
 *                d L / d alpha = Z0 g_depth, d L / d beta = g_depth.
 * Serial over pairs in list order (a fixed accumulation order).                                                     */
void orc_joint_grad(int N, int W, int H, const float* K, const double* poses, const int32_t* edge_off,
                    const uint16_t* uv, const float* z, const float* dtf, int64_t P, const int32_t* pairs,
                    double lambda, double delta, double z_min, int coord_fp32, double* g_logf, double* g_depth) {
  int max_n = 1;
  for (int i = 0; i < N; ++i) if (edge_off[i + 1] - edge_off[i] > max_n) max_n = edge_off[i + 1] - edge_off[i];
  double* dZ = (double*)malloc((size_t)max_n * sizeof(double));
  for (int i = 0; i < N; ++i) g_logf[i] = 0.0;
  for (int64_t e = 0; e < edge_off[N]; ++e) g_depth[e] = 0.0;
  for (int64_t p = 0; p < P; ++p) {
    const int s = pairs[2 * p], t = pairs[2 * p + 1], n = edge_off[s + 1] - edge_off[s];
    double Ks[4], Kt[4], S, G[12], J[2]; int32_t nv, nr[2];
    for (int i = 0; i < 4; ++i) { Ks[i] = K[4 * s + i]; Kt[i] = K[4 * t + i]; }
    orc_pair_loss_grad_joint(W, H, n, uv + 2 * (size_t)edge_off[s], z + edge_off[s], Ks, Kt, poses + 12 * (size_t)s,
                             poses + 12 * (size_t)t, dtf + (size_t)t * W * H, lambda, delta, z_min, coord_fp32, &S, &nv, G, nr,
                             J, dZ);
    if (nv == 0) continue;
    g_logf[t] += J[0] / nv; g_logf[s] += J[1] / nv;
    for (int e = 0; e < n; ++e) g_depth[edge_off[s] + e] += dZ[e] / nv;
  }
  for (int i = 0; i < N; ++i) g_logf[i] /= (double)P;
  for (int64_t e = 0; e < edge_off[N]; ++e) g_depth[e] /= (double)P;
  free(dZ);
}

void orc_loss_grad(int N, int W, int H, const float* K, const double* poses, const int32_t* edge_off,
                   const uint16_t* uv, const float* z, const float* dtf, int64_t P, const int32_t* pairs,
                   double lambda, double delta, double z_min, int coord_fp32, double* pair_loss,
                   int32_t* pair_valid, double* pair_G, int32_t* near, double* grad, double* loss) {
  double* Gall = (double*)malloc((size_t)P * 12 * sizeof(double));
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t p = 0; p < P; ++p) {
    int s = pairs[2 * p], t = pairs[2 * p + 1];
    double Ks[4], Kt[4], S; int32_t nv, nr[2];
    for (int i = 0; i < 4; ++i) { Ks[i] = K[4 * s + i]; Kt[i] = K[4 * t + i]; }
    orc_pair_loss_grad(W, H, edge_off[s + 1] - edge_off[s], uv + 2 * (size_t)edge_off[s], z + edge_off[s],
                       Ks, Kt, poses + 12 * (size_t)s, poses + 12 * (size_t)t, dtf + (size_t)t * W * H,
                       lambda, delta, z_min, coord_fp32, &S, &nv, Gall + 12 * p, nr);
    pair_loss[p] = nv > 0 ? S / nv : 0.0;
    pair_valid[p] = nv;
    if (near) { near[2 * p] = nr[0]; near[2 * p + 1] = nr[1]; }
  }
  for (int i = 0; i < 6 * N; ++i) grad[i] = 0.0;
  double L = 0.0;
  for (int64_t p = 0; p < P; ++p) {
    int s = pairs[2 * p], t = pairs[2 * p + 1];
    L += pair_loss[p];
    if (pair_valid[p] > 0)
      for (int k = 0; k < 6; ++k) {
        grad[6 * t + k] += Gall[12 * p + k] / pair_valid[p];
        grad[6 * s + k] += Gall[12 * p + 6 + k] / pair_valid[p];
      }
  }
  for (int i = 0; i < 6 * N; ++i) grad[i] /= (double)P;
  *loss = L / (double)P;
  if (pair_G) memcpy(pair_G, Gall, (size_t)P * 12 * sizeof(double));
  free(Gall);
}

/* =================================================================================================
 * Event slack: how far may a CORRECT binary32 evaluation of the same loss be from this all-double one?
 * (SURVEY.md 8(c) "Tolerance realism" (2); reading T1.)
 *
 * The paper computes the geometry in FP32.  The loss is continuous in the projected position, but
 * three decisions per sample are discrete: valid or not (z > z_min, 0 <= x <= W-1, 0 <= y <= H-1: a sample
 * enters or leaves the pair's mean), the bilinear cell (x0, y0) (the spatial gradient of the interpolant
 * jumps at a cell border), and the clamp test d <= lambda (rho' jumps from min(d, delta) to 0).  A binary32
 * evaluation places the sample up to its own rounding error away from where double places it, and so may decide
 * differently for samples that lie that close to a boundary.  This function bounds, from the double side alone
 * and without reference to any particular binary32 program, what those decisions can change.
 *
 * Position error of ANY evaluation that rounds every operation of rows a-2..a-4 to binary32 (u = 2^-24), for the
 * natural formulas  x_s = Z (u - cx_s)/fx_s,  X = r00 x_s + r01 y_s + r02 z_s + t_x,  x = fx_t X / Z + cx_t:
 *   |dX| <= 8 u S_X,  S_X = |r00 x_s| + |r01 y_s| + |r02 z_s| + |t_x|      (same for Y, Z)
 *           [1 u: T_ts rounded to binary32; <= 4 u: the point x_s (difference, reciprocal or division by fx, two
 *            products); 3 u: the three additions (or FMAs) of the row sum]
 *   r_x = fx_t |dX| / Z + |x - cx_t| (|dZ| / Z + 3 u) + u |x|
 *           [product fx_t X, reciprocal or division by Z, their product, the final addition of cx_t]
 *   r_d = |dd/dx| r_x + |dd/dy| r_y + 6 u max|D|                            (the interpolated distance)
 * For every sample the alternatives a binary32 evaluation can reach are enumerated -- valid / not valid if the
 * position is within (r_x, r_y) of the image border (or Z within |dZ| of z_min), the neighbouring cell in x and/or
 * y if the position is within r of a cell border, the other clamp branch if |d - lambda| <= r_d -- and the largest
 * change of the sample's contribution to the pair's un-normalised target sum, source sum (6-vectors, 2-norm)
 * and loss sum is added to the pair's slack:
 *   E_t, E_s, E_rho   sums of those largest changes
 *   k_out, k_in       samples that double counts valid but binary32 may drop / that double drops but binary32
 *                     may count (they change the pair's n_valid)
 * With n' in [n - k_out, n + k_in] and n_lo = max(n - k_out, 1):
 *   | G'/n' - G/n | <= E / n_lo + |G| max(k_out, k_in) / (n n_lo)          (loss sums likewise)
 * and per camera  slack_c = (1/P) [ sum_{t = c} (target bound) + sum_{s = c} (source bound) ].
 * A parity test then asserts  | g_gpu,c - g_oracle,c | <= 1e-4 | g_oracle,c | + slack_c : the contract's tolerance
 * for everything that is continuous, plus exactly what the flagged samples can move.
 * `check` (nullable, [14] per pair) receives S, n and the 12 sums accumulated through THIS function's per-sample
 * routine for the nominal decisions, so that a test can tie it to orc_pair_loss_grad.
 * ================================================================================================= */
#define ORC_U32 5.9604644775390625e-08 /* 2^-24 */

/* contribution of one sample at position (x, y), evaluated in cell (x0, y0) with the clamp branch `inside`
 * (1: d <= lambda taken as true): rho, target 6-vector, source 6-vector.  Same formulas as the pair routine above. */
static void orc_sample_terms(int W, const float* dtf_t, const double Kt[4], const double Tts[12], const double xs[3],
                             const double xt[3], double x, double y, int x0, int y0, int inside, double lambda,
                             double delta, double* rho, double gt[6], double gs[6], double* d_out, double dd[2],
                             double* Dmax, double jz[3] /* nullable: d rho / d ln f_t, d rho / d ln f_s, d rho / d Z_s */) {
  double wx = x - x0, wy = y - y0;
  double D00 = dtf_t[(size_t)y0 * W + x0], D01 = dtf_t[(size_t)y0 * W + x0 + 1];
  double D10 = dtf_t[(size_t)(y0 + 1) * W + x0], D11 = dtf_t[(size_t)(y0 + 1) * W + x0 + 1];
  double d = (1.0 - wy) * ((1.0 - wx) * D00 + wx * D01) + wy * ((1.0 - wx) * D10 + wx * D11);
  double ddx = (1.0 - wy) * (D01 - D00) + wy * (D11 - D10);
  double ddy = (1.0 - wx) * (D10 - D00) + wx * (D11 - D01);
  double dhat = d < lambda ? d : lambda;
  *rho = dhat <= delta ? 0.5 * dhat * dhat : delta * (dhat - 0.5 * delta);
  double drho = inside ? (d < delta ? d : delta) : 0.0;
  double iz = 1.0 / xt[2], a[3], b[3];
  a[0] = drho * ddx * Kt[0] * iz;
  a[1] = drho * ddy * Kt[1] * iz;
  a[2] = -drho * (ddx * Kt[0] * xt[0] + ddy * Kt[1] * xt[1]) * iz * iz;
  gt[0] = a[0]; gt[1] = a[1]; gt[2] = a[2];
  gt[3] = xt[1] * a[2] - xt[2] * a[1];
  gt[4] = xt[2] * a[0] - xt[0] * a[2];
  gt[5] = xt[0] * a[1] - xt[1] * a[0];
  for (int i = 0; i < 3; ++i) b[i] = Tts[i] * a[0] + Tts[4 + i] * a[1] + Tts[8 + i] * a[2];
  gs[0] = -b[0]; gs[1] = -b[1]; gs[2] = -b[2];
  gs[3] = -(xs[1] * b[2] - xs[2] * b[1]);
  gs[4] = -(xs[2] * b[0] - xs[0] * b[2]);
  gs[5] = -(xs[0] * b[1] - xs[1] * b[0]);
  if (jz) {   /* the joint phase's terms, as in orc_pair_loss_grad_joint */
    jz[0] = drho * (ddx * (x - Kt[2]) + ddy * (y - Kt[3]));
    jz[1] = -(b[0] * xs[0] + b[1] * xs[1]);
    jz[2] = (b[0] * xs[0] + b[1] * xs[1] + b[2] * xs[2]) / xs[2];
  }
  *d_out = d; dd[0] = ddx; dd[1] = ddy;
  double m = fabs(D00);
  if (fabs(D01) > m) m = fabs(D01);
  if (fabs(D10) > m) m = fabs(D10);
  if (fabs(D11) > m) m = fabs(D11);
  *Dmax = m;
}

static double orc_norm6(const double a[6], const double b[6] /* nullable: norm of a - b */) {
  double q = 0.0;
  for (int i = 0; i < 6; ++i) { double v = b ? a[i] - b[i] : a[i]; q += v * v; }
  return sqrt(q);
}

/* One pair.  out[8] = { E_t, E_s, E_rho, k_out, k_in, flagged samples, Q_t, Q_s }; check[14] nullable.
 * Q_t, Q_s = sums over the valid samples of the SQUARED 2-norm of the sample's target / source 6-vector: the scale of
 * the pair's gradient before its terms cancel (reading T2: near a minimum |G| -> 0 while the terms do not, and an
 * error "relative to |G|" loses its meaning; a tolerance is then taken relative to max(|g|, root-sum-square)). */
void orc_pair_event_slack_joint(int W, int H, int n_edges, const uint16_t* uv, const float* z, const double Ks[4],
                                const double Kt[4], const double Ts[12], const double Tt[12], const float* dtf_t,
                                double lambda, double delta, double z_min, double out[8], double* check,
                                double* jout /* nullable [4]: E_Jt, E_Js, Q_Jt, Q_Js (joint phase: the focal sums) */,
                                double* dz_slack /* nullable [n_edges]: largest change of d rho / d Z_s of each sample */) {
  double Tts[12];
  orc_relative_pose(Ts, Tt, Tts);
  double Et = 0.0, Es = 0.0, Er = 0.0, Qt = 0.0, Qs = 0.0; int k_out = 0, k_in = 0, flagged = 0;
  double EJt = 0.0, EJs = 0.0, QJt = 0.0, QJs = 0.0;
  if (check) for (int i = 0; i < 14; ++i) check[i] = 0.0;
  if (dz_slack) for (int e = 0; e < n_edges; ++e) dz_slack[e] = 0.0;
  const double xmax = (double)(W - 1), ymax = (double)(H - 1);
  for (int e = 0; e < n_edges; ++e) {
    double xs[3], xt[3], S3[3];
    orc_backproject_cam(Ks, (double)uv[2 * e], (double)uv[2 * e + 1], (double)z[e], xs);
    for (int i = 0; i < 3; ++i) {
      xt[i] = Tts[4 * i] * xs[0] + Tts[4 * i + 1] * xs[1] + Tts[4 * i + 2] * xs[2] + Tts[4 * i + 3];
      S3[i] = fabs(Tts[4 * i] * xs[0]) + fabs(Tts[4 * i + 1] * xs[1]) + fabs(Tts[4 * i + 2] * xs[2]) + fabs(Tts[4 * i + 3]);
    }
    const double eX = 8.0 * ORC_U32 * S3[0], eY = 8.0 * ORC_U32 * S3[1], eZ = 8.0 * ORC_U32 * S3[2];
    const int z_ok = xt[2] > z_min, z_unsure = fabs(xt[2] - z_min) <= eZ;
    if (!z_ok && !z_unsure) continue;                  /* behind the camera on both sides */
    /* A depth within rounding of z_min: with z' <= z + |dZ| the projection is at least fx (|X| - |dX|) / (z + |dZ|) away
     * from the principal point -- far outside the image unless the point sits on the optical centre itself.  Then the
     * sample is invalid on both sides whatever z' is; otherwise nothing bounds its position and the slack is infinite. */
    if (z_unsure) {
      const double z_hi = xt[2] + eZ;
      const double ax = fabs(xt[0]) - eX, ay = fabs(xt[1]) - eY;
      const double far_x = fabs(Kt[2]) + fabs(xmax - Kt[2]) + 1.0, far_y = fabs(Kt[3]) + fabs(ymax - Kt[3]) + 1.0;
      if (z_hi > 0.0 && ((ax > 0.0 && Kt[0] * ax / z_hi > far_x) || (ay > 0.0 && Kt[1] * ay / z_hi > far_y))) {
        if (!z_ok) continue;                           /* invalid here, and outside the image for any z' > z_min */
        /* valid-by-depth here: it continues below and is found outside the image */
      } else {
        flagged++; if (z_ok) k_out++; else k_in++; Et = Es = Er = EJt = EJs = INFINITY;
        if (dz_slack) dz_slack[e] = INFINITY;
        continue;
      }
    }
    double px[2];
    orc_project_px(Kt, xt, px);
    const double x = px[0], y = px[1];
    const double rx = (Kt[0] * eX + fabs(x - Kt[2]) * eZ) / xt[2] + ORC_U32 * (3.0 * fabs(x - Kt[2]) + fabs(x));
    const double ry = (Kt[1] * eY + fabs(y - Kt[3]) * eZ) / xt[2] + ORC_U32 * (3.0 * fabs(y - Kt[3]) + fabs(y));
    const int valid = x >= 0.0 && x <= xmax && y >= 0.0 && y <= ymax;
    const int reach = x >= -rx && x <= xmax + rx && y >= -ry && y <= ymax + ry;   /* binary32 may find it inside */
    if (!reach) continue;
    const int edge_near = x < rx || x > xmax - rx || y < ry || y > ymax - ry;     /* binary32 may decide the other way */
    /* where the alternatives are evaluated: the position itself, moved onto the image if it is just outside */
    const double xe = x < 0.0 ? 0.0 : (x > xmax ? xmax : x), ye = y < 0.0 ? 0.0 : (y > ymax ? ymax : y);
    int x0 = (int)floor(xe), y0 = (int)floor(ye);
    if (x0 > W - 2) x0 = W - 2;
    if (y0 > H - 2) y0 = H - 2;
    /* neighbouring cells a binary32 position may fall into */
    int cxs[2] = { x0, x0 }, cys[2] = { y0, y0 }, ncx = 1, ncy = 1;
    if (xe - x0 < rx && x0 >= 1) { cxs[1] = x0 - 1; ncx = 2; }
    else if (x0 + 1 - xe < rx && x0 + 1 <= W - 2) { cxs[1] = x0 + 1; ncx = 2; }
    if (ye - y0 < ry && y0 >= 1) { cys[1] = y0 - 1; ncy = 2; }
    else if (y0 + 1 - ye < ry && y0 + 1 <= H - 2) { cys[1] = y0 + 1; ncy = 2; }
    /* nominal terms (only meaningful if valid) */
    double rho0 = 0.0, gt0[6] = {0, 0, 0, 0, 0, 0}, gs0[6] = {0, 0, 0, 0, 0, 0}, d0, dd0[2], Dm, jz0[3] = {0, 0, 0};
    orc_sample_terms(W, dtf_t, Kt, Tts, xs, xt, xe, ye, x0, y0, 1, lambda, delta, &rho0, gt0, gs0, &d0, dd0, &Dm, jz0);
    const int inside0 = d0 <= lambda;
    if (!inside0) orc_sample_terms(W, dtf_t, Kt, Tts, xs, xt, xe, ye, x0, y0, 0, lambda, delta, &rho0, gt0, gs0, &d0, dd0, &Dm, jz0);
    const double rd = fabs(dd0[0]) * rx + fabs(dd0[1]) * ry + 6.0 * ORC_U32 * Dm;
    const int lam_unsure = fabs(d0 - lambda) <= rd;
    if (valid && check) {
      check[0] += rho0; check[1] += 1.0;
      for (int i = 0; i < 6; ++i) { check[2 + i] += gt0[i]; check[8 + i] += gs0[i]; }
    }
    if (valid) { double a = orc_norm6(gt0, NULL), b = orc_norm6(gs0, NULL); Qt += a * a; Qs += b * b; QJt += jz0[0] * jz0[0]; QJs += jz0[1] * jz0[1]; }
    if (!valid) { rho0 = 0.0; for (int i = 0; i < 6; ++i) gt0[i] = gs0[i] = 0.0; jz0[0] = jz0[1] = jz0[2] = 0.0; }
    if (!edge_near && ncx == 1 && ncy == 1 && !lam_unsure) continue;               /* nothing discrete in reach */
    flagged++;
    if (edge_near) { if (valid) k_out++; else k_in++; }
    double wt = 0.0, ws = 0.0, wr = 0.0, wj[3] = {0, 0, 0};
    if (valid && edge_near) {   /* dropped */
      wt = orc_norm6(gt0, NULL); ws = orc_norm6(gs0, NULL); wr = rho0;
      for (int i = 0; i < 3; ++i) wj[i] = fabs(jz0[i]);
    }
    for (int ix = 0; ix < ncx; ++ix)
      for (int iy = 0; iy < ncy; ++iy)
        for (int br = 0; br < 2; ++br) {
          const int inside = br == 0 ? inside0 : !inside0;
          if (br == 1 && !lam_unsure) continue;
          double rho1, gt1[6], gs1[6], d1, dd1[2], Dm1, jz1[3];
          orc_sample_terms(W, dtf_t, Kt, Tts, xs, xt, xe, ye, cxs[ix], cys[iy], inside, lambda, delta, &rho1, gt1, gs1, &d1, dd1, &Dm1, jz1);
          double a = orc_norm6(gt1, gt0), b = orc_norm6(gs1, gs0), c = fabs(rho1 - rho0);
          if (a > wt) wt = a;
          if (b > ws) ws = b;
          if (c > wr) wr = c;
          for (int i = 0; i < 3; ++i) if (fabs(jz1[i] - jz0[i]) > wj[i]) wj[i] = fabs(jz1[i] - jz0[i]);
        }
    Et += wt; Es += ws; Er += wr; EJt += wj[0]; EJs += wj[1];
    if (dz_slack) dz_slack[e] = wj[2];
  }
  if (jout) { jout[0] = EJt; jout[1] = EJs; jout[2] = QJt; jout[3] = QJs; }
  out[0] = Et; out[1] = Es; out[2] = Er; out[3] = k_out; out[4] = k_in; out[5] = flagged; out[6] = Qt; out[7] = Qs;
}

void orc_pair_event_slack(int W, int H, int n_edges, const uint16_t* uv, const float* z, const double Ks[4],
                          const double Kt[4], const double Ts[12], const double Tt[12], const float* dtf_t,
                          double lambda, double delta, double z_min, double out[8], double* check) {
  orc_pair_event_slack_joint(W, H, n_edges, uv, z, Ks, Kt, Ts, Tt, dtf_t, lambda, delta, z_min, out, check, NULL, NULL);
}

/* The same bound for the joint phase's gradients (orc_joint_grad): logf_slack [N] on d L / d ln f_c, logf_rss [N] its
 * root-sum-square scale (reading T2), gz_slack [E] on d L / d Z of every edge-list entry.  Serial over pairs. */
void orc_joint_slack(int N, int W, int H, const float* K, const double* poses, const int32_t* edge_off,
                     const uint16_t* uv, const float* z, const float* dtf, int64_t P, const int32_t* pairs,
                     double lambda, double delta, double z_min, double* logf_slack, double* logf_rss, double* gz_slack) {
  int max_n = 1;
  for (int i = 0; i < N; ++i) if (edge_off[i + 1] - edge_off[i] > max_n) max_n = edge_off[i + 1] - edge_off[i];
  double* dzs = (double*)malloc((size_t)max_n * sizeof(double));
  double* dZ = (double*)malloc((size_t)max_n * sizeof(double));
  for (int i = 0; i < N; ++i) logf_slack[i] = logf_rss[i] = 0.0;
  for (int64_t e = 0; e < edge_off[N]; ++e) gz_slack[e] = 0.0;
  for (int64_t p = 0; p < P; ++p) {
    const int s = pairs[2 * p], t = pairs[2 * p + 1], n_e = edge_off[s + 1] - edge_off[s];
    double Ks[4], Kt[4], S, G[12], J[2], o[8], jo[4]; int32_t nv, nr[2];
    for (int i = 0; i < 4; ++i) { Ks[i] = K[4 * s + i]; Kt[i] = K[4 * t + i]; }
    orc_pair_loss_grad_joint(W, H, n_e, uv + 2 * (size_t)edge_off[s], z + edge_off[s], Ks, Kt, poses + 12 * (size_t)s,
                             poses + 12 * (size_t)t, dtf + (size_t)t * W * H, lambda, delta, z_min, 0, &S, &nv, G, nr, J, dZ);
    orc_pair_event_slack_joint(W, H, n_e, uv + 2 * (size_t)edge_off[s], z + edge_off[s], Ks, Kt, poses + 12 * (size_t)s,
                               poses + 12 * (size_t)t, dtf + (size_t)t * W * H, lambda, delta, z_min, o, NULL, jo, dzs);
    const double n = (double)nv, k_out = o[3], k_in = o[4], kmax = k_out > k_in ? k_out : k_in;
    const double n_lo = n - k_out >= 1.0 ? n - k_out : 1.0;
    logf_slack[t] += jo[0] / n_lo + (n > 0.0 ? fabs(J[0]) * kmax / (n * n_lo) : 0.0);
    logf_slack[s] += jo[1] / n_lo + (n > 0.0 ? fabs(J[1]) * kmax / (n * n_lo) : 0.0);
    if (n > 0.0) { logf_rss[t] += jo[2] / (n * n); logf_rss[s] += jo[3] / (n * n); }
    for (int e = 0; e < n_e; ++e)
      gz_slack[edge_off[s] + e] += dzs[e] / n_lo + (n > 0.0 ? fabs(dZ[e]) * kmax / (n * n_lo) : 0.0);
  }
  for (int i = 0; i < N; ++i) { logf_slack[i] /= (double)P; logf_rss[i] = sqrt(logf_rss[i]) / (double)P; }
  for (int64_t e = 0; e < edge_off[N]; ++e) gz_slack[e] /= (double)P;
  free(dzs); free(dZ);
}

/* Whole list: per-camera gradient slack [N], per-pair loss slack [P], per-pair (k_out, k_in, flagged) [P][3].
 * pair_valid / pair_G are the nominal results of orc_loss_grad on the same inputs (pair_G [P][12] un-normalised). */
void orc_event_slack(int N, int W, int H, const float* K, const double* poses, const int32_t* edge_off,
                     const uint16_t* uv, const float* z, const float* dtf, int64_t P, const int32_t* pairs,
                     double lambda, double delta, double z_min, const double* pair_loss, const int32_t* pair_valid,
                     const double* pair_G, double* cam_slack, double* pair_loss_slack, int32_t* pair_flags,
                     double* cam_rss /* [N]: root-sum-square of the terms of each camera's gradient (reading T2) */) {
  double* bt = (double*)malloc((size_t)P * sizeof(double));
  double* bs = (double*)malloc((size_t)P * sizeof(double));
  double* qt = (double*)malloc((size_t)P * sizeof(double));
  double* qs = (double*)malloc((size_t)P * sizeof(double));
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t p = 0; p < P; ++p) {
    int s = pairs[2 * p], t = pairs[2 * p + 1];
    double Ks[4], Kt[4], o[8];
    for (int i = 0; i < 4; ++i) { Ks[i] = K[4 * s + i]; Kt[i] = K[4 * t + i]; }
    orc_pair_event_slack_joint(W, H, edge_off[s + 1] - edge_off[s], uv + 2 * (size_t)edge_off[s], z + edge_off[s], Ks, Kt,
                               poses + 12 * (size_t)s, poses + 12 * (size_t)t, dtf + (size_t)t * W * H, lambda, delta, z_min, o, NULL,
                               NULL, NULL);
    const double n = (double)pair_valid[p], k_out = o[3], k_in = o[4], kmax = k_out > k_in ? k_out : k_in;
    const double n_lo = n - k_out >= 1.0 ? n - k_out : 1.0;
    const double Gt = orc_norm6(pair_G + 12 * p, NULL), Gs = orc_norm6(pair_G + 12 * p + 6, NULL);
    bt[p] = o[0] / n_lo + (n > 0.0 ? Gt * kmax / (n * n_lo) : 0.0);
    bs[p] = o[1] / n_lo + (n > 0.0 ? Gs * kmax / (n * n_lo) : 0.0);
    pair_loss_slack[p] = o[2] / n_lo + (n > 0.0 ? pair_loss[p] * kmax / n_lo : 0.0);
    pair_flags[3 * p] = (int32_t)k_out; pair_flags[3 * p + 1] = (int32_t)k_in; pair_flags[3 * p + 2] = (int32_t)o[5];
    qt[p] = n > 0.0 ? o[6] / (n * n) : 0.0; qs[p] = n > 0.0 ? o[7] / (n * n) : 0.0;
  }
  for (int i = 0; i < N; ++i) cam_slack[i] = cam_rss[i] = 0.0;
  for (int64_t p = 0; p < P; ++p) {
    cam_slack[pairs[2 * p + 1]] += bt[p]; cam_slack[pairs[2 * p]] += bs[p];
    cam_rss[pairs[2 * p + 1]] += qt[p]; cam_rss[pairs[2 * p]] += qs[p];
  }
  for (int i = 0; i < N; ++i) { cam_slack[i] /= (double)P; cam_rss[i] = sqrt(cam_rss[i]) / (double)P; }
  free(bt); free(bs); free(qt); free(qs);
}

/* =================================================================================================
 * Edge extraction: "the edge map E_i via the Canny edge detector [4]" (Alg. 1 l.6).
 * The paper names the detector and nothing else; this is Canny's scheme [4] -- smooth, gradient, non-maximum
 * suppression along the gradient, hysteresis thresholding -- in integer arithmetic on 8-bit images (readings C1-C6):
 *   C1 smoothing   separable binomial [1 4 6 4 1]/16 (sigma ~ 1), replicate border, b = (sum w_y w_x p + 128) >> 8
 *   C2 gradient    Sobel 3x3 on b, replicate border: gx = [-1 0 1; -2 0 2; -1 0 1], gy = its transpose
 *   C3 magnitude   m2 = gx^2 + gy^2 (the squared L2 norm: thresholds are compared squared, no square root)
 *   C4 direction   4 sectors by integer tests with tan(22.5 deg) ~ 13573 / 32768: |gy| 32768 < |gx| 13573 -> compare the
 *                  left/right neighbours; |gy| 13573 > |gx| 32768 -> up/down; else the diagonal with the gradient's sign
 *   C5 suppression a candidate has m2 > low^2, m2 > m2(first neighbour) and m2 >= m2(second neighbour) (first = left,
 *                  up, or upper diagonal neighbour: of two equal neighbours the first one stays); border pixels are never candidates
 *   C6 hysteresis  strong = candidate with m2 > high^2; the edge map = candidates 8-connected, through candidates,
 *                  to a strong one.  Output 1 / 0.
 * Stages are separate functions so that each can be checked on its own.
 * ================================================================================================= */
static inline int orc_clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* C7 colour -> grey.  The paper extracts edges from the RGB images and says nothing about the
 * conversion; reading C7: the ITU-R BT.601 luma weights (0.299, 0.587, 0.114) in 8-bit fixed point,
 *   Y = (77 R + 150 G + 29 B + 128) >> 8     (77 + 150 + 29 = 256: a grey pixel R = G = B keeps its value),
 * interleaved input [n_px][3]. */
void orc_rgb_to_grey(int64_t n_px, const uint8_t* rgb, uint8_t* grey) {
  for (int64_t i = 0; i < n_px; ++i)
    grey[i] = (uint8_t)((77 * (int)rgb[3 * i] + 150 * (int)rgb[3 * i + 1] + 29 * (int)rgb[3 * i + 2] + 128) >> 8);
}

void orc_canny_blur(int W, int H, const uint8_t* img, uint8_t* out) {
  static const int w[5] = {1, 4, 6, 4, 1};
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      int acc = 0;
      for (int dy = -2; dy <= 2; ++dy)
        for (int dx = -2; dx <= 2; ++dx)
          acc += w[dy + 2] * w[dx + 2] * (int)img[(size_t)orc_clampi(y + dy, 0, H - 1) * W + orc_clampi(x + dx, 0, W - 1)];
      out[(size_t)y * W + x] = (uint8_t)((acc + 128) >> 8);
    }
}

void orc_canny_sobel(int W, int H, const uint8_t* b, int32_t* gx, int32_t* gy) {
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      int p[3][3];
      for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx)
          p[dy + 1][dx + 1] = (int)b[(size_t)orc_clampi(y + dy, 0, H - 1) * W + orc_clampi(x + dx, 0, W - 1)];
      gx[(size_t)y * W + x] = (p[0][2] - p[0][0]) + 2 * (p[1][2] - p[1][0]) + (p[2][2] - p[2][0]);
      gy[(size_t)y * W + x] = (p[2][0] - p[0][0]) + 2 * (p[2][1] - p[0][1]) + (p[2][2] - p[0][2]);
    }
}

/* cand[y][x]: 0 = no, 1 = candidate (weak), 2 = strong */
void orc_canny_suppress(int W, int H, const int32_t* gx, const int32_t* gy, int low, int high, uint8_t* cand) {
  const int64_t lo2 = (int64_t)low * low, hi2 = (int64_t)high * high;
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      uint8_t c = 0;
      if (x > 0 && y > 0 && x < W - 1 && y < H - 1) {
        const size_t i = (size_t)y * W + x;
        const int64_t ax = llabs((long long)gx[i]), ay = llabs((long long)gy[i]);
        const int64_t m2 = ax * ax + ay * ay;
        if (m2 > lo2) {
          int dx1, dy1;                       /* first neighbour; the second is its mirror image */
          if (ay * 32768 < ax * 13573) { dx1 = -1; dy1 = 0; }
          else if (ay * 13573 > ax * 32768) { dx1 = 0; dy1 = -1; }
          else if ((gx[i] < 0) == (gy[i] < 0)) { dx1 = -1; dy1 = -1; }
          else { dx1 = 1; dy1 = -1; }
          const size_t a = (size_t)(y + dy1) * W + (x + dx1), b = (size_t)(y - dy1) * W + (x - dx1);
          const int64_t ma = (int64_t)gx[a] * gx[a] + (int64_t)gy[a] * gy[a], mb = (int64_t)gx[b] * gx[b] + (int64_t)gy[b] * gy[b];
          if (m2 > ma && m2 >= mb) c = m2 > hi2 ? 2 : 1;
        }
      }
      cand[(size_t)y * W + x] = c;
    }
}

void orc_canny_hysteresis(int W, int H, const uint8_t* cand, uint8_t* edges) {
  int32_t* stack = (int32_t*)malloc((size_t)W * H * sizeof(int32_t));
  int64_t top = 0;
  for (int64_t i = 0; i < (int64_t)W * H; ++i) { edges[i] = 0; if (cand[i] == 2) { edges[i] = 1; stack[top++] = (int32_t)i; } }
  while (top > 0) {
    const int32_t i = stack[--top];
    const int x = i % W, y = i / W;
    for (int dy = -1; dy <= 1; ++dy)
      for (int dx = -1; dx <= 1; ++dx) {
        const int xx = x + dx, yy = y + dy;
        if (xx < 0 || yy < 0 || xx >= W || yy >= H) continue;
        const int32_t j = yy * W + xx;
        if (cand[j] && !edges[j]) { edges[j] = 1; stack[top++] = j; }
      }
  }
  free(stack);
}

void orc_canny(int N, int W, int H, const uint8_t* img, int low, int high, uint8_t* edges) {
#pragma omp parallel for schedule(dynamic)
  for (int n = 0; n < N; ++n) {
    const size_t px = (size_t)W * H;
    uint8_t* b = (uint8_t*)malloc(px); uint8_t* c = (uint8_t*)malloc(px);
    int32_t* gx = (int32_t*)malloc(px * sizeof(int32_t)); int32_t* gy = (int32_t*)malloc(px * sizeof(int32_t));
    orc_canny_blur(W, H, img + n * px, b);
    orc_canny_sobel(W, H, b, gx, gy);
    orc_canny_suppress(W, H, gx, gy, low, high, c);
    orc_canny_hysteresis(W, H, c, edges + n * px);
    free(b); free(c); free(gx); free(gy);
  }
}

/* =================================================================================================
 * Viewgraph estimation by exhaustive cycle-consistent reprojection (Eq. 2; 117; 380-384; 396).
 * "we project each pixel p of image I_i onto I_j using pi (Eq. 2) ... The resulting p_{i->j} is then projected back
 * onto I_i to obtain p_{i->j->i}.  An image pair is called valid if sufficiently many pixels satisfy a bidirectional
 * reprojection error || p - p_{i->j->i} ||_2 < tau" -- "at least 12.5% of their reprojected 2D points ... below
 * tau = 3.0 pixels"; "for every one of the C(N,2) candidate pairs a kernel projects a grid of source
 * pixels into the target view and back".
 *
 * orc_viewgraph_counts: for every ORDERED pair (i, j), i != j, counts[(i N + j) 2 + {0,1}] = {consistent, usable}:
 *   grid   p = (u, v), u = stride/2 + a stride < W, v = stride/2 + b stride < H               (reading V1)
 *   usable Z_i(p) finite and > z_min                                                          (reading V2)
 *   p_ij = pi(K_i, K_j, P_i, P_j, Z_i; p): x_j = T_j T_i^-1 K_i^-1 [u,v,1]^T Z_i, needs x_j.z > z_min and
 *          0 <= x <= W-1, 0 <= y <= H-1                                                       (reading V3)
 *   Z_j at the pixel nearest to p_ij, (floor(x + 1/2), floor(y + 1/2)); finite and > z_min    (reading V4)
 *   p_iji = pi(K_j, K_i, P_j, P_i, that depth; p_ij) from the SUB-PIXEL position p_ij; needs z > z_min  (reading V5)
 *   consistent iff (x' - u)^2 + (y' - v)^2 < tau^2                                            (Eq. text; reading V6)
 * coord_fp32 = 1 evaluates the positions in IEEE binary32 with one stated operation order (the order of the loss
 * path, reading P1, both ways) so that the integer decisions (bounds, nearest pixel, threshold) are the
 * ones an FP32 implementation takes; coord_fp32 = 0 is everything in double.
 * ================================================================================================= */
static int orc_cycle_f64(int W, int H, const double Ki[4], const double Kj[4], const double Tji[12], const double Tij[12],
                         const float* Zj_map, double u, double v, double Zi, double z_min, double tau) {
  double xs[3], xt[3], px[2], back[3], xi[3], q[2];
  orc_backproject_cam(Ki, u, v, Zi, xs);
  for (int r = 0; r < 3; ++r) xt[r] = Tji[4 * r] * xs[0] + Tji[4 * r + 1] * xs[1] + Tji[4 * r + 2] * xs[2] + Tji[4 * r + 3];
  if (!(xt[2] > z_min)) return 0;
  orc_project_px(Kj, xt, px);
  if (!(px[0] >= 0.0 && px[0] <= (double)(W - 1) && px[1] >= 0.0 && px[1] <= (double)(H - 1))) return 0;
  const int xn = (int)floor(px[0] + 0.5), yn = (int)floor(px[1] + 0.5);
  const double Zj = (double)Zj_map[(size_t)yn * W + xn];
  if (!(isfinite(Zj) && Zj > z_min)) return 0;
  orc_backproject_cam(Kj, px[0], px[1], Zj, back);
  for (int r = 0; r < 3; ++r) xi[r] = Tij[4 * r] * back[0] + Tij[4 * r + 1] * back[1] + Tij[4 * r + 2] * back[2] + Tij[4 * r + 3];
  if (!(xi[2] > z_min)) return 0;
  orc_project_px(Ki, xi, q);
  const double dx = q[0] - u, dy = q[1] - v;
  return dx * dx + dy * dy < tau * tau;
}

/* The same cycle with the question "could a correct binary32 evaluation decide this grid point differently?" answered
 * from the double side (reading T1, as orc_pair_event_slack does for the loss): position error radii of a
 * binary32 evaluation of rows a-2..a-4 (|dX| <= 8 u S_X etc., see there), and a point is UNCERTAIN when one of its
 * integer decisions lies within them -- z within |dZ| of z_min (either way), the landing within (r_x, r_y) of the image
 * border or of a half-integer (the nearest pixel, whose depth then differs arbitrarily), or the round-trip error
 * within the accumulated radius of tau.  Returns the decision in bit 0 and "uncertain" in bit 1. */
static int orc_cycle_f64_flag(int W, int H, const double Ki[4], const double Kj[4], const double Tji[12], const double Tij[12],
                              const float* Zj_map, double u, double v, double Zi, double z_min, double tau) {
  const double U32 = 5.9604644775390625e-08;
  double xs[3], xt[3], S3[3], px[2], back[3], xi[3], S3b[3], q[2];
  orc_backproject_cam(Ki, u, v, Zi, xs);
  for (int r = 0; r < 3; ++r) {
    xt[r] = Tji[4 * r] * xs[0] + Tji[4 * r + 1] * xs[1] + Tji[4 * r + 2] * xs[2] + Tji[4 * r + 3];
    S3[r] = fabs(Tji[4 * r] * xs[0]) + fabs(Tji[4 * r + 1] * xs[1]) + fabs(Tji[4 * r + 2] * xs[2]) + fabs(Tji[4 * r + 3]);
  }
  const double eX = 8.0 * U32 * S3[0], eY = 8.0 * U32 * S3[1], eZ = 8.0 * U32 * S3[2];
  if (fabs(xt[2] - z_min) <= eZ) return (xt[2] > z_min ? 0 : 0) | 2;      /* position unbounded: undecidable here */
  if (!(xt[2] > z_min)) return 0;
  orc_project_px(Kj, xt, px);
  const double rx = (Kj[0] * eX + fabs(px[0] - Kj[2]) * eZ) / xt[2] + U32 * (3.0 * fabs(px[0] - Kj[2]) + fabs(px[0]));
  const double ry = (Kj[1] * eY + fabs(px[1] - Kj[3]) * eZ) / xt[2] + U32 * (3.0 * fabs(px[1] - Kj[3]) + fabs(px[1]));
  const double xmax = (double)(W - 1), ymax = (double)(H - 1);
  const int inside = px[0] >= 0.0 && px[0] <= xmax && px[1] >= 0.0 && px[1] <= ymax;
  const int reach = px[0] >= -rx && px[0] <= xmax + rx && px[1] >= -ry && px[1] <= ymax + ry;
  if (!inside) return reach ? 2 : 0;
  int unsure = px[0] < rx || px[0] > xmax - rx || px[1] < ry || px[1] > ymax - ry;
  const double hx = px[0] + 0.5, hy = px[1] + 0.5;
  if (hx - floor(hx) < rx || hx - floor(hx) > 1.0 - rx || hy - floor(hy) < ry || hy - floor(hy) > 1.0 - ry) unsure = 1;
  const int xn = (int)floor(hx), yn = (int)floor(hy);
  const double Zj = (double)Zj_map[(size_t)yn * W + xn];
  if (!(isfinite(Zj) && Zj > z_min)) return unsure ? 2 : 0;
  orc_backproject_cam(Kj, px[0], px[1], Zj, back);
  for (int r = 0; r < 3; ++r) {
    xi[r] = Tij[4 * r] * back[0] + Tij[4 * r + 1] * back[1] + Tij[4 * r + 2] * back[2] + Tij[4 * r + 3];
    S3b[r] = fabs(Tij[4 * r] * back[0]) + fabs(Tij[4 * r + 1] * back[1]) + fabs(Tij[4 * r + 2] * back[2]) + fabs(Tij[4 * r + 3]);
  }
  /* the way back starts from a landing that is itself off by (r_x, r_y): the lifted point moves by Z_j r / f */
  const double sx = Zj * rx / Kj[0], sy = Zj * ry / Kj[1];
  const double fX = 8.0 * U32 * S3b[0] + fabs(Tij[0]) * sx + fabs(Tij[1]) * sy;
  const double fY = 8.0 * U32 * S3b[1] + fabs(Tij[4]) * sx + fabs(Tij[5]) * sy;
  const double fZ = 8.0 * U32 * S3b[2] + fabs(Tij[8]) * sx + fabs(Tij[9]) * sy;
  if (fabs(xi[2] - z_min) <= fZ) return 2;
  if (!(xi[2] > z_min)) return unsure ? 2 : 0;
  orc_project_px(Ki, xi, q);
  const double qx = (Ki[0] * fX + fabs(q[0] - Ki[2]) * fZ) / xi[2] + U32 * (3.0 * fabs(q[0] - Ki[2]) + fabs(q[0]));
  const double qy = (Ki[1] * fY + fabs(q[1] - Ki[3]) * fZ) / xi[2] + U32 * (3.0 * fabs(q[1] - Ki[3]) + fabs(q[1]));
  const double dx = q[0] - u, dy = q[1] - v, err = sqrt(dx * dx + dy * dy);
  if (fabs(err - tau) <= qx + qy + 4.0 * U32 * tau) unsure = 1;
  return (err < tau ? 1 : 0) | (unsure ? 2 : 0);
}

/* counts3 [N][N][3] = {consistent, usable, uncertain} of every ordered pair, everything in double */
void orc_viewgraph_counts_slack(int N, int W, int H, const float* K, const double* poses, const float* depth, int stride,
                                double tau, double z_min, int32_t* counts3) {
#pragma omp parallel for schedule(dynamic)
  for (int ij = 0; ij < N * N; ++ij) {
    const int i = ij / N, j = ij % N;
    int32_t cons = 0, usable = 0, unsure = 0;
    if (i != j) {
      double Ki[4], Kj[4], Tji[12], Tij[12];
      for (int k = 0; k < 4; ++k) { Ki[k] = K[4 * i + k]; Kj[k] = K[4 * j + k]; }
      orc_relative_pose(poses + 12 * i, poses + 12 * j, Tji);
      orc_relative_pose(poses + 12 * j, poses + 12 * i, Tij);
      const float* Zi_map = depth + (size_t)i * W * H;
      const float* Zj_map = depth + (size_t)j * W * H;
      for (int v = stride / 2; v < H; v += stride)
        for (int u = stride / 2; u < W; u += stride) {
          const float Zi = Zi_map[(size_t)v * W + u];
          if (!(isfinite(Zi) && (double)Zi > z_min)) continue;
          ++usable;
          const int f = orc_cycle_f64_flag(W, H, Ki, Kj, Tji, Tij, Zj_map, (double)u, (double)v, (double)Zi, z_min, tau);
          cons += f & 1; unsure += (f >> 1) & 1;
        }
    }
    counts3[3 * ij] = cons; counts3[3 * ij + 1] = usable; counts3[3 * ij + 2] = unsure;
  }
}

/* binary32 positions, operation order:  ifx = 1/fx;  x_s = Z ((u - cx) ifx), y_s likewise, z_s = Z;
 * X = fma(r00, x_s, fma(r01, y_s, fma(r02, z_s, t_x))) (Y, Z likewise);  iz = 1/Z;  x = fma(fx' X, iz, cx');
 * nearest pixel floor(x + 0.5f);  error e2 = fma(dx, dx, dy dy) against tau*tau (one rounded product).          */
static int orc_cycle_f32(int W, int H, const double Ki[4], const double Kj[4], const double Tji[12], const double Tij[12],
                         const float* Zj_map, float u, float v, float Zi, double z_min, double tau) {
  float A[12], B[12];
  for (int k = 0; k < 12; ++k) { A[k] = (float)Tji[k]; B[k] = (float)Tij[k]; }
  const float fxi = (float)Ki[0], fyi = (float)Ki[1], cxi = (float)Ki[2], cyi = (float)Ki[3];
  const float fxj = (float)Kj[0], fyj = (float)Kj[1], cxj = (float)Kj[2], cyj = (float)Kj[3];
  const float zmin = (float)z_min, tauf = (float)tau, tau2 = tauf * tauf;
  const float ifxi = 1.0f / fxi, ifyi = 1.0f / fyi, ifxj = 1.0f / fxj, ifyj = 1.0f / fyj;
  const float a_ = (u - cxi) * ifxi, b_ = (v - cyi) * ifyi;
  const float xs = Zi * a_, ys = Zi * b_, zs = Zi;
  const float X = fmaf(A[0], xs, fmaf(A[1], ys, fmaf(A[2], zs, A[3])));
  const float Y = fmaf(A[4], xs, fmaf(A[5], ys, fmaf(A[6], zs, A[7])));
  const float Z = fmaf(A[8], xs, fmaf(A[9], ys, fmaf(A[10], zs, A[11])));
  if (!(Z > zmin)) return 0;
  const float iz = 1.0f / Z;
  const float fX = fxj * X, fY = fyj * Y;
  const float x = fmaf(fX, iz, cxj), y = fmaf(fY, iz, cyj);
  if (!(x >= 0.0f && x <= (float)(W - 1) && y >= 0.0f && y <= (float)(H - 1))) return 0;
  const float xh = x + 0.5f, yh = y + 0.5f;
  const int xn = (int)floorf(xh), yn = (int)floorf(yh);
  const float Zj = Zj_map[(size_t)yn * W + xn];
  if (!(isfinite(Zj) && Zj > zmin)) return 0;
  const float c_ = (x - cxj) * ifxj, d_ = (y - cyj) * ifyj;
  const float xb = Zj * c_, yb = Zj * d_, zb = Zj;
  const float X2 = fmaf(B[0], xb, fmaf(B[1], yb, fmaf(B[2], zb, B[3])));
  const float Y2 = fmaf(B[4], xb, fmaf(B[5], yb, fmaf(B[6], zb, B[7])));
  const float Z2 = fmaf(B[8], xb, fmaf(B[9], yb, fmaf(B[10], zb, B[11])));
  if (!(Z2 > zmin)) return 0;
  const float iz2 = 1.0f / Z2;
  const float gX = fxi * X2, gY = fyi * Y2;
  const float x2 = fmaf(gX, iz2, cxi), y2 = fmaf(gY, iz2, cyi);
  const float dx = x2 - u, dy = y2 - v;
  const float dy2 = dy * dy;
  const float e2 = fmaf(dx, dx, dy2);
  return e2 < tau2;
}

void orc_viewgraph_counts(int N, int W, int H, const float* K, const double* poses, const float* depth, int stride,
                          double tau, double z_min, int coord_fp32, int32_t* counts) {
#pragma omp parallel for schedule(dynamic)
  for (int ij = 0; ij < N * N; ++ij) {
    const int i = ij / N, j = ij % N;
    int32_t cons = 0, usable = 0;
    if (i != j) {
      double Ki[4], Kj[4], Tji[12], Tij[12];
      for (int k = 0; k < 4; ++k) { Ki[k] = K[4 * i + k]; Kj[k] = K[4 * j + k]; }
      orc_relative_pose(poses + 12 * i, poses + 12 * j, Tji);      /* source i -> target j */
      orc_relative_pose(poses + 12 * j, poses + 12 * i, Tij);      /* and back */
      const float* Zi_map = depth + (size_t)i * W * H;
      const float* Zj_map = depth + (size_t)j * W * H;
      for (int v = stride / 2; v < H; v += stride)
        for (int u = stride / 2; u < W; u += stride) {
          const float Zi = Zi_map[(size_t)v * W + u];
          if (!(isfinite(Zi) && (double)Zi > z_min)) continue;
          ++usable;
          cons += coord_fp32 ? orc_cycle_f32(W, H, Ki, Kj, Tji, Tij, Zj_map, (float)u, (float)v, Zi, z_min, tau)
                             : orc_cycle_f64(W, H, Ki, Kj, Tji, Tij, Zj_map, (double)u, (double)v, (double)Zi, z_min, tau);
        }
    }
    counts[2 * ij] = cons; counts[2 * ij + 1] = usable;
  }
}

/* The viewgraph: unordered pair {i, j} is valid iff BOTH directions keep at least min_frac of their usable grid points
 * (reading V7: the loss uses both directions of a pair, Alg. 3 l.10); output = directed pairs (i, j), (j, i) for
 * i < j ascending.  Returns the number of directed pairs; pairs may be NULL to count only.                         */
int64_t orc_viewgraph_pairs(int N, const int32_t* counts, double min_frac, int32_t* pairs) {
  int64_t n = 0;
  for (int i = 0; i < N; ++i)
    for (int j = i + 1; j < N; ++j) {
      const int32_t *a = counts + 2 * ((size_t)i * N + j), *b = counts + 2 * ((size_t)j * N + i);
      const int ok = a[1] > 0 && b[1] > 0 && (double)a[0] >= min_frac * (double)a[1] && (double)b[0] >= min_frac * (double)b[1];
      if (!ok) continue;
      if (pairs) { pairs[2 * n] = i; pairs[2 * n + 1] = j; pairs[2 * n + 2] = j; pairs[2 * n + 3] = i; }
      n += 2;
    }
  return n;
}

/* ---------------------------------------------------------------------------------------------------------
 * Stochastic viewgraph sub-sampling (Alg. 3 l.3-6; PAPER.md:500 A1.3): "at each iteration we
 * evaluate the loss on a fresh uniform random subset S of E of size min(|E|, M)".
 * The draw is a pure function of (seed, step, pair): pair p (0-based position in the caller's list) gets the key
 *   key(step, p) = output number (step * 2^32 + p + 1) of the SplitMix64 generator seeded with `seed`
 *                = mix(seed + 0x9E3779B97F4A7C15 * (step * 2^32 + p + 1)),
 * and S = the M pairs with the smallest (key, p) -- a uniformly random M-subset (the keys induce a uniformly
 * random order), without replacement, fresh for every step.  Written out as the definition: all keys, a full
 * sort, the first M.  flags[p] = 1 iff pair p is in S; returns |S|.
 * ------------------------------------------------------------------------------------------------------- */
static uint64_t orc_splitmix_output(uint64_t seed, uint64_t n) {
  uint64_t z = seed + 0x9E3779B97F4A7C15ULL * n;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}

uint64_t orc_subset_key(uint64_t seed, int step, int64_t p) {
  return orc_splitmix_output(seed, ((uint64_t)(uint32_t)step << 32) + (uint64_t)p + 1ULL);
}

typedef struct { uint64_t key; int64_t p; } orc_keyed;
static int orc_keyed_cmp(const void* a, const void* b) {
  const orc_keyed *x = (const orc_keyed*)a, *y = (const orc_keyed*)b;
  if (x->key != y->key) return x->key < y->key ? -1 : 1;
  return x->p < y->p ? -1 : (x->p > y->p ? 1 : 0);
}

int64_t orc_pair_subset(uint64_t seed, int step, int64_t P, int64_t M, uint8_t* flags) {
  if (M <= 0 || P <= M) { for (int64_t p = 0; p < P; ++p) flags[p] = 1; return P; }   /* S = E (Alg. 3 l.5) */
  orc_keyed* k = (orc_keyed*)malloc((size_t)P * sizeof(orc_keyed));
  for (int64_t p = 0; p < P; ++p) { k[p].key = orc_subset_key(seed, step, p); k[p].p = p; flags[p] = 0; }
  qsort(k, (size_t)P, sizeof(orc_keyed), orc_keyed_cmp);
  for (int64_t j = 0; j < M; ++j) flags[k[j].p] = 1;
  free(k);
  return M;
}

/* =================================================================================================
 * O7  Schedules, Adam, SE(3) exponential  (readings S4, S10, S11)
 * ================================================================================================= */
/* clamp lambda: clamp_start -> clamp_end linearly over the first clamp_steps steps */
double orc_lambda(int s, double clamp_start, double clamp_end, int clamp_steps) {
  int m = s < clamp_steps ? s : clamp_steps;
  return clamp_start + (clamp_end - clamp_start) * (double)m / (double)clamp_steps;
}
/* "linear learning rate warmup from 0 to 3e-3 over the first 25 steps, followed by cosine annealing
 *  decay over a maximum of N=2000 iterations" */
double orc_lr(int s, double lr_max, int warmup, int max_steps) {
  if (s < warmup) return lr_max * (double)(s + 1) / (double)warmup;
  return lr_max * 0.5 * (1.0 + cos(ORC_PI * (double)(s - warmup) / (double)(max_steps - warmup)));
}

/* Exp(v, w) = [ Exp_SO3(w), V(w) v ; 0, 1 ]; V = I + (1-cos th)/th^2 [w]x + (th - sin th)/th^3 [w]x^2;
 * Taylor forms for th < 1e-4. */
void orc_se3_exp(const double eps[6], double T[12]) {
  const double* v = eps; const double* w = eps + 3;
  double th2 = w[0] * w[0] + w[1] * w[1] + w[2] * w[2], th = sqrt(th2);
  double A, B, C;   /* sin th/th, (1-cos th)/th^2, (th - sin th)/th^3 */
  if (th < 1e-4) { A = 1.0 - th2 / 6.0; B = 0.5 - th2 / 24.0; C = 1.0 / 6.0 - th2 / 120.0; }
  else { A = sin(th) / th; B = (1.0 - cos(th)) / th2; C = (th - sin(th)) / (th2 * th); }
  double Wx[9] = { 0, -w[2], w[1], w[2], 0, -w[0], -w[1], w[0], 0 }, W2[9];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      W2[3 * i + j] = Wx[3 * i] * Wx[j] + Wx[3 * i + 1] * Wx[3 + j] + Wx[3 * i + 2] * Wx[6 + j];
  for (int i = 0; i < 3; ++i) {
    double tv = 0.0;
    for (int j = 0; j < 3; ++j) {
      double I = (i == j) ? 1.0 : 0.0;
      T[4 * i + j] = I + A * Wx[3 * i + j] + B * W2[3 * i + j];
      tv += (I + B * Wx[3 * i + j] + C * W2[3 * i + j]) * v[j];
    }
    T[4 * i + 3] = tv;
  }
}
/* T <- E T for 3x4 [R|t] matrices */
void orc_se3_compose(const double E[12], const double T[12], double out[12]) {
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 4; ++j)
      out[4 * i + j] = E[4 * i] * T[j] + E[4 * i + 1] * T[4 + j] + E[4 * i + 2] * T[8 + j];
    out[4 * i + 3] += E[4 * i + 3];
  }
}
/* One Adam step on the n-vector g (step index s = 0,1,..): returns the increment eps = -lr m^/(sqrt v^ + eps). */
void orc_adam(int n, const double* g, double* m, double* v, int s, double lr, double beta1, double beta2,
              double adam_eps, double* eps_out) {
  double c1 = 1.0 - pow(beta1, (double)(s + 1)), c2 = 1.0 - pow(beta2, (double)(s + 1));
  for (int i = 0; i < n; ++i) {
    m[i] = beta1 * m[i] + (1.0 - beta1) * g[i];
    v[i] = beta2 * v[i] + (1.0 - beta2) * g[i] * g[i];
    eps_out[i] = -lr * (m[i] / c1) / (sqrt(v[i] / c2) + adam_eps);
  }
}

/* AdamW [28] on the joint phase's variables ("All parameters are optimized with the AdamW optimizer with
 * beta1 = 0.9, beta2 = 0.999, and weight decay 0.01"), in place: decoupled decay first, then the Adam step,
 *   p <- p - lr wd (p - p_id) ;  m, v as in Adam ;  p <- p - lr (m / c1) / (sqrt(v / c2) + eps),  c_k = 1 - beta_k^t
 * with t the 1-based count of steps THIS variable group has taken.  p_id is the variable's identity value (gamma: 0,
 * alpha: 1, beta: 0; "initialized to their identity values"): the decay pulls towards it (reading J6;
 * for p_id = 0 this is torch.optim.AdamW exactly).                                                                  */
void orc_adamw(int64_t n, double* p, const double* g, double* m, double* v, int t, double lr, double beta1, double beta2,
               double adam_eps, double wd, double p_id) {
  const double c1 = 1.0 - pow(beta1, (double)t), c2 = 1.0 - pow(beta2, (double)t);
  for (int64_t i = 0; i < n; ++i) {
    p[i] -= lr * wd * (p[i] - p_id);
    m[i] = beta1 * m[i] + (1.0 - beta1) * g[i];
    v[i] = beta2 * v[i] + (1.0 - beta2) * g[i] * g[i];
    p[i] -= lr * (m[i] / c1) / (sqrt(v[i] / c2) + adam_eps);
  }
}

/* =================================================================================================
 * O8  Pose change and the windowed two-phase stopping rule
 * ================================================================================================= */
static double clip1(double c) { return c > 1.0 ? 1.0 : (c < -1.0 ? -1.0 : c); }
/* Eq. 9 */
double orc_delta_R_deg(const double Tcur[12], const double Tprev[12]) {
  double tr = 0.0;                                  /* tr(R^s (R^{s-1})^T) = sum_ij R^s_ij R^{s-1}_ij */
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) tr += Tcur[4 * i + j] * Tprev[4 * i + j];
  return (180.0 / ORC_PI) * acos(clip1((tr - 1.0) / 2.0));
}
/* Eq. 10; 0 if either norm < 1e-12 (reading S13) */
double orc_delta_t_deg(const double Tcur[12], const double Tprev[12]) {
  double a[3] = { Tcur[3], Tcur[7], Tcur[11] }, b[3] = { Tprev[3], Tprev[7], Tprev[11] };
  double na = sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]), nb = sqrt(b[0] * b[0] + b[1] * b[1] + b[2] * b[2]);
  if (na < 1e-12 || nb < 1e-12) return 0.0;
  double c = (a[0] / na) * (b[0] / nb) + (a[1] / na) * (b[1] / nb) + (a[2] / na) * (b[2] / nb);
  return (180.0 / ORC_PI) * acos(clip1(c));
}
static int cmp_double(const void* a, const void* b) {
  double x = *(const double*)a, y = *(const double*)b; return (x > y) - (x < y);
}
/* q-th percentile with linear interpolation at rank q/100 (n-1) (reading S12) */
double orc_percentile(int n, const double* x, double q) {
  double* a = (double*)malloc((size_t)n * sizeof(double));
  memcpy(a, x, (size_t)n * sizeof(double));
  qsort(a, (size_t)n, sizeof(double), cmp_double);
  double rank = q / 100.0 * (double)(n - 1);
  int k = (int)floor(rank); double f = rank - k, r;
  r = (k + 1 < n) ? a[k] + f * (a[k + 1] - a[k]) : a[n - 1];
  free(a); return r;
}
/* theta95 = max(dR95, dt95) */
double orc_theta95(int N, const double* cur, const double* prev) {
  double* dR = (double*)malloc((size_t)N * sizeof(double)); double* dt = (double*)malloc((size_t)N * sizeof(double));
  for (int c = 0; c < N; ++c) { dR[c] = orc_delta_R_deg(cur + 12 * c, prev + 12 * c); dt[c] = orc_delta_t_deg(cur + 12 * c, prev + 12 * c); }
  double r = orc_percentile(N, dR, 95.0), t = orc_percentile(N, dt, 95.0);
  free(dR); free(dt);
  return r > t ? r : t;
}
/* Converged(theta_{0..s}; w, eps).  smooth != 0: moving average of width w, "fires only when every
 * smoothed value in the window is below eps"; smooth == 0: "remains below eps for w
 * consecutive steps".  Reading A2. */
int orc_converged(const double* theta, int s, int w, double eps, int smooth) {
  if (smooth) {
    if (s < 2 * w - 2) return 0;
    for (int k = s - w + 1; k <= s; ++k) {
      double m = 0.0;
      for (int j = k - w + 1; j <= k; ++j) m += theta[j];
      if (!(m / w < eps)) return 0;
    }
    return 1;
  }
  if (s < w - 1) return 0;
  for (int k = s - w + 1; k <= s; ++k) if (!(theta[k] < eps)) return 0;
  return 1;
}

typedef struct {
  double huber_delta, clamp_start, clamp_end; int32_t clamp_steps;
  double lr_max; int32_t warmup_steps, max_steps;
  double beta1, beta2, adam_eps, eps1, eps2; int32_t w1, w2, smooth_window, early_stop;
  double z_min;
  int32_t coord_fp32;   /* 0: everything in double; 1: projected positions decided in fp32 (reading P1) */
  int32_t stop_rule;    /* second-stage stopping rule: 0 pose-based (Eq. 9-10, the paper's), 1 loss-based */
  int32_t w_loss; double eps_loss;   /* 100, 5e-4 */
} orc_config;

/* =================================================================================================
 * The loop of Alg. 2 with the se(3)-Adam parameterisation (reading S9):
 *   for s = start .. : lambda_s -> loss + gradient at the current poses -> Adam -> T_c <- Exp(eps_c) T_c
 *   -> theta95^s vs the previous poses -> Converged tests (phase 0 -> 1 -> 2 = stop).
 * poses [N][12] in/out; m, v [N][6] in/out; theta_hist [max_steps] in/out; *step, *phase in/out.
 * trace_loss[s] = loss at the poses BEFORE update s.  Returns the number of iterations executed.
 * ================================================================================================= */
/* Loss-based stopping criterion (Tab. 7): "monitors relative changes in the loss, stopping when it remains
 * below a threshold eps_2 = 5e-4 for w_2 = 100 consecutive steps".  Relative change of step k >= 1:
 * r_k = |L_k - L_{k-1}| / |L_{k-1}| (infinite if L_{k-1} = 0 and L_k != 0, zero if both are 0); the rule holds at step s
 * iff r_k < eps for the w steps k = s-w+1 .. s, which needs s >= w (reading L1).  It replaces only the SECOND-stage test:
 * "All criteria share the same first stage".                                                                        */
int orc_converged_loss(const double* loss, int s, int w, double eps) {
  if (w < 1 || s < w) return 0;
  for (int k = s - w + 1; k <= s; ++k) {
    const double a = loss[k - 1], d = fabs(loss[k] - a);
    const double r = a != 0.0 ? d / fabs(a) : (d == 0.0 ? 0.0 : INFINITY);
    if (!(r < eps)) return 0;
  }
  return 1;
}

int orc_run(const orc_config* cfg, int n_iters, int N, int W, int H, const float* K, double* poses,
            const int32_t* edge_off, const uint16_t* uv, const float* z, const float* dtf, int64_t P,
            const int32_t* pairs, double* m, double* v, double* theta_hist, double* trace_loss,
            int32_t* step, int32_t* phase, double* poses_log /* nullable [n_iters][N][12] */) {
  double* pl = (double*)malloc((size_t)P * sizeof(double));
  int32_t* pv = (int32_t*)malloc((size_t)P * sizeof(int32_t));
  double* g = (double*)malloc((size_t)N * 6 * sizeof(double));
  double* eps = (double*)malloc((size_t)N * 6 * sizeof(double));
  double* prev = (double*)malloc((size_t)N * 12 * sizeof(double));
  int done = 0;
  while (done < n_iters && *step < cfg->max_steps && !(cfg->early_stop && *phase == 2)) {
    int s = *step; double L;
    double lambda = orc_lambda(s, cfg->clamp_start, cfg->clamp_end, cfg->clamp_steps);
    orc_loss_grad(N, W, H, K, poses, edge_off, uv, z, dtf, P, pairs, lambda, cfg->huber_delta, cfg->z_min,
                  cfg->coord_fp32, pl, pv, NULL, NULL, g, &L);
    trace_loss[s] = L;
    orc_adam(6 * N, g, m, v, s, orc_lr(s, cfg->lr_max, cfg->warmup_steps, cfg->max_steps), cfg->beta1,
             cfg->beta2, cfg->adam_eps, eps);
    memcpy(prev, poses, (size_t)N * 12 * sizeof(double));
    for (int c = 0; c < N; ++c) {
      double E[12], Tn[12];
      orc_se3_exp(eps + 6 * c, E);
      orc_se3_compose(E, prev + 12 * c, Tn);
      memcpy(poses + 12 * c, Tn, sizeof(Tn));
    }
    theta_hist[s] = orc_theta95(N, poses, prev);
    if (*phase == 0) { if (orc_converged(theta_hist, s, cfg->w1, cfg->eps1, cfg->smooth_window)) *phase = 1; }
    else if (*phase == 1) {
      if (cfg->stop_rule == 1 ? orc_converged_loss(trace_loss, s, cfg->w_loss, cfg->eps_loss)
                              : orc_converged(theta_hist, s, cfg->w2, cfg->eps2, cfg->smooth_window)) *phase = 2;
    }
    if (poses_log) memcpy(poses_log + (size_t)done * N * 12, poses, (size_t)N * 12 * sizeof(double));
    *step = s + 1; ++done;
  }
  free(pl); free(pv); free(g); free(eps); free(prev);
  return done;
}
