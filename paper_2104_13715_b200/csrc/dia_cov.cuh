// Kernels of dia_covariance (include/dia.h): covariance estimate Sigma = H^-1 of Eq. 16-17 with
// the validity test of PAPER.md:193, all in FP64 on the device.
//
// H = L L' by a blocked left-looking Cholesky factorisation, two launches per panel of kCholPanel = 32 columns (12
// panels at np = 362, 70 at np = 2219; the unblocked form took one launch per column):
//   chol_panel_update_kernel  one warp per row i >= j0: P[i][c] = H[i][j0+c] - sum_{k<j0} L[i][k] L[j0+c][k] for the 32
//                             columns of the panel (the panel's rows of L staged through shared memory in chunks of k);
//   chol_panel_factor_kernel  every CTA factorises the 32 x 32 diagonal block of P in shared memory (redundantly: it is
//                             32 short steps), then one warp per row below solves l_i L_dd' = P_i.
// A symmetric matrix is positive definite -- every eigenvalue positive, hence a positive determinant: the two tests
// the paper lists -- exactly when every pivot d_j = H_jj - sum_k L_jk^2 is positive, so the pivots are the test
// (R20).
// L is stored in the lower triangle of the workspace W and L' in its upper triangle, so that both triangular solves
// read contiguous rows.  Then one warp per right-hand side (cov_solve_warp): y = L^-1 e_k (forward), sigma_k = |y|
// (Sigma_kk = e_k' L^-T L^-1 e_k), x = L^-T y (backward) = row k of Sigma; one more warp solves for u (1 on the kernel
// pixels, Eq. 3) and gives sigma_P = |L^-1 u|.  Every sum has a fixed order: bit-reproducible.
#pragma once
#include <cuda_runtime.h>

#include "dia_eval.cuh"   // warp_sum_f64

namespace dia {

constexpr int kCholWarps = 8;    // rows per CTA in the Cholesky kernels
constexpr int kSolveWarps = 4;   // right-hand sides per CTA in cov_solve_kernel
constexpr int kCovInfo = 5;      // valid, ln det H, sigma_P, smallest pivot, first non-positive pivot (-1: none)

__global__ void cov_init_kernel(double* __restrict__ info) {
  info[0] = 1.0;  info[1] = 0.0;  info[2] = 0.0;  info[3] = INFINITY;  info[4] = -1.0;
}

constexpr int kCholPanel = 32;   // columns per panel
constexpr int kCholChunk = 128;  // k values of the panel's rows staged per pass of the update kernel

// P[i][c] for rows i >= j0 and the nb columns of the panel: the rows below the diagonal block are written over
// W[i][j0+c], the block itself (c <= i - j0) goes to `diag` [kCholPanel][kCholPanel] -- every CTA of the factor
// kernel reads it while CTA 0 writes the factorised block into W.
// grid: ceil((np - j0) / kCholWarps) CTAs of kCholWarps warps; smem: kCholPanel x kCholChunk doubles.
__global__ void __launch_bounds__(kCholWarps * 32)
chol_panel_update_kernel(const double* __restrict__ H, double* __restrict__ W, double* __restrict__ diag, int np, int j0,
                         int nb) {
  __shared__ double S[kCholPanel][kCholChunk + 1];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int i = j0 + blockIdx.x * kCholWarps + warp;
  const bool live = i < np;
  const double* Wi = W + (size_t)(live ? i : j0) * np;
  double t[kCholPanel];
#pragma unroll
  for (int c = 0; c < kCholPanel; ++c) t[c] = 0.0;
  for (int k0 = 0; k0 < j0; k0 += kCholChunk) {
    const int kn = min(kCholChunk, j0 - k0);
    __syncthreads();
    for (int idx = threadIdx.x; idx < kCholPanel * kCholChunk; idx += blockDim.x) {
      const int c = idx / kCholChunk, k = idx - c * kCholChunk;
      S[c][k] = (c < nb && k < kn) ? W[(size_t)(j0 + c) * np + k0 + k] : 0.0;
    }
    __syncthreads();
    for (int k = lane; k < kn; k += 32) {
      const double a = Wi[k0 + k];
#pragma unroll
      for (int c = 0; c < kCholPanel; ++c) t[c] = fma(a, S[c][k], t[c]);
    }
  }
#pragma unroll
  for (int c = 0; c < kCholPanel; ++c) t[c] = warp_sum_f64(t[c]);
  if (!live) return;
  double mine = 0.0;                                  // lane c keeps column c
#pragma unroll
  for (int c = 0; c < kCholPanel; ++c) if (lane == c) mine = t[c];
  if (lane < nb && j0 + lane <= i) {
    const double v = H[(size_t)i * np + j0 + lane] - mine;
    if (i < j0 + nb) diag[(i - j0) * kCholPanel + lane] = v;
    else W[(size_t)i * np + j0 + lane] = v;
  }
}

// Factorises the diagonal block of the panel and solves the rows below it.  grid: max(1, ceil((np - j0 - nb) /
// kCholWarps)) CTAs of kCholWarps warps.  CTA 0 writes the block itself and the pivots' record.
__global__ void __launch_bounds__(kCholWarps * 32)
chol_panel_factor_kernel(double* __restrict__ W, const double* __restrict__ diag, int np, int j0, int nb,
                         double* __restrict__ info) {
  __shared__ double D[kCholPanel][kCholPanel + 1];
  __shared__ double piv[kCholPanel];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int idx = threadIdx.x; idx < kCholPanel * kCholPanel; idx += blockDim.x) {
    const int r = idx / kCholPanel, c = idx - r * kCholPanel;
    D[r][c] = (r < nb && c <= r) ? diag[r * kCholPanel + c] : 0.0;
  }
  __syncthreads();
  if (warp == 0) {                                    // lane r owns row r of the block
    for (int c = 0; c < nb; ++c) {
      double s = 0.0;
      for (int k = 0; k < c; ++k) s = fma(D[c][k], D[c][k], s);
      const double d = D[c][c] - s;                   // the same value in every lane
      const double lcc = sqrt(d);                     // NaN from here on if d < 0: info[0] says so
      double v = 0.0;
      if (lane > c && lane < nb) {
        double tt = 0.0;
        for (int k = 0; k < c; ++k) tt = fma(D[lane][k], D[c][k], tt);
        v = (D[lane][c] - tt) / lcc;
      }
      __syncwarp();
      if (lane == c) { D[c][c] = lcc;  piv[c] = d; }
      if (lane > c && lane < nb) D[lane][c] = v;
      __syncwarp();
    }
  }
  __syncthreads();
  if (blockIdx.x == 0) {
    for (int idx = threadIdx.x; idx < nb * nb; idx += blockDim.x) {
      const int r = idx / nb, c = idx - r * nb;
      if (c <= r) {
        W[(size_t)(j0 + r) * np + j0 + c] = D[r][c];
        W[(size_t)(j0 + c) * np + j0 + r] = D[r][c];
      }
    }
    if (threadIdx.x == 0) {
      for (int c = 0; c < nb; ++c) {
        const double d = piv[c];
        if (!(d > 0.0) || !isfinite(d)) {
          if (info[4] < 0.0) info[4] = (double)(j0 + c);
          info[0] = 0.0;
        }
        info[1] += log(d);
        if (d < info[3]) info[3] = d;                 // NaN pivots after a failure leave it alone
      }
    }
  }
  const int i = j0 + nb + blockIdx.x * kCholWarps + warp;
  if (i >= np) return;
  double* Wi = W + (size_t)i * np + j0;
  const double pc = lane < nb ? Wi[lane] : 0.0;       // P[i][lane]
  double l = 0.0;                                     // l[lane] once column lane is done
  for (int c = 0; c < nb; ++c) {
    const double t = warp_sum_f64((lane < c) ? l * D[c][lane] : 0.0);
    if (lane == c) l = (pc - t) / D[c][c];
  }
  if (lane < nb) {
    Wi[lane] = l;
    W[(size_t)(j0 + lane) * np + i] = l;
  }
}

// The two triangular solves of one right-hand side by one warp, column by column: the vector lives in registers
// (element k in lane k % 32, slot k / 32; S slots), step i takes y_i = b_i / L_ii from its owner lane by a shuffle and
// subtracts y_i times column i of L from the elements below -- no dot product, hence no butterfly in the chain of np
// dependent steps (the row-oriented form spent ~900 cycles per step on it: 0.65 ms at np = 362; this one 0.1 ms).
// Column i of L is row i of the upper triangle of W (L' is stored there) and row i of L serves the backward solve, so
// every load is contiguous; the next step's column is requested while the current one is applied (PF).
// warp r < np: right-hand side e_r -> sigma[r] = |L^-1 e_r| and row r of the covariance; warp r == np: u (1 on the
// kernel pixels) -> info[2] = sigma_P.  invd [np]: 1 / L_ii in shared memory.
template <int S, bool PF>
__device__ __forceinline__ void cov_solve_warp(const double* __restrict__ W, const double* __restrict__ invd, int np, int n_kernel,
                                               int r, double* __restrict__ cov, double* __restrict__ sigma,
                                               double* __restrict__ info) {
  const int lane = threadIdx.x & 31;
  const bool unit = r < np;
  const int i0 = unit ? r : 0;                       // y_i = 0 above the first non-zero of the right-hand side
  double b[S], c[S], cn[S];
#pragma unroll
  for (int t = 0; t < S; ++t) {
    const int k = 32 * t + lane;
    b[t] = (k < np && (unit ? k == r : k < n_kernel)) ? 1.0 : 0.0;
    c[t] = 0.0;  cn[t] = 0.0;
  }
  auto load = [&](int i, int t_lo, int t_hi, double* dst) {      // elements of row i of W in slots t_lo .. t_hi
#pragma unroll
    for (int t = 0; t < S; ++t) {
      const int k = 32 * t + lane;
      if (t >= t_lo && t <= t_hi && k < np) dst[t] = W[(size_t)i * np + k];
    }
  };
  double norm2 = 0.0;
  if (PF) load(i0, i0 >> 5, S - 1, c);
#pragma unroll
  for (int s = 0; s < S; ++s) {                      // forward: L y = b, y overwrites b
    if (32 * s + 31 < i0 || 32 * s >= np) continue;
#pragma unroll 1
    for (int l = 0; l < 32; ++l) {
      const int i = 32 * s + l;
      if (i < i0 || i >= np) continue;
      if (PF) { if (i + 1 < np) load(i + 1, (i + 1) >> 5, S - 1, cn); }
      else load(i, s, S - 1, c);
      const double yi = __shfl_sync(0xffffffffu, b[s], l) * invd[i];
      norm2 = fma(yi, yi, norm2);
      if (lane == l) b[s] = yi;
#pragma unroll
      for (int t = s; t < S; ++t) {
        const int k = 32 * t + lane;
        if (k > i && k < np) b[t] = fma(-yi, c[t], b[t]);
        if (PF) c[t] = cn[t];
      }
    }
  }
  if (lane == 0) {
    if (unit) sigma[r] = sqrt(norm2); else info[2] = sqrt(norm2);
  }
  if (!unit || !cov) return;
  if (PF) load(np - 1, 0, (np - 1) >> 5, c);
#pragma unroll
  for (int s = S - 1; s >= 0; --s) {                 // backward: L' x = y, x overwrites b; row i of L: W[i][k], k < i
    if (32 * s >= np) continue;
#pragma unroll 1
    for (int l = 31; l >= 0; --l) {
      const int i = 32 * s + l;
      if (i >= np) continue;
      if (PF) { if (i > 0) load(i - 1, 0, (i - 1) >> 5, cn); }
      else load(i, 0, s, c);
      const double xi = __shfl_sync(0xffffffffu, b[s], l) * invd[i];
      if (lane == l) b[s] = xi;
#pragma unroll
      for (int t = 0; t <= s; ++t) {
        const int k = 32 * t + lane;
        if (k < i) b[t] = fma(-xi, c[t], b[t]);
        if (PF) c[t] = cn[t];
      }
    }
  }
  double* out = cov + (size_t)r * np;
#pragma unroll
  for (int t = 0; t < S; ++t) { const int k = 32 * t + lane; if (k < np) out[k] = b[t]; }
}

// grid: ceil((np + 1) / kSolveWarps) CTAs of kSolveWarps warps; smem: np doubles (1 / L_ii)
template <int S, bool PF>
__global__ void __launch_bounds__(kSolveWarps * 32)
cov_solve_kernel(const double* __restrict__ W, int np, int n_kernel, double* __restrict__ cov,
                 double* __restrict__ sigma, double* __restrict__ info) {
  extern __shared__ double invd[];
  for (int i = threadIdx.x; i < np; i += blockDim.x) invd[i] = 1.0 / W[(size_t)i * np + i];
  __syncthreads();
  const int r = blockIdx.x * kSolveWarps + (threadIdx.x >> 5);
  if (r > np) return;
  cov_solve_warp<S, PF>(W, invd, np, n_kernel, r, cov, sigma, info);
}

// The row-oriented form of the same solves for np > 1536 (48 register slots per lane are the most that pay):
// the vector in shared memory, one dot product (lane-strided partial sums, a butterfly) per step.
// warp r < np: right-hand side e_r; warp r == np: u.  smem: kSolveWarps x np doubles.
__global__ void __launch_bounds__(kSolveWarps * 32)
cov_solve_rows_kernel(const double* __restrict__ W, int np, int n_kernel, double* __restrict__ cov,
                 double* __restrict__ sigma, double* __restrict__ info) {
  extern __shared__ double ysm[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int r = blockIdx.x * kSolveWarps + warp;
  if (r > np) return;
  double* y = ysm + (size_t)warp * np;
  const bool unit = r < np;
  const int i0 = unit ? r : 0;                       // y_i = 0 above the first non-zero of the right-hand side
  for (int i = lane; i < i0; i += 32) y[i] = 0.0;
  double norm2 = 0.0;
  for (int i = i0; i < np; ++i) {                    // L y = b
    const double* Wi = W + (size_t)i * np;
    double t = 0.0;
    for (int k = i0 + lane; k < i; k += 32) t = fma(Wi[k], y[k], t);
    t = warp_sum_f64(t);
    const double b = unit ? (i == r ? 1.0 : 0.0) : (i < n_kernel ? 1.0 : 0.0);
    const double yi = (b - t) / Wi[i];
    norm2 = fma(yi, yi, norm2);
    if (lane == 0) y[i] = yi;
    __syncwarp();
  }
  if (lane == 0) {
    if (unit) sigma[r] = sqrt(norm2); else info[2] = sqrt(norm2);
  }
  if (!unit || !cov) return;
  for (int i = np - 1; i >= 0; --i) {                // L' x = y, x overwrites y
    const double* Wi = W + (size_t)i * np;           // row i of the upper triangle = column i of L
    double t = 0.0;
    for (int k = i + 1 + lane; k < np; k += 32) t = fma(Wi[k], y[k], t);
    t = warp_sum_f64(t);
    if (lane == 0) y[i] = (y[i] - t) / Wi[i];
    __syncwarp();
  }
  double* out = cov + (size_t)r * np;
  for (int i = lane; i < np; i += 32) out[i] = y[i];
}

// the instantiation for np parameters (slots of 32): prefetch of the next column while it fits the register file
inline const void* cov_solve_kernel_for(int np, size_t* smem_bytes) {
  const int s = (np + 31) / 32;
  *smem_bytes = sizeof(double) * (size_t)np;
  if (s <= 2) return (const void*)cov_solve_kernel<2, true>;
  if (s <= 4) return (const void*)cov_solve_kernel<4, true>;
  if (s <= 8) return (const void*)cov_solve_kernel<8, true>;
  if (s <= 12) return (const void*)cov_solve_kernel<12, true>;
  if (s <= 20) return (const void*)cov_solve_kernel<20, true>;
  if (s <= 32) return (const void*)cov_solve_kernel<32, false>;        // measured at np = 730 / 1090 / 2210 (ms per
  if (s <= 48) return (const void*)cov_solve_kernel<48, false>;        // dia_covariance): 1.8 / 3.1 / 30.8 against
  *smem_bytes = sizeof(double) * (size_t)kSolveWarps * np;              // 2.9 / 5.1 / 18.5 for the row form
  return (const void*)cov_solve_rows_kernel;
}

}  // namespace dia
