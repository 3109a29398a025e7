// Kernels of dia_covariance (include/dia.h): covariance estimate Sigma = H^-1 of Eq. 16-17 with
// the validity test of PAPER.md:193, all in FP64 on the device.
//
// H = L L' by a left-looking Cholesky factorisation, one launch per column (column j needs columns 0..j-1 complete;
// inside a launch one warp owns one row i > j and forms the dot product of rows i and j of L).  A symmetric matrix is
// positive definite -- every eigenvalue positive, hence a positive determinant: the two tests the paper lists --
// exactly when every pivot d_j = H_jj - sum_k L_jk^2 is positive, so the pivots are the test (R20).
// L is stored in the lower triangle of the workspace W and L' in its upper triangle, so that both triangular solves
// read rows.  Then one warp per right-hand side: y = L^-1 e_k (forward), sigma_k = |y| (Sigma_kk = e_k' L^-T L^-1 e_k),
// x = L^-T y (backward) = row k of Sigma; one more warp solves for u (1 on the kernel pixels, Eq. 3) and gives
// sigma_P = |L^-1 u|.  Every sum has a fixed order (lane-strided partial sums, then a butterfly): bit-reproducible.
#pragma once
#include <cuda_runtime.h>

#include "dia_eval.cuh"   // warp_sum_f64

namespace dia {

constexpr int kCholWarps = 8;    // rows per CTA in chol_column_kernel
constexpr int kSolveWarps = 2;   // right-hand sides per CTA in cov_solve_kernel
constexpr int kCovInfo = 5;      // valid, ln det H, sigma_P, smallest pivot, first non-positive pivot (-1: none)

__global__ void cov_init_kernel(double* __restrict__ info) {
  info[0] = 1.0;  info[1] = 0.0;  info[2] = 0.0;  info[3] = INFINITY;  info[4] = -1.0;
}

// column j of L.  grid: ceil((np - 1 - j) / kCholWarps) CTAs (at least one), kCholWarps warps; smem: j doubles
__global__ void __launch_bounds__(kCholWarps * 32)
chol_column_kernel(const double* __restrict__ H, double* __restrict__ W, int np, int j, double* __restrict__ info) {
  extern __shared__ double rowj[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const double* Wj = W + (size_t)j * np;
  for (int k = threadIdx.x; k < j; k += blockDim.x) rowj[k] = Wj[k];
  __syncthreads();
  double s = 0.0;
  for (int k = lane; k < j; k += 32) s = fma(rowj[k], rowj[k], s);
  const double d = H[(size_t)j * np + j] - warp_sum_f64(s);   // the same value in every warp of every CTA
  const double ljj = sqrt(d);                                  // NaN from here on if d < 0: info[0] says so
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    W[(size_t)j * np + j] = ljj;
    if (!(d > 0.0) || !isfinite(d)) {
      if (info[4] < 0.0) info[4] = (double)j;
      info[0] = 0.0;
    }
    info[1] += log(d);
    if (d < info[3]) info[3] = d;                              // NaN pivots after a failure leave it alone
  }
  const int i = j + 1 + blockIdx.x * kCholWarps + warp;
  if (i >= np) return;
  const double* Wi = W + (size_t)i * np;
  double t = 0.0;
  for (int k = lane; k < j; k += 32) t = fma(Wi[k], rowj[k], t);
  t = warp_sum_f64(t);
  if (lane == 0) {
    const double l = (H[(size_t)i * np + j] - t) / ljj;
    W[(size_t)i * np + j] = l;
    W[(size_t)j * np + i] = l;
  }
}

// warp r < np: right-hand side e_r; warp r == np: u.  smem: kSolveWarps x np doubles.
__global__ void __launch_bounds__(kSolveWarps * 32)
cov_solve_kernel(const double* __restrict__ W, int np, int n_kernel, double* __restrict__ cov,
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

}  // namespace dia
