// Helpers of dia_hessian (include/dia.h; Eq. 15-17).  The rows of the Hessian themselves come
// from the fused kernel in Hessian mode (EvalParams::hess_q0, dia_eval.cuh).
#pragma once
#include <cuda_runtime.h>

namespace dia {

constexpr int kHessRows = 32;   // kernel-pixel rows of H per hess_block_kernel launch: 1 forward + 32 gradient passes

struct HessWorkspace {
  double* loss = nullptr;      // [np] scratch for the loss row of the partials (unused in Hessian mode)
  float* ident = nullptr;      // [np][np] identity: unit parameter vectors for the penalty's second derivative
  double* partials = nullptr;  // [kHessRows][np+1][CTAs] block partials of hess_block_kernel (its own: the row count
                               // per launch does not depend on the handle's max_epochs)
  double* chol = nullptr;      // [np][np] Cholesky factor of dia_covariance (L below, L' above the diagonal)
  double* tc_partials = nullptr;   // [CTAs][256][128] FP64 blocks of hess_tc_kernel (dia_hess_tc.cuh), allocated on first use
  int tc_grid = 0;             // CTAs those blocks were sized for
  short* tc_perm = nullptr;    // [128 G] parameter of every operand slot of hess_tc_kernel (hess_tc_make_perm)
};

inline void hess_workspace_destroy(HessWorkspace* w) {
  cudaFree(w->loss); cudaFree(w->ident); cudaFree(w->partials); cudaFree(w->chol); cudaFree(w->tc_partials); cudaFree(w->tc_perm);
  *w = HessWorkspace();
}

__global__ void hess_identity_kernel(float* __restrict__ A, int np) {
  const int total = np * np;
  for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x)
    A[idx] = (idx / np == idx % np) ? 1.f : 0.f;
}

// Entries H[q][nk + t] of the kernel-pixel rows q < nk, which hess_block_kernel leaves at zero: by symmetry the
// entries H[nk + t][q] of the background rows.
__global__ void hess_fill_columns_kernel(double* __restrict__ H, int np, int nk) {
  const int nb = np - nk, total = nk * nb;
  for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
    const int q = idx / nb, t = idx - q * nb;
    H[(size_t)q * np + nk + t] = H[(size_t)(nk + t) * np + q];
  }
}

// H <- (H + H') / 2: rows p and q were accumulated in different FP32 orders
__global__ void hess_symmetrise_kernel(double* __restrict__ H, int np) {
  const int total = np * np;
  for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
    const int p = idx / np, q = idx - p * np;
    if (p < q) {
      const double a = 0.5 * (H[idx] + H[(size_t)q * np + p]);
      H[idx] = a;
      H[(size_t)q * np + p] = a;
    }
  }
}

}  // namespace dia
