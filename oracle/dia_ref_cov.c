/* dia_ref_cov.c -- CPU ORACLE, covariance estimate from the observed Fisher information (test infrastructure only).
 *
 * PAPER.md:185-187 (Eq. 16): Sigma = F(theta_MLE)^-1; PAPER.md:189-191 (Eq. 17): uncertainty of parameter p is
 * sqrt(Sigma_pp).  PAPER.md:193: Sigma is valid only if it is positive definite -- "if either the determinant of
 * Sigma is negative, or (after diagonalising the matrix) any eigenvalue is found to be negative or zero, then
 * Sigma is not valid"; both tests are made here exactly as stated:
 *   (1) Sigma by Gauss-Jordan elimination with partial pivoting on [H | 1]; det H = product of the pivots times
 *       the sign of the row permutation, det Sigma = 1 / det H;
 *   (2) eigenvalues of the symmetrised Sigma by the cyclic Jacobi rotation method (diagonalisation).
 * The photometric scale factor is P = sum of the kernel pixels (Eq. 3), a linear function u'theta with
 * u = 1 on the n_kernel kernel parameters and 0 on the background ones, so var P = u' Sigma u (linear error
 * propagation; reading R20).
 * Pins (tests/test_oracle_pins.py): closed-form 2x2 and diagonal cases, numpy.linalg.inv / slogdet / eigvalsh on
 * random SPD and indefinite matrices, H Sigma = 1.
 */
#include "dia_ref.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* Eigenvalues of the symmetric n x n matrix A (destroyed) by cyclic Jacobi sweeps; ev[n] out, unsorted. */
static void jacobi_eigenvalues(double* A, int n, double* ev) {
  for (int sweep = 0; sweep < 100; ++sweep) {
    double off = 0.0, diag = 0.0;
    for (int p = 0; p < n; ++p) {
      diag += A[(size_t)p * n + p] * A[(size_t)p * n + p];
      for (int q = p + 1; q < n; ++q) off += A[(size_t)p * n + q] * A[(size_t)p * n + q];
    }
    if (off <= 1e-30 * diag || off == 0.0) break;
    for (int p = 0; p < n - 1; ++p)
      for (int q = p + 1; q < n; ++q) {
        const double apq = A[(size_t)p * n + q];
        if (apq == 0.0) continue;
        const double app = A[(size_t)p * n + p], aqq = A[(size_t)q * n + q];
        const double tau = (aqq - app) / (2.0 * apq);
        const double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
        const double c = 1.0 / sqrt(1.0 + t * t), s = t * c;
        for (int k = 0; k < n; ++k) {            /* A <- A J   (columns p, q) */
          const double akp = A[(size_t)k * n + p], akq = A[(size_t)k * n + q];
          A[(size_t)k * n + p] = c * akp - s * akq;
          A[(size_t)k * n + q] = s * akp + c * akq;
        }
        for (int k = 0; k < n; ++k) {            /* A <- J' A  (rows p, q) */
          const double apk = A[(size_t)p * n + k], aqk = A[(size_t)q * n + k];
          A[(size_t)p * n + k] = c * apk - s * aqk;
          A[(size_t)q * n + k] = s * apk + c * aqk;
        }
      }
  }
  for (int p = 0; p < n; ++p) ev[p] = A[(size_t)p * n + p];
}

int dia_ref_covariance(int n, int n_kernel, const double* H, double* cov, double* sigma, double* info) {
  if (n < 1 || n_kernel < 0 || n_kernel > n || !H || !cov || !sigma || !info) return DIA_REF_ERR_INVALID_ARG;
  double* A = (double*)malloc(sizeof(double) * (size_t)n * n);
  double* W = (double*)malloc(sizeof(double) * (size_t)n * n);
  double* ev = (double*)malloc(sizeof(double) * (size_t)n);
  if (!A || !W || !ev) { free(A); free(W); free(ev); return DIA_REF_ERR_ALLOC; }
  memcpy(A, H, sizeof(double) * (size_t)n * n);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) cov[(size_t)i * n + j] = (i == j) ? 1.0 : 0.0;

  /* (1) Gauss-Jordan with partial pivoting: A -> 1, cov -> H^-1 */
  double logabsdet = 0.0, sign = 1.0;
  int singular = 0;
  for (int c = 0; c < n && !singular; ++c) {
    int piv = c;
    for (int r = c + 1; r < n; ++r)
      if (fabs(A[(size_t)r * n + c]) > fabs(A[(size_t)piv * n + c])) piv = r;
    if (piv != c) {
      for (int k = 0; k < n; ++k) {
        double t = A[(size_t)c * n + k]; A[(size_t)c * n + k] = A[(size_t)piv * n + k]; A[(size_t)piv * n + k] = t;
        t = cov[(size_t)c * n + k]; cov[(size_t)c * n + k] = cov[(size_t)piv * n + k]; cov[(size_t)piv * n + k] = t;
      }
      sign = -sign;
    }
    const double d = A[(size_t)c * n + c];
    if (d == 0.0 || !isfinite(d)) { singular = 1; break; }
    logabsdet += log(fabs(d));
    if (d < 0.0) sign = -sign;
    for (int k = 0; k < n; ++k) { A[(size_t)c * n + k] /= d; cov[(size_t)c * n + k] /= d; }
    for (int r = 0; r < n; ++r) {
      if (r == c) continue;
      const double f = A[(size_t)r * n + c];
      if (f == 0.0) continue;
      for (int k = 0; k < n; ++k) {
        A[(size_t)r * n + k] -= f * A[(size_t)c * n + k];
        cov[(size_t)r * n + k] -= f * cov[(size_t)c * n + k];
      }
    }
  }

  double min_ev = NAN, var_P = NAN;
  if (!singular) {
    /* (2) diagonalise the symmetrised Sigma */
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) W[(size_t)i * n + j] = 0.5 * (cov[(size_t)i * n + j] + cov[(size_t)j * n + i]);
    jacobi_eigenvalues(W, n, ev);
    min_ev = ev[0];
    for (int p = 1; p < n; ++p) if (ev[p] < min_ev) min_ev = ev[p];
    var_P = 0.0;
    for (int i = 0; i < n_kernel; ++i)
      for (int j = 0; j < n_kernel; ++j) var_P += cov[(size_t)i * n + j];
  }
  for (int p = 0; p < n; ++p) sigma[p] = singular ? NAN : sqrt(cov[(size_t)p * n + p]);   /* NaN if Sigma_pp < 0 */
  info[0] = (!singular && sign > 0.0 && min_ev > 0.0) ? 1.0 : 0.0;   /* det > 0 and all eigenvalues > 0 */
  info[1] = singular ? NAN : logabsdet;                              /* ln |det H| = -ln |det Sigma| */
  info[2] = singular ? NAN : sqrt(var_P);                            /* sigma_P */
  info[3] = min_ev;                                                  /* smallest eigenvalue of Sigma */
  info[4] = singular ? 0.0 : sign;                                   /* sign of det H (= sign of det Sigma) */
  free(A); free(W); free(ev);
  return DIA_REF_OK;
}
