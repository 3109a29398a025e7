/* dia_ref_b08.c -- CPU ORACLE, classical B08 normal-equation solve (test infrastructure only).
 *
 * PAPER.md:34 (normal matrix, O(n^2 m^4)), PAPER.md:81 (iterate with fixed sigma estimates,
 * at least 3 iterations), PAPER.md:481/588 (3 iterations, clip |eps| > 5 on the third only).
 * Design columns X_p(i,j) = R[i-h+a][j-h+b] for p = a*m+b, X_{m*m}(i,j) = 1.
 * Iteration 1 takes sigma from Eq. 6 with M := max(I, 0) (reading R10), later iterations from
 * the previous model, floored as in R1.  H = sum_V X X'/v, rhs = sum_V X I/v, Cholesky solve.
 */
#include "dia_ref.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* In-place Cholesky H = L L' (lower), then solve; returns 0 if not positive definite. */
static int cholesky_solve(double* A, double* x, int n) {
  for (int j = 0; j < n; ++j) {
    double s = A[(size_t)j * n + j];
    for (int k = 0; k < j; ++k) s -= A[(size_t)j * n + k] * A[(size_t)j * n + k];
    if (!(s > 0.0)) return 0;
    const double ljj = sqrt(s);
    A[(size_t)j * n + j] = ljj;
    for (int i = j + 1; i < n; ++i) {
      double t = A[(size_t)i * n + j];
      for (int k = 0; k < j; ++k) t -= A[(size_t)i * n + k] * A[(size_t)j * n + k];
      A[(size_t)i * n + j] = t / ljj;
    }
  }
  for (int i = 0; i < n; ++i) {           /* L y = b */
    double t = x[i];
    for (int k = 0; k < i; ++k) t -= A[(size_t)i * n + k] * x[k];
    x[i] = t / A[(size_t)i * n + i];
  }
  for (int i = n - 1; i >= 0; --i) {      /* L' x = y */
    double t = x[i];
    for (int k = i + 1; k < n; ++k) t -= A[(size_t)k * n + i] * x[k];
    x[i] = t / A[(size_t)i * n + i];
  }
  return 1;
}

int dia_ref_b08_solve(const dia_ref_config* cfg, const float* R, const float* I,
                      const unsigned char* mask, const float* var_fixed, int n_iters,
                      int clip_last, double* theta, double* H_out) {
  if (!cfg || !R || !I || !theta || n_iters < 1) return DIA_REF_ERR_INVALID_ARG;
  if (cfg->m < 1 || cfg->m % 2 == 0 || cfg->n_rows < cfg->m || cfg->n_cols < cfg->m) return DIA_REF_ERR_INVALID_ARG;
  const int m = cfg->m, h = (m - 1) / 2, np = m * m + 1;
  const int nr = cfg->n_rows, nc = cfg->n_cols;
  double* H = (double*)malloc(sizeof(double) * (size_t)np * np);
  double* Hc = (double*)malloc(sizeof(double) * (size_t)np * np);
  double* rhs = (double*)malloc(sizeof(double) * np);
  double* X = (double*)malloc(sizeof(double) * np);
  if (!H || !Hc || !rhs || !X) return DIA_REF_ERR_ALLOC;
  int rc = DIA_REF_OK;
  for (int it = 1; it <= n_iters; ++it) {
    memset(H, 0, sizeof(double) * (size_t)np * np);
    memset(rhs, 0, sizeof(double) * np);
    for (int i = h; i < nr - h; ++i)
      for (int j = h; j < nc - h; ++j) {
        const size_t p = (size_t)i * nc + j;
        if (mask && mask[p] == 0) continue;
        for (int a = 0; a < m; ++a)
          for (int b = 0; b < m; ++b)
            X[a * m + b] = (double)R[(size_t)(i - h + a) * nc + (j - h + b)];
        X[m * m] = 1.0;
        double Mprev = 0.0;
        if (it > 1) for (int q = 0; q < np; ++q) Mprev += theta[q] * X[q];
        double v;
        if (var_fixed) {
          v = (double)var_fixed[p];
        } else {
          const double F = cfg->flat ? (double)cfg->flat[p] : 1.0;
          const double Mv = (it == 1) ? (double)I[p] : Mprev;        /* R10 */
          v = cfg->sigma0 * cfg->sigma0 / (F * F) + (Mv > 0.0 ? Mv : 0.0) / (cfg->gain * F);
        }
        if (clip_last && it == n_iters && it > 1) {
          const double eps = ((double)I[p] - Mprev) / sqrt(v);
          if (fabs(eps) > 5.0) continue;
        }
        const double iv = 1.0 / v;
        for (int q = 0; q < np; ++q) {
          const double xq = X[q] * iv;
          rhs[q] += xq * (double)I[p];
          for (int s = q; s < np; ++s) H[(size_t)q * np + s] += xq * X[s];   /* upper triangle */
        }
      }
    for (int q = 0; q < np; ++q)
      for (int s = 0; s < q; ++s) H[(size_t)q * np + s] = H[(size_t)s * np + q];
    memcpy(Hc, H, sizeof(double) * (size_t)np * np);
    for (int q = 0; q < np; ++q) theta[q] = rhs[q];
    if (!cholesky_solve(Hc, theta, np)) { rc = DIA_REF_ERR_NOT_PD; break; }
  }
  if (H_out) memcpy(H_out, H, sizeof(double) * (size_t)np * np);
  free(H); free(Hc); free(rhs); free(X);
  return rc;
}
