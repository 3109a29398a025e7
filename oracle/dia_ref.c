/* dia_ref.c -- CPU ORACLE (test infrastructure only; see dia_ref.h).
 *
 * Plain FP64 loops in the paper's order and notation.  No blocking, fusion or reordering
 * beyond what the definitions state; OpenMP (optional) splits image rows over threads and
 * sums per-thread partials in thread-index order, so results are deterministic for a fixed
 * thread count.
 */
#include "dia_ref.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int dia_ref_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

static int check_cfg(const dia_ref_config* c) {
  if (!c) return 0;
  if (c->m < 1 || (c->m % 2) == 0) return 0;
  if (c->n_rows < c->m || c->n_cols < c->m) return 0;
  if (c->loss != DIA_REF_LOSS_GAUSSIAN && c->loss != DIA_REF_LOSS_HUBER) return 0;
  if (c->noise != DIA_REF_NOISE_MODEL && c->noise != DIA_REF_NOISE_FIXED) return 0;
  if (c->noise == DIA_REF_NOISE_MODEL && !(c->gain > 0.0 && c->sigma0 >= 0.0)) return 0;
  if (c->loss == DIA_REF_LOSS_HUBER && !(c->huber_c > 0.0)) return 0;
  if (c->bg_degree < 0 || c->bg_degree > 4) return 0;
  return 1;
}

int dia_ref_num_params(const dia_ref_config* cfg) {
  const int d = cfg->bg_degree > 0 ? cfg->bg_degree : 0;
  return cfg->m * cfg->m + (d + 1) * (d + 2) / 2;
}

/* Eq. 18-19: B(x, y) = sum_{m=0..d} sum_{n=0..d-m} b_mn eta^m xi^n with the normalised
 * coordinates eta = (x - x_c)/N_x, xi = (y - y_c)/N_y.  Readings (R18): x = column index j, y = row
 * index i, centre (x_c, y_c) = ((n_cols-1)/2, (n_rows-1)/2).  basis (nullable) receives eta^m xi^n in the
 * coefficient order, which is also dB/db_mn. */
static double background(const dia_ref_config* cfg, const float* b, int i, int j, double* basis) {
  const int d = cfg->bg_degree > 0 ? cfg->bg_degree : 0;
  const double eta = ((double)j - 0.5 * (cfg->n_cols - 1)) / (double)cfg->n_cols;
  const double xi = ((double)i - 0.5 * (cfg->n_rows - 1)) / (double)cfg->n_rows;
  double B = 0.0;
  int t = 0;
  for (int mm = 0; mm <= d; ++mm)
    for (int nn = 0; nn <= d - mm; ++nn, ++t) {
      const double f = pow(eta, mm) * pow(xi, nn);
      if (basis) basis[t] = f;
      B += (double)b[t] * f;
    }
  return B;
}

/* Eq. 2: M_ij = sum_lm K_lm R_(i+l)(j+m) + B0, cross-correlation, no flip
 * (reading R2).  (i, j) are image coordinates of a valid pixel. */
static double model_pixel(const dia_ref_config* cfg, const float* R, int n_cols, int m, const float* theta, int i, int j) {
  const int h = (m - 1) / 2;
  double M = 0.0;
  for (int a = 0; a < m; ++a)
    for (int b = 0; b < m; ++b)
      M += (double)theta[a * m + b] * (double)R[(size_t)(i - h + a) * n_cols + (j - h + b)];
  return M + background(cfg, theta + m * m, i, j, NULL);     /* B0, or Eq. 18 */
}

int dia_ref_model(const dia_ref_config* cfg, const float* R, const float* theta, double* M) {
  if (!check_cfg(cfg) || !R || !theta || !M) return DIA_REF_ERR_INVALID_ARG;
  const int m = cfg->m, h = (m - 1) / 2;
  const int vr = cfg->n_rows - m + 1, vc = cfg->n_cols - m + 1;
#pragma omp parallel for schedule(static)
  for (int i = 0; i < vr; ++i)
    for (int j = 0; j < vc; ++j)
      M[(size_t)i * vc + j] = model_pixel(cfg, R, cfg->n_cols, m, theta, i + h, j + h);
  return DIA_REF_OK;
}

/* One epoch of c.1.  part_* are per-call scratch of size (m*m+1). */
static void eval_one(const dia_ref_config* cfg, const float* R, const float* I,
                     const unsigned char* mask, const float* var, const float* theta,
                     double* loss_out, double* grad, double* gscale) {
  const int m = cfg->m, h = (m - 1) / 2, np = dia_ref_num_params(cfg), nbg = np - m * m;
  const int nr = cfg->n_rows, nc = cfg->n_cols;
  int nthreads = dia_ref_num_threads();
  double* tl = (double*)calloc((size_t)nthreads, sizeof(double));
  double* tg = (double*)calloc((size_t)nthreads * np, sizeof(double));
  double* ts = (double*)calloc((size_t)nthreads * np, sizeof(double));

#pragma omp parallel
  {
#ifdef _OPENMP
    const int tid = omp_get_thread_num();
#else
    const int tid = 0;
#endif
    double L = 0.0;
    double* g = tg + (size_t)tid * np;
    double* s = ts + (size_t)tid * np;
#pragma omp for schedule(static)
    for (int i = h; i < nr - h; ++i) {
      for (int j = h; j < nc - h; ++j) {
        const size_t p = (size_t)i * nc + j;
        if (mask && mask[p] == 0) continue;                 /* reading R4 */
        const double M = model_pixel(cfg, R, nc, m, theta, i, j);
        double v, bp;
        if (cfg->noise == DIA_REF_NOISE_MODEL) {
          /* Eq. 6: sigma^2 = sigma0^2/F^2 + M/(G F); reading R1: photon
           * term uses max(M, 0) and its derivative is 0 there. */
          const double F = cfg->flat ? (double)cfg->flat[p] : 1.0;
          const double a_ij = cfg->sigma0 * cfg->sigma0 / (F * F);
          const double b_ij = 1.0 / (cfg->gain * F);
          v = a_ij + b_ij * (M > 0.0 ? M : 0.0);
          bp = (M > 0.0) ? b_ij : 0.0;
        } else {
          v = (double)var[p];
          bp = 0.0;
        }
        const double r = (double)I[p] - M;
        const double sd = sqrt(v);
        const double z = r / sd;
        double rho, psi;
        if (cfg->loss == DIA_REF_LOSS_HUBER && fabs(z) > cfg->huber_c) {
          /* Eq. 12 */
          rho = cfg->huber_c * (fabs(z) - 0.5 * cfg->huber_c);
          psi = (z > 0.0) ? cfg->huber_c : -cfg->huber_c;
        } else {
          rho = 0.5 * z * z;
          psi = z;
        }
        /* Eq. 8 / Eq. 13 without theta-independent constants (reading R3); in FIXED mode
         * sum ln sigma is a constant and is dropped. */
        L += rho;
        if (cfg->noise == DIA_REF_NOISE_MODEL) L += 0.5 * log(v);
        /* D1: w = dL/dM = -psi/s - psi z b'/(2v) + b'/(2v) */
        const double w = -psi / sd - psi * z * bp / (2.0 * v) + bp / (2.0 * v);
        const double aw = fabs(w);
        for (int a = 0; a < m; ++a)
          for (int b = 0; b < m; ++b) {
            const double x = (double)R[(size_t)(i - h + a) * nc + (j - h + b)];
            g[a * m + b] += w * x;
            s[a * m + b] += aw * fabs(x);
          }
        double basis[16];
        background(cfg, theta + m * m, i, j, basis);          /* dM/db_mn = eta^m xi^n (1 for B0) */
        for (int t = 0; t < nbg; ++t) {
          g[m * m + t] += w * basis[t];
          s[m * m + t] += aw * fabs(basis[t]);
        }
      }
    }
    tl[tid] = L;
  }
  double L = 0.0;
  for (int t = 0; t < nthreads; ++t) L += tl[t];
  *loss_out = L;
  for (int k = 0; k < np; ++k) {
    double gs = 0.0, ss = 0.0;
    for (int t = 0; t < nthreads; ++t) {
      gs += tg[(size_t)t * np + k];
      ss += ts[(size_t)t * np + k];
    }
    grad[k] = gs;
    if (gscale) gscale[k] = ss;
  }
  free(tl); free(tg); free(ts);
}

/* Eq. 20-21: penalty lambda N_data theta' L' L theta with L the graph Laplacian of the
 * kernel pixels (L_uu = number of adjacent kernel pixels, L_uv = -1 for adjacent u, v; the B0 row and
 * column are zero).  Readings (R14): "adjacent" = the 4 edge neighbours inside the m x m grid;
 * N_data = number of valid-region pixels (n_rows-m+1)(n_cols-m+1).  L is symmetric, so the penalty is
 * lambda N |L theta|^2 and its gradient 2 lambda N L (L theta).  Adds to *loss and grad[0..m*m). */
static void laplacian_apply(int m, const double* x, double* y) {
  for (int a = 0; a < m; ++a)
    for (int b = 0; b < m; ++b) {
      int nadj = 0;
      double s = 0.0;
      if (a > 0)     { nadj++; s += x[(a - 1) * m + b]; }
      if (a < m - 1) { nadj++; s += x[(a + 1) * m + b]; }
      if (b > 0)     { nadj++; s += x[a * m + b - 1]; }
      if (b < m - 1) { nadj++; s += x[a * m + b + 1]; }
      y[a * m + b] = nadj * x[a * m + b] - s;
    }
}
static void add_penalty(const dia_ref_config* cfg, const float* theta, double* loss, double* grad) {
  const int m = cfg->m, nk = m * m;
  const double N = (double)(cfg->n_rows - m + 1) * (double)(cfg->n_cols - m + 1);
  double* x = (double*)malloc(sizeof(double) * 3 * nk);
  double* u = x + nk; double* v = u + nk;
  for (int k = 0; k < nk; ++k) x[k] = (double)theta[k];
  laplacian_apply(m, x, u);
  laplacian_apply(m, u, v);
  double pen = 0.0;
  for (int k = 0; k < nk; ++k) pen += u[k] * u[k];
  *loss += cfg->lambda_reg * N * pen;
  for (int k = 0; k < nk; ++k) grad[k] += 2.0 * cfg->lambda_reg * N * v[k];
  free(x);
}

int dia_ref_eval_loss_grad(const dia_ref_config* cfg, const float* R, int n_epochs,
                           const float* I, const unsigned char* mask, const float* var,
                           const float* theta, double* loss, double* grad, double* grad_scale) {
  if (!check_cfg(cfg) || !R || !I || !theta || !loss || !grad || n_epochs < 1)
    return DIA_REF_ERR_INVALID_ARG;
  if (cfg->noise == DIA_REF_NOISE_FIXED && !var) return DIA_REF_ERR_INVALID_ARG;
  const size_t npix = (size_t)cfg->n_rows * cfg->n_cols;
  const int np = dia_ref_num_params(cfg);
  for (int e = 0; e < n_epochs; ++e) {
    eval_one(cfg, R, I + e * npix, mask ? mask + e * npix : NULL, var ? var + e * npix : NULL,
             theta + (size_t)e * np, loss + e, grad + (size_t)e * np,
             grad_scale ? grad_scale + (size_t)e * np : NULL);
    if (cfg->lambda_reg > 0.0) add_penalty(cfg, theta + (size_t)e * np, loss + e, grad + (size_t)e * np);
  }
  return DIA_REF_OK;
}

int dia_ref_difference_image(const dia_ref_config* cfg, const float* R, const float* I,
                             const unsigned char* mask, const float* var, const float* theta,
                             double* D, double* metrics) {
  if (!check_cfg(cfg) || !R || !I || !theta || !D || !metrics) return DIA_REF_ERR_INVALID_ARG;
  if (cfg->noise == DIA_REF_NOISE_FIXED && !var) return DIA_REF_ERR_INVALID_ARG;
  const int m = cfg->m, h = (m - 1) / 2, nr = cfg->n_rows, nc = cfg->n_cols;
  for (size_t p = 0; p < (size_t)nr * nc; ++p) D[p] = 0.0;
  /* first pass: D and eps; MFB (Eq. 29) needs the mean before MFV (Eq. 30) can be formed as printed */
  double n_used = 0.0, s1 = 0.0, chi2 = 0.0;
  double* eps = (double*)malloc(sizeof(double) * (size_t)nr * nc);
  if (!eps) return DIA_REF_ERR_ALLOC;
  for (int i = h; i < nr - h; ++i)
    for (int j = h; j < nc - h; ++j) {
      const size_t p = (size_t)i * nc + j;
      const double M = model_pixel(cfg, R, nc, m, theta, i, j);
      D[p] = (double)I[p] - M;
      eps[p] = 0.0;
      if (mask && mask[p] == 0) continue;
      double v;
      if (cfg->noise == DIA_REF_NOISE_MODEL) {
        const double F = cfg->flat ? (double)cfg->flat[p] : 1.0;
        v = cfg->sigma0 * cfg->sigma0 / (F * F) + (M > 0.0 ? M : 0.0) / (cfg->gain * F);      /* Eq. 6, R1 */
      } else {
        v = (double)var[p];
      }
      eps[p] = D[p] / sqrt(v);
      n_used += 1.0;  s1 += eps[p];  chi2 += eps[p] * eps[p];
    }
  const double mfb = n_used > 0.0 ? s1 / n_used : 0.0;                                       /* Eq. 29 */
  double s2 = 0.0;
  for (int i = h; i < nr - h; ++i)
    for (int j = h; j < nc - h; ++j) {
      const size_t p = (size_t)i * nc + j;
      if (mask && mask[p] == 0) continue;
      s2 += (eps[p] - mfb) * (eps[p] - mfb);
    }
  metrics[0] = n_used;  metrics[1] = mfb;
  metrics[2] = n_used > 1.0 ? s2 / (n_used - 1.0) : 0.0;                                     /* Eq. 30 */
  metrics[3] = chi2;
  free(eps);
  return DIA_REF_OK;
}

/* D3: second derivative of the pixel term l = rho(z) + (1/2) ln v with respect to M, with r = I - M,
 * v = a + b' M, z = r / sqrt(v).  Gaussian: w = -r/v - b' r^2/(2 v^2) + b'/(2v), so
 *   dw/dM = 1/v + 2 b' r / v^2 + b'^2 r^2 / v^3 - b'^2 / (2 v^2).
 * Huber, linear branch (|z| > c, psi = +-c): w = -psi/s - psi z b'/(2v) + b'/(2v), s = sqrt v, z = r/s; with
 * ds/dM = b'/(2s), dz/dM = -1/s - z b'/(2v):
 *   dw/dM = psi b'/(2 s v) - psi b'/(2v) dz/dM + psi z b'^2/(2 v^2) - b'^2/(2 v^2). */
static double pixel_d2(const dia_ref_config* cfg, double r, double v, double bp) {
  const double sd = sqrt(v), z = r / sd;
  if (cfg->loss == DIA_REF_LOSS_HUBER && fabs(z) > cfg->huber_c) {
    const double psi = (z > 0.0) ? cfg->huber_c : -cfg->huber_c;
    const double dz = -1.0 / sd - z * bp / (2.0 * v);
    return psi * bp / (2.0 * sd * v) - psi * bp / (2.0 * v) * dz + psi * z * bp * bp / (2.0 * v * v) -
           bp * bp / (2.0 * v * v);
  }
  return 1.0 / v + 2.0 * bp * r / (v * v) + bp * bp * r * r / (v * v * v) - bp * bp / (2.0 * v * v);
}

int dia_ref_hessian(const dia_ref_config* cfg, const float* R, const float* I, const unsigned char* mask,
                    const float* var, const float* theta, double* H) {
  if (!check_cfg(cfg) || !R || !I || !theta || !H) return DIA_REF_ERR_INVALID_ARG;
  if (cfg->noise == DIA_REF_NOISE_FIXED && !var) return DIA_REF_ERR_INVALID_ARG;
  const int m = cfg->m, h = (m - 1) / 2, nk = m * m, np = dia_ref_num_params(cfg), nbg = np - nk;
  const int nr = cfg->n_rows, nc = cfg->n_cols;
  double* X = (double*)malloc(sizeof(double) * np);
  if (!X) return DIA_REF_ERR_ALLOC;
  for (size_t q = 0; q < (size_t)np * np; ++q) H[q] = 0.0;
  for (int i = h; i < nr - h; ++i)
    for (int j = h; j < nc - h; ++j) {
      const size_t p = (size_t)i * nc + j;
      if (mask && mask[p] == 0) continue;
      const double M = model_pixel(cfg, R, nc, m, theta, i, j);
      double v, bp;
      if (cfg->noise == DIA_REF_NOISE_MODEL) {
        const double F = cfg->flat ? (double)cfg->flat[p] : 1.0;
        const double b_ij = 1.0 / (cfg->gain * F);
        v = cfg->sigma0 * cfg->sigma0 / (F * F) + b_ij * (M > 0.0 ? M : 0.0);
        bp = (M > 0.0) ? b_ij : 0.0;
      } else {
        v = (double)var[p];
        bp = 0.0;
      }
      const double d2 = pixel_d2(cfg, (double)I[p] - M, v, bp);
      for (int a = 0; a < m; ++a)
        for (int b = 0; b < m; ++b) X[a * m + b] = (double)R[(size_t)(i - h + a) * nc + (j - h + b)];
      background(cfg, theta + nk, i, j, X + nk);
      for (int q = 0; q < np; ++q) {
        const double xq = d2 * X[q];
        for (int s = q; s < np; ++s) H[(size_t)q * np + s] += xq * X[s];
      }
    }
  for (int q = 0; q < np; ++q)
    for (int s = 0; s < q; ++s) H[(size_t)q * np + s] = H[(size_t)s * np + q];
  (void)nbg;
  if (cfg->lambda_reg > 0.0) {           /* Eq. 20: + 2 lambda N L'L on the kernel block */
    const double N = (double)(nr - m + 1) * (double)(nc - m + 1);
    double* e = (double*)calloc((size_t)3 * nk, sizeof(double));
    if (!e) { free(X); return DIA_REF_ERR_ALLOC; }
    double* u = e + nk; double* w2 = u + nk;
    for (int k = 0; k < nk; ++k) {
      e[k] = 1.0;
      laplacian_apply(m, e, u);
      laplacian_apply(m, u, w2);
      for (int q = 0; q < nk; ++q) H[(size_t)q * np + k] += 2.0 * cfg->lambda_reg * N * w2[q];
      e[k] = 0.0;
    }
    free(e);
  }
  free(X);
  return DIA_REF_OK;
}

/* Eq. 14: Q = N ln( sqrt(2 pi) erf(c/sqrt 2) + 2 exp(-c^2/2)/c ). */
double dia_ref_huber_Q(double c, double N) {
  const double pi = 3.14159265358979323846;
  return N * log(sqrt(2.0 * pi) * erf(c / sqrt(2.0)) + 2.0 * exp(-0.5 * c * c) / c);
}
