/* dia_ref_fit.c -- CPU ORACLE, optimiser part (test infrastructure only; see dia_ref.h).
 *
 * Adam (Eq. 9; Kingma & Ba Algorithm 1) followed by L-BFGS (PAPER.md:132-135
 * Eq. 10; Nocedal & Wright Alg. 7.4 two-loop recursion, Alg. 7.5), with the switch and stop
 * rules of PAPER.md:244, 248-255 under readings R5-R9 of DESIGN.md.  All optimiser state is
 * FP64; theta is rounded to float32 only where it enters the objective (R9).
 */
#include "dia_ref.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

void dia_ref_default_fit_opts(dia_ref_fit_opts* o) {
  o->lr_kernel = 1e-3;  o->lr_b0 = 10.0;
  o->adam_beta1 = 0.9;  o->adam_beta2 = 0.999;  o->adam_eps = 1e-8;   /* R5 */
  o->tol_switch = 1e-6;
  o->lbfgs_lr = 1.0;
  o->lbfgs_history = 100;  o->lbfgs_backtrack = 0;             /* R7 */
  o->tol_change_rel = 1e-8;  o->tol_grad_abs = 1e-7;  o->tol_grad_rel = 0.0;   /* PAPER.md:244, R8 */
  o->max_adam_iters = 20000;  o->max_lbfgs_iters = 500;
  o->force_adam_iters = -1;  o->force_lbfgs_iters = -1;
}

typedef struct {
  const dia_ref_config* cfg;
  const float* R; const float* I; const unsigned char* mask; const float* var;
  int np;
  float* th32;
  int n_evals;
  /* optional FP64 record of the iterates (dia_ref_fit_trace): row r = theta after update r, its loss column the
     loss that update was computed from (Adam: at the pre-update iterate) or reached (L-BFGS: at the new iterate) */
  double* tr_theta; double* tr_loss; int tr_cap, tr_n;
} objective;

static void record(objective* ob, const double* th, double L) {
  if (!ob->tr_theta || ob->tr_n >= ob->tr_cap) return;
  memcpy(ob->tr_theta + (size_t)ob->tr_n * ob->np, th, sizeof(double) * ob->np);
  if (ob->tr_loss) ob->tr_loss[ob->tr_n] = L;
  ob->tr_n++;
}

/* Evaluate the objective at the float32 rounding of theta (R9). */
static void eval_at(objective* ob, const double* theta, double* L, double* g) {
  for (int k = 0; k < ob->np; ++k) ob->th32[k] = (float)theta[k];
  dia_ref_eval_loss_grad(ob->cfg, ob->R, 1, ob->I, ob->mask, ob->var, ob->th32, L, g, NULL);
  ob->n_evals++;
}

static double inf_norm(const double* g, int n) {
  double m = 0.0;
  for (int k = 0; k < n; ++k) { double a = fabs(g[k]); if (a > m || a != a) m = a; }
  return m;
}
static double dot(const double* a, const double* b, int n) {
  double s = 0.0;
  for (int k = 0; k < n; ++k) s += a[k] * b[k];
  return s;
}

static int fit_one(objective* ob, const dia_ref_fit_opts* o, float* theta_io, dia_ref_fit_result* res) {
  const int np = ob->np, nk = ob->cfg->m * ob->cfg->m;
  const int hist = o->lbfgs_history > 0 ? o->lbfgs_history : 1;
  double* th = (double*)malloc(sizeof(double) * np);
  double* g = (double*)malloc(sizeof(double) * np);
  double* m1 = (double*)calloc(np, sizeof(double));
  double* m2 = (double*)calloc(np, sizeof(double));
  double* d = (double*)malloc(sizeof(double) * np);
  double* thn = (double*)malloc(sizeof(double) * np);
  double* gn = (double*)malloc(sizeof(double) * np);
  double* S = (double*)malloc(sizeof(double) * (size_t)hist * np);
  double* Y = (double*)malloc(sizeof(double) * (size_t)hist * np);
  double* rho = (double*)malloc(sizeof(double) * hist);
  double* alpha = (double*)malloc(sizeof(double) * hist);
  if (!th || !g || !m1 || !m2 || !d || !thn || !gn || !S || !Y || !rho || !alpha) return DIA_REF_ERR_ALLOC;
  for (int k = 0; k < np; ++k) th[k] = (double)theta_io[k];
  ob->n_evals = 0;
  int n_adam = 0, n_lbfgs = 0, status = DIA_REF_FIT_MAX_ITERS;
  double L = 0.0, Lprev = 0.0;

  /* ---------------- ADAM PHASE ---------------- */
  double b1t = 1.0, b2t = 1.0;
  for (int t = 1;; ++t) {
    eval_at(ob, th, &L, g);
    if (!isfinite(L)) { status = DIA_REF_FIT_NONFINITE; goto done; }
    if (o->force_adam_iters >= 0) {
      if (t > o->force_adam_iters) break;
    } else {
      /* R6: losses at consecutive pre-update iterates, strict <, denominator |L_{t-1}| */
      if (t >= 2 && fabs(L - Lprev) < o->tol_switch * fabs(Lprev)) break;
      if (t > o->max_adam_iters) break;
    }
    b1t *= o->adam_beta1;  b2t *= o->adam_beta2;
    for (int k = 0; k < np; ++k) {
      m1[k] = o->adam_beta1 * m1[k] + (1.0 - o->adam_beta1) * g[k];
      m2[k] = o->adam_beta2 * m2[k] + (1.0 - o->adam_beta2) * g[k] * g[k];
      const double mh = m1[k] / (1.0 - b1t), vh = m2[k] / (1.0 - b2t);
      const double lr = (k < nk) ? o->lr_kernel : o->lr_b0;
      th[k] -= lr * mh / (sqrt(vh) + o->adam_eps);
    }
    n_adam++;
    Lprev = L;
    record(ob, th, L);
  }

  /* ---------------- L-BFGS PHASE ---------------- */
  {
    int n_pairs = 0, head = 0;     /* ring buffer: oldest at head, newest at head+n_pairs-1 */
    const double g_switch = inf_norm(g, np);
    for (int k = 1;; ++k) {
      if (o->force_lbfgs_iters >= 0) {
        if (k > o->force_lbfgs_iters) { status = DIA_REF_FIT_MAX_ITERS; break; }
      } else {
        const double gi = inf_norm(g, np);
        if (gi < o->tol_grad_abs || gi < o->tol_grad_rel * g_switch) { status = DIA_REF_FIT_CONVERGED_GRAD; break; }
      }
      /* two-loop recursion: d = -H g, H0 = gamma I, gamma = s'y / y'y of the newest pair */
      for (int q = 0; q < np; ++q) d[q] = g[q];
      for (int i = n_pairs - 1; i >= 0; --i) {
        const int id = (head + i) % hist;
        alpha[i] = rho[id] * dot(S + (size_t)id * np, d, np);
        for (int q = 0; q < np; ++q) d[q] -= alpha[i] * Y[(size_t)id * np + q];
      }
      double gamma = 1.0;
      if (n_pairs > 0) {
        const int id = (head + n_pairs - 1) % hist;
        gamma = dot(S + (size_t)id * np, Y + (size_t)id * np, np) / dot(Y + (size_t)id * np, Y + (size_t)id * np, np);
      }
      for (int q = 0; q < np; ++q) d[q] *= gamma;
      for (int i = 0; i < n_pairs; ++i) {
        const int id = (head + i) % hist;
        const double beta = rho[id] * dot(Y + (size_t)id * np, d, np);
        for (int q = 0; q < np; ++q) d[q] += (alpha[i] - beta) * S[(size_t)id * np + q];
      }
      for (int q = 0; q < np; ++q) d[q] = -d[q];
      double gtd = dot(g, d, np);
      if (!(gtd < 0.0)) {                 /* not a descent direction: drop history */
        n_pairs = 0; head = 0;
        for (int q = 0; q < np; ++q) d[q] = -g[q];
        gtd = dot(g, d, np);
      }
      /* R7: unit step, except with empty history the first step is scaled by min(1, 1/|g|_1) */
      double a = o->lbfgs_lr;
      if (n_pairs == 0) {
        double g1 = 0.0;
        for (int q = 0; q < np; ++q) g1 += fabs(g[q]);
        a *= (g1 > 1.0) ? 1.0 / g1 : 1.0;
      }
      double Ln;
      for (int q = 0; q < np; ++q) thn[q] = th[q] + a * d[q];
      eval_at(ob, thn, &Ln, gn);
      if (o->lbfgs_backtrack) {
        int nbt = 0;
        while ((!isfinite(Ln) || Ln > L + 1e-4 * a * gtd) && nbt < 20) {
          a *= 0.5;
          for (int q = 0; q < np; ++q) thn[q] = th[q] + a * d[q];
          eval_at(ob, thn, &Ln, gn);
          nbt++;
        }
      }
      if (!isfinite(Ln)) { status = DIA_REF_FIT_NONFINITE; break; }
      /* s = a d, y = g+ - g; keep the pair iff s'y > 1e-10 (R7), FIFO eviction */
      double sty = 0.0;
      for (int q = 0; q < np; ++q) sty += (a * d[q]) * (gn[q] - g[q]);
      if (sty > 1e-10) {
        int id;
        if (n_pairs < hist) { id = (head + n_pairs) % hist; n_pairs++; }
        else { id = head; head = (head + 1) % hist; }
        for (int q = 0; q < np; ++q) { S[(size_t)id * np + q] = a * d[q]; Y[(size_t)id * np + q] = gn[q] - g[q]; }
        rho[id] = 1.0 / sty;
      }
      const double dL = fabs(Ln - L);
      for (int q = 0; q < np; ++q) { th[q] = thn[q]; g[q] = gn[q]; }
      L = Ln;
      n_lbfgs++;
      record(ob, th, L);
      if (o->force_lbfgs_iters < 0) {
        if (dL <= o->tol_change_rel * fabs(L)) { status = DIA_REF_FIT_CONVERGED_CHANGE; break; }   /* R8 */
        if (k >= o->max_lbfgs_iters) { status = DIA_REF_FIT_MAX_ITERS; break; }
      }
    }
  }
done:
  for (int k = 0; k < np; ++k) theta_io[k] = (float)th[k];
  res->loss = L;
  res->grad_inf_norm = inf_norm(g, np);
  double P = 0.0;
  for (int k = 0; k < nk; ++k) P += th[k];            /* Eq. 3 */
  res->photometric_scale = P;
  res->n_adam = n_adam;  res->n_lbfgs = n_lbfgs;  res->n_evals = ob->n_evals;  res->status = status;
  free(th); free(g); free(m1); free(m2); free(d); free(thn); free(gn); free(S); free(Y); free(rho); free(alpha);
  return DIA_REF_OK;
}

int dia_ref_fit(const dia_ref_config* cfg, const float* R, const dia_ref_fit_opts* opts,
                int n_epochs, const float* I, const unsigned char* mask, const float* var,
                float* theta, dia_ref_fit_result* result) {
  if (!cfg || !R || !opts || !I || !theta || !result || n_epochs < 1) return DIA_REF_ERR_INVALID_ARG;
  if (cfg->m < 1 || cfg->m % 2 == 0) return DIA_REF_ERR_INVALID_ARG;
  if (cfg->noise == DIA_REF_NOISE_FIXED && !var) return DIA_REF_ERR_INVALID_ARG;
  const size_t npix = (size_t)cfg->n_rows * cfg->n_cols;
  const int np = dia_ref_num_params(cfg);
  float* th32 = (float*)malloc(sizeof(float) * np);
  if (!th32) return DIA_REF_ERR_ALLOC;
  int rc = DIA_REF_OK;
  for (int e = 0; e < n_epochs && rc == DIA_REF_OK; ++e) {
    objective ob = { cfg, R, I + e * npix, mask ? mask + e * npix : NULL, var ? var + e * npix : NULL, np, th32, 0,
                     NULL, NULL, 0, 0 };
    rc = fit_one(&ob, opts, theta + (size_t)e * np, result + e);
  }
  free(th32);
  return rc;
}


/* dia_ref_fit for one epoch that also records the FP64 iterates (the float32 theta of dia_ref_fit hides 1e-8 of
 * them): trace_theta [trace_cap][np] receives theta after every Adam / L-BFGS update in order, trace_loss
 * [trace_cap] the loss belonging to it, *trace_n the number of rows written.  Same arithmetic as dia_ref_fit --
 * it is the same fit_one -- so that the optimiser can be pinned against library / textbook recursions
 * (tests/test_oracle_optimiser_pins.py). */
int dia_ref_fit_trace(const dia_ref_config* cfg, const float* R, const dia_ref_fit_opts* opts,
                      const float* I, const unsigned char* mask, const float* var,
                      float* theta, dia_ref_fit_result* result,
                      double* trace_theta, double* trace_loss, int trace_cap, int* trace_n) {
  if (!cfg || !R || !opts || !I || !theta || !result || !trace_theta || !trace_n || trace_cap < 0)
    return DIA_REF_ERR_INVALID_ARG;
  if (cfg->m < 1 || cfg->m % 2 == 0) return DIA_REF_ERR_INVALID_ARG;
  if (cfg->noise == DIA_REF_NOISE_FIXED && !var) return DIA_REF_ERR_INVALID_ARG;
  const int np = dia_ref_num_params(cfg);
  float* th32 = (float*)malloc(sizeof(float) * np);
  if (!th32) return DIA_REF_ERR_ALLOC;
  objective ob = { cfg, R, I, mask, var, np, th32, 0, trace_theta, trace_loss, trace_cap, 0 };
  const int rc = fit_one(&ob, opts, theta, result);
  *trace_n = ob.tr_n;
  free(th32);
  return rc;
}
