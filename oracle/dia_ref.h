/* dia_ref.h -- CPU ORACLE for the DIA objective/gradient/fit.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, FP64 restatement of what the hot path computes, written from the paper
 * (PAPER.md = arxiv 2104.13715, "PyTorchDIA") and the readings listed in DESIGN.md.
 * It shares no code, header, table or helper with the CUDA library in
 * paper_2104_13715_b200/csrc and is used only by tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs.  All pointers are HOST pointers.
 *
 * Layout conventions (identical in meaning to include/dia.h, restated here on purpose):
 *   images row-major [n_rows][n_cols]; kernel K row-major [m][m], K[a][b] with
 *   a = l + h, b = mm + h, h = (m-1)/2, (l, mm) the kernel coordinates of Eq. 2
 *   (PAPER.md:60); theta = [K (m*m values), B0]; the valid set is
 *   h <= i < n_rows-h, h <= j < n_cols-h intersected with mask != 0.
 *
 * Pin status (tests/test_oracle_*.py): model, noise, both losses, gradient, Hessian, covariance, B08 solve,
 * fixed-weight fit and planted recovery are pinned; the optimiser's arithmetic is pinned step by step
 * (tests/test_oracle_optimiser_pins.py: the Adam trajectory against torch.optim.Adam in float64, every L-BFGS
 * direction against the dense BFGS recursion with and without eviction, the switch rule on crafted tolerances).
 * What stays "parity unpinned" is the ITERATE AT WHICH a free-running fit on noisy data stops under the paper's
 * loss-change rule: no external value exists for it.
 */
#ifndef DIA_REF_H
#define DIA_REF_H

#ifdef __cplusplus
extern "C" {
#endif

enum { DIA_REF_OK = 0, DIA_REF_ERR_INVALID_ARG = -1, DIA_REF_ERR_ALLOC = -3, DIA_REF_ERR_NOT_PD = -5 };
enum { DIA_REF_LOSS_GAUSSIAN = 0 /* Eq. 8 */, DIA_REF_LOSS_HUBER = 1 /* Eq. 13 */ };
enum { DIA_REF_NOISE_MODEL = 0 /* Eq. 6 */, DIA_REF_NOISE_FIXED = 1 /* caller variance */ };
enum { DIA_REF_FIT_CONVERGED_GRAD = 0, DIA_REF_FIT_CONVERGED_CHANGE = 1, DIA_REF_FIT_MAX_ITERS = 2,
       DIA_REF_FIT_NONFINITE = 3 };

typedef struct {
  int n_rows, n_cols, m;      /* m odd */
  int loss;    double huber_c;          /* c = 1.345 default */
  int noise;   double sigma0, gain;     /* Eq. 6 parameters */
  const float* flat;                    /* [n_rows][n_cols] or NULL => F == 1 */
  double lambda_reg;                    /* Eq. 20: lambda of the Laplacian penalty, 0 = off */
  int bg_degree;                        /* Eq. 18: degree d of the polynomial background, 0 = scalar B0.
                                           theta = [K (m*m), b_mn for m = 0..d, n = 0..d-m]; (d+1)(d+2)/2 coefficients */
} dia_ref_config;

typedef struct {                        /* PAPER.md:242-244; [reading] marks DESIGN.md readings */
  double lr_kernel, lr_b0;              /* 1e-3; 1, 10 or 100 */
  double adam_beta1, adam_beta2, adam_eps;          /* [reading R5] 0.9, 0.999, 1e-8 */
  double tol_switch;                    /* 1e-6 */
  double lbfgs_lr;                      /* 1.0 */
  int    lbfgs_history;                 /* [reading R7] 100 */
  int    lbfgs_backtrack;               /* [reading R7] 0 = fixed step (default), 1 = Armijo back-off */
  double tol_change_rel, tol_grad_abs, tol_grad_rel;   /* 1e-8, 1e-7, [reading] 0 = off */
  int    max_adam_iters, max_lbfgs_iters;              /* [reading] 20000, 500 */
  int    force_adam_iters, force_lbfgs_iters;          /* [reading] -1 = off (lock-step mode) */
} dia_ref_fit_opts;

typedef struct {
  double loss, grad_inf_norm, photometric_scale;
  int n_adam, n_lbfgs, n_evals, status;
} dia_ref_fit_result;

void dia_ref_default_fit_opts(dia_ref_fit_opts* o);

/* Number of parameters per epoch: m*m + (d+1)(d+2)/2. */
int dia_ref_num_params(const dia_ref_config* cfg);

/* Model image of Eq. 2 on the valid region: M [n_rows-m+1][n_cols-m+1] (FP64). */
int dia_ref_model(const dia_ref_config* cfg, const float* R, const float* theta, double* M);

/* Loss and gradient (SURVEY/DESIGN c.1).  theta float32 [n_epochs][m*m+1];
 * loss [n_epochs]; grad [n_epochs][m*m+1].  grad_scale (nullable) receives
 * S_p = sum_V |w_ij| |X_p(i,j)|, the cancellation-free magnitude used by the parity protocol. */
int dia_ref_eval_loss_grad(const dia_ref_config* cfg, const float* R, int n_epochs,
                           const float* I, const unsigned char* mask, const float* var,
                           const float* theta, double* loss, double* grad, double* grad_scale);

/* Difference image D = I - M on the valid region (0 elsewhere), [n_rows][n_cols] FP64, and the fit-quality
 * metrics of Eq. 29-30 over the unmasked valid pixels, with sigma from Eq. 6 at the model
 * (or the caller's variance map): metrics = { N_used, MFB, MFV, chi^2 }.  One epoch. */
int dia_ref_difference_image(const dia_ref_config* cfg, const float* R, const float* I,
                             const unsigned char* mask, const float* var, const float* theta,
                             double* D, double* metrics);

/* Hessian of the objective at theta, H [np][np] row-major FP64 (np = dia_ref_num_params): the observed Fisher
 * information of Eq. 15 when theta is the MLE; its inverse is the covariance of Eq. 16-17.
 * Analytic: H = sum_V h_ij X X' (+ 2 lambda N L'L), X the design vector (shifted reference pixels, background
 * basis) and h_ij = d^2 l_ij / dM^2 (D3).  One epoch. */
int dia_ref_hessian(const dia_ref_config* cfg, const float* R, const float* I, const unsigned char* mask,
                    const float* var, const float* theta, double* H);

/* Covariance estimate Sigma = H^-1 (Eq. 16), parameter uncertainties sqrt(Sigma_pp) (Eq. 17,
 * PAPER.md:189-191) and the validity tests of PAPER.md:193 (determinant of Sigma not negative, every eigenvalue of
 * Sigma positive).  H [n][n] row-major FP64 symmetric; the first n_kernel parameters are the kernel pixels, whose sum
 * is the photometric scale factor P (Eq. 3).  Out: cov [n][n], sigma [n],
 * info[5] = { valid (1/0), ln|det H|, sigma_P = sqrt(u' Sigma u), smallest eigenvalue of Sigma, sign of det H }. */
int dia_ref_covariance(int n, int n_kernel, const double* H, double* cov, double* sigma, double* info);

/* Adam -> L-BFGS fit (DESIGN c.2), one epoch after another.  theta in/out float32. */
int dia_ref_fit(const dia_ref_config* cfg, const float* R, const dia_ref_fit_opts* opts,
                int n_epochs, const float* I, const unsigned char* mask, const float* var,
                float* theta, dia_ref_fit_result* result);

/* dia_ref_fit for ONE epoch, recording the FP64 iterates: trace_theta [trace_cap][np] = theta after every Adam /
 * L-BFGS update in order, trace_loss [trace_cap] (nullable) = the loss the Adam update was computed from / the
 * L-BFGS update reached, *trace_n = rows written.  Same arithmetic (same routine) as dia_ref_fit. */
int dia_ref_fit_trace(const dia_ref_config* cfg, const float* R, const dia_ref_fit_opts* opts,
                      const float* I, const unsigned char* mask, const float* var,
                      float* theta, dia_ref_fit_result* result,
                      double* trace_theta, double* trace_loss, int trace_cap, int* trace_n);

/* B08 iterated normal-equation solve (DESIGN c.3).  One epoch.
 * var_fixed (nullable): if given, every iteration uses this variance map instead of Eq. 6.
 * theta out FP64 [m*m+1]; H (nullable) out [(m*m+1)^2] row-major, the last normal matrix. */
int dia_ref_b08_solve(const dia_ref_config* cfg, const float* R, const float* I,
                      const unsigned char* mask, const float* var_fixed, int n_iters,
                      int clip_last, double* theta, double* H);

/* Normalising constant Q of Eq. 14 for N pixels. */
double dia_ref_huber_Q(double c, double N);

int dia_ref_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
