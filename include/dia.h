/* dia.h -- C ABI of the B200-native DIA objective/gradient/fit engine.
 *
 * Hot path of PyTorchDIA (arxiv 2104.13715; citations are PAPER.md:<line>): the repeated
 * evaluation of the objective and its analytic gradient for the B08 discrete-pixel kernel
 * model, the on-device Adam -> L-BFGS optimiser with its convergence test, and a batched mode
 * that fits many target epochs against one resident reference.
 *
 * CONVENTIONS
 *  - Every `d_*` pointer is a DEVICE pointer owned by the caller (e.g. a torch tensor's
 *    data_ptr()); the library never frees or reallocates caller memory.  Struct pointers
 *    (dia_config, dia_fit_opts) are HOST pointers read during the call.
 *  - Images are row-major [n_rows][n_cols] float32.  The kernel K is row-major [m][m] with
 *    K[a][b], a = l + h, b = mm + h, h = (m-1)/2, (l, mm) the kernel coordinates of Eq. 2
 *    (PAPER.md:60): M_ij = sum_ab K[a][b] R[i-h+a][j-h+b] + B0 -- a cross-correlation, no flip.
 *    theta = [K (m*m values, row-major), B0], m*m+1 parameters per epoch.
 *  - The valid set V is h <= i < n_rows-h, h <= j < n_cols-h, intersected with
 *    mask != 0 when a mask is given.  Pixels of mask, var, flat outside V are never read; pixels of I
 *    outside V (and under mask == 0) may be fetched with their tile but never influence a result
 *    (they may hold NaN).
 *  - Every call is ASYNCHRONOUS on cfg.stream and performs no host synchronisation
 *    (dia_create / dia_destroy may).  Outputs are valid once the caller synchronises the stream.
 *  - Argument errors are detected on the host before any launch and return a negative code
 *    with outputs untouched.  Numerical failure (non-finite loss) is data dependent and is
 *    reported per epoch in dia_fit_result.status, not by return code.
 *  - Same inputs => bit-identical outputs on repeated calls (fixed tile->block map, fixed-order
 *    FP64 reductions, no floating-point atomics).
 *  - Threads: different handles may be driven from different host threads at the same time, on the same or on
 *    different streams (handles of one kernel size that share a stream also share a constant-memory block; the
 *    library serialises the enqueues that refresh and use it).  ONE handle must not be used by two threads at once:
 *    it owns a single workspace, and its calls are ordered by its stream only.
 *  - There is no CPU fallback: without a CUDA device every entry point fails with DIA_ERR_CUDA.
 */
#ifndef DIA_H
#define DIA_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dia_handle dia_handle;     /* opaque; owns only its own workspace */

enum { DIA_OK = 0, DIA_ERR_INVALID_ARG = -1, DIA_ERR_CUDA = -2, DIA_ERR_ALLOC = -3,
       DIA_ERR_UNSUPPORTED = -4 };
enum { DIA_LOSS_GAUSSIAN = 0 /* Eq. 8 */, DIA_LOSS_HUBER = 1 /* Eq. 12-13 */ };
enum { DIA_NOISE_MODEL = 0 /* Eq. 6: sigma depends on theta */,
       DIA_NOISE_FIXED = 1 /* caller variance map */ };
enum { DIA_FIT_CONVERGED_GRAD = 0, DIA_FIT_CONVERGED_CHANGE = 1, DIA_FIT_MAX_ITERS = 2,
       DIA_FIT_NONFINITE = 3 };

#define DIA_MAX_KERNEL_SIZE 47            /* m odd, 1 <= m <= 47: the largest kernel of the paper's real-data fits
                                             (PAPER.md:475); m >= 33 runs one CTA per SM instead of two */
#define DIA_MAX_BG_DEGREE 3               /* polynomial background degree d <= 3 in this build */

typedef struct {
  int n_rows, n_cols, m;          /* m odd, 1 <= m <= min(n_rows, n_cols, DIA_MAX_KERNEL_SIZE) */
  int max_epochs;                 /* batch capacity of the handle, >= 1 */
  int loss;    float huber_c;     /* c > 0; 1.345 is the paper's default */
  int noise;   float sigma0, gain;/* Eq. 6: read noise [ADU] >= 0, gain [e-/ADU] > 0 */
  const float* d_flat;            /* master flat F [n_rows][n_cols] or NULL => F == 1; borrowed for handle life */
  void* stream;                   /* cudaStream_t; NULL = legacy default stream */
  int n_refs;                     /* 0 or 1: one reference shared by all epochs (d_R is [n_rows][n_cols]);
                                     == max_epochs: one reference per epoch (d_R is [max_epochs][n_rows][n_cols]) --
                                     many independent small image pairs fitted in one launch sequence, the
                                     shape of the paper's stamp workloads */
  float lambda_reg;               /* Eq. 20: adds lambda N_data theta' L' L theta to the objective, L the
                                     graph Laplacian of the kernel pixels (Eq. 21; 4 edge neighbours, B0 not penalised,
                                     N_data = valid-region pixels); 0 = off (the paper's own experiments) */
  int bg_degree;                  /* Eq. 18-19: degree d of the polynomial background
                                     B(x,y) = sum_{m=0..d} sum_{n=0..d-m} b_mn eta^m xi^n, eta = (x - x_c)/N_x,
                                     xi = (y - y_c)/N_y, x = column, y = row, centre ((N-1)/2); 0 = scalar B0.
                                     theta then holds (d+1)(d+2)/2 coefficients after K, b_00 first (m outer, n inner),
                                     all stepped with lr_b0; every [m*m+1] below reads [m*m + (d+1)(d+2)/2] */
} dia_config;

typedef struct {                  /* PAPER.md:242-244 unless marked [reading] */
  float  lr_kernel;               /* Adam learning rate of the kernel pixels, 1e-3 */
  float  lr_b0;                   /* Adam learning rate of B0: 1, 10 or 100 */
  double adam_beta1, adam_beta2, adam_eps;   /* [reading R5] 0.9, 0.999, 1e-8 */
  double tol_switch;              /* Adam -> L-BFGS when |dL| < tol_switch |L|, 1e-6 */
  double lbfgs_lr;                /* 1.0 */
  int    lbfgs_history;           /* [reading R7] 100; 1 <= history <= 128 */
  int    lbfgs_backtrack;         /* [reading R7] 0 = fixed step as in the paper's library route (default);
                                     1 = Armijo back-off (<= 20 halvings) */
  double tol_change_rel;          /* stop when |dL| <= tol_change_rel |L|, 1e-8 [R8] */
  double tol_grad_abs;            /* stop when max|g| < tol_grad_abs, 1e-7 */
  double tol_grad_rel;            /* [reading] stop when max|g| < tol_grad_rel * max|g at switch|; 0 = off */
  int    max_adam_iters, max_lbfgs_iters;    /* [reading] 20000, 500 */
  int    force_adam_iters, force_lbfgs_iters;/* [reading] -1 = off; >= 0 replaces the data-dependent
                                                exits by fixed counts (lock-step parity mode) */
} dia_fit_opts;

typedef struct {
  double loss, grad_inf_norm, photometric_scale;   /* final L, max|g|, P = sum K (Eq. 3) */
  int n_adam, n_lbfgs, n_evals, status;            /* status: DIA_FIT_* */
} dia_fit_result;

/* Fills `opts` (HOST) with the defaults listed above. */
void dia_default_fit_opts(dia_fit_opts* opts);

/* Creates a handle for one reference image d_R [n_rows][n_cols] (DEVICE, borrowed for the
 * handle's life, must stay unchanged; [max_epochs][n_rows][n_cols] when cfg->n_refs == max_epochs).
 * Allocates the workspace for cfg->max_epochs epochs.
 * May synchronise.  Errors: INVALID_ARG (bad sizes/enums/NULLs), UNSUPPORTED (m too large),
 * CUDA, ALLOC. */
int dia_create(const dia_config* cfg, const float* d_R, dia_handle** out);

/* Loss and gradient of the objective (Eq. 8 or Eq. 13 without theta-independent constants,
 * with the noise model of Eq. 6 or a fixed variance map) for n_epochs targets, each at its own
 * theta:   M = R (x) K + B0 (Eq. 2);  r = I - M;  v = sigma0^2/F^2 + max(M,0)/(G F);
 *          L = sum_V rho(r/sqrt v) + 1/2 ln v;   dL/dK[a][b] = sum_V w_ij R[i-h+a][j-h+b],
 *          dL/dB0 = sum_V w_ij,  w = dL/dM.
 * 1 <= n_epochs <= max_epochs.  Asynchronous on the handle's stream. */
int dia_eval_loss_grad(dia_handle* h, int n_epochs,
                       const float* d_I,            /* [n_epochs][n_rows][n_cols] */
                       const unsigned char* d_mask, /* same shape, 1 = use; or NULL */
                       const float* d_var,          /* variance map, same shape; required iff DIA_NOISE_FIXED, else NULL */
                       const float* d_theta,        /* [n_epochs][m*m+1] */
                       double* d_loss,              /* out [n_epochs] */
                       double* d_grad);             /* out [n_epochs][m*m+1] */

/* Full fit: Adam (Eq. 9) until the relative loss change drops below
 * tol_switch, then L-BFGS (Eq. 10) until convergence, all on the device; the host enqueues one
 * graph launch and never reads a per-iteration value.  d_theta holds the initial theta on entry
 * and the fitted theta on exit.  d_result [n_epochs] is DEVICE memory. */
int dia_fit(dia_handle* h, const dia_fit_opts* opts, int n_epochs,
            const float* d_I, const unsigned char* d_mask, const float* d_var,
            float* d_theta, dia_fit_result* d_result);

/* Hessian of the objective at theta for ONE target image: the observed Fisher information of Eq. 15
 * when theta is the MLE; its inverse is the covariance matrix of Eq. 16-17, whose diagonal
 * gives the parameter uncertainties (the caller inverts it and checks positive-definiteness).
 * The paper takes second derivatives by automatic differentiation; here they are analytic like the gradient:
 * with X the design vector of a pixel (the m*m shifted reference pixels, then the background basis) and
 * h_ij = d^2 l_ij / dM^2 (D3), row q of H is sum_V (h_ij X_q) X -- the gradient sum of
 * dia_eval_loss_grad with the per-pixel weight h_ij X_q in place of w_ij -- so the stencil code of the fused kernel
 * computes the rows, 32 kernel-pixel rows per launch with h_ij evaluated once per launch (whatever the handle's
 * max_epochs); the penalty of Eq. 20 adds 2 lambda N L'L, and H is symmetrised.
 *   d_I [n_rows][n_cols], d_mask / d_var as in dia_eval_loss_grad for one epoch; d_theta [np] float32;
 *   d_H [np][np] float64 DEVICE, row-major, out.
 * The first call allocates a small workspace (synchronises once); later calls are asynchronous.  Handles created
 * with one reference per epoch (n_refs > 1) are rejected with DIA_ERR_UNSUPPORTED. */
int dia_hessian(dia_handle* h, const float* d_I, const unsigned char* d_mask, const float* d_var,
                const float* d_theta, double* d_H);

/* Covariance estimate of the fitted parameters from the Hessian of dia_hessian (Eq. 16-17):
 * Sigma = H^-1, sigma_p = sqrt(Sigma_pp), with the validity test of PAPER.md:193 ("if either the determinant of Sigma
 * is negative, or ... any eigenvalue is found to be negative or zero, then Sigma is not valid").  H is factorised as
 * L L' in FP64 on the device; a symmetric matrix is positive definite -- all eigenvalues > 0, hence det > 0 -- exactly
 * when every Cholesky pivot is positive, so one pivot test stands for both of the paper's (R20).
 *   d_H     [np][np] float64 DEVICE, row-major, symmetric (only the lower triangle is read); not modified;
 *   d_cov   [np][np] float64 DEVICE out, or NULL when only the uncertainties are wanted (skips the back-substitution);
 *   d_sigma [np] float64 DEVICE out: sqrt(Sigma_pp), the Cramer-Rao bound of Eq. 17;
 *   d_info  [5] float64 DEVICE out: { valid (1 = positive definite, 0 = the paper's warning flag), ln det H
 *           (= -ln det Sigma), sigma_P = sqrt(u' Sigma u) for the photometric scale factor P = sum K (Eq. 3; u = 1 on
 *           the m*m kernel pixels), smallest Cholesky pivot, index of the first non-positive pivot or -1 }.
 * When valid == 0 the numbers in d_cov, d_sigma, ln det H and sigma_P are NaN or meaningless.  The first call
 * allocates an np x np workspace (synchronises once); later calls are asynchronous on the handle's stream. */
int dia_covariance(dia_handle* h, const double* d_H, double* d_cov, double* d_sigma, double* d_info);

/* Host-buffer forms of dia_eval_loss_grad and dia_fit: the same operations for callers whose data live in HOST memory
 * (page-locked buffers make the copies asynchronous; pageable ones work, slower).  The library owns the device staging
 * buffers (allocated on first use for cfg->max_epochs epochs, freed by dia_destroy) and a copy stream; both calls
 * SYNCHRONISE before they return, and the host outputs are complete then.  Plain noise model only (no d_var).
 *   dia_eval_loss_grad_host: h_I [n_epochs][n_rows][n_cols], h_theta [n_epochs][np] in; h_loss [n_epochs],
 *     h_grad [n_epochs][np] out.
 *   dia_fit_host: h_theta holds theta0 on entry and theta-hat on exit, h_result [n_epochs] out, h_mask NULL or
 *     [n_epochs][n_rows][n_cols].  The batch is cut into `chunks` groups of epochs (0 = default: 4 when there are at
 *     least 8 epochs, else 1): the copy of group k+1 runs on the copy stream while group k is being fitted, so only the
 *     first copy is exposed; the groups are fitted by dia_fit one after the other, which gives the same result per
 *     epoch as one dia_fit over the whole batch.
 * Errors: as dia_eval_loss_grad / dia_fit, ALLOC for the staging buffers, UNSUPPORTED with DIA_NOISE_FIXED. */
int dia_eval_loss_grad_host(dia_handle* h, int n_epochs, const float* h_I, const float* h_theta,
                            double* h_loss, double* h_grad);
int dia_fit_host(dia_handle* h, const dia_fit_opts* opts, int n_epochs, const float* h_I,
                 const unsigned char* h_mask, float* h_theta, dia_fit_result* h_result, int chunks);

/* Difference image and fit-quality metrics for n_epochs targets at the given theta (the science product,
 * PAPER.md:20; metrics of Eq. 29-30):
 *   D_ij = I_ij - M_ij on the valid region V (mask or not), 0 outside V;
 *   eps_ij = D_ij / sigma_ij over the unmasked pixels of V, sigma from Eq. 6 at the model M (or the caller's
 *   variance map in DIA_NOISE_FIXED);  d_metrics[e] = { N_used, MFB = mean(eps), MFV = sum (eps - MFB)^2 / (N - 1),
 *   chi^2 = sum eps^2 }.
 * d_D [n_epochs][n_rows][n_cols] float32 and d_metrics [n_epochs][4] float64 are DEVICE buffers.  Asynchronous. */
int dia_difference_image(dia_handle* h, int n_epochs, const float* d_I, const unsigned char* d_mask,
                         const float* d_var, const float* d_theta, float* d_D, double* d_metrics);

/* dia_eval_loss_grad for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same operation (see dia_eval_loss_grad above), the same kernels
 * (eval_kernel + reduce_partials_kernel [+ penalty_kernel]), no handle.  The per-CTA FP64 block partials -- the only
 * scratch memory of that path, which dia_create allocates with cudaMalloc -- live in a file-scope __device__ array of
 * DIA_STATIC_SCRATCH_BYTES that every GPU which loads the library holds until the process exits.
 *   cfg      as for dia_create (cfg->max_epochs is ignored: the batch is n_epochs; cfg->stream is the stream);
 *   d_R      [n_rows][n_cols] DEVICE ([n_epochs][..][..] when cfg->n_refs == n_epochs); the other arguments exactly
 *            as for dia_eval_loss_grad.  Inputs and outputs are the caller's; nothing is kept after the call.
 * The call allocates nothing: no cudaMalloc / cudaFree / allocating library routine, on any path.  The first call on a
 * device looks the array's address up (cudaGetSymbolAddress) and the first call per (device, m) sets the kernels'
 * shared-memory attribute; later calls only encode two TMA descriptors on the host and enqueue the kernels.
 * Asynchronous on cfg->stream.  Results are bit-identical to dia_eval_loss_grad on a handle created with
 * max_epochs == n_epochs whenever that handle runs the shared-memory variant of the generic kernel (always, apart from
 * m <= 5 plain objectives and launches long enough for the constant-bank variant, whose sums agree to rounding).
 * Limits and errors: UNSUPPORTED with a message naming both numbers when the partials
 *   8 * n_epochs * (m*m + n_bg + 1) * min(tiles, resident CTAs)  bytes   (tiles = 64 x 64 tiles of the valid region)
 * exceed DIA_STATIC_SCRATCH_BYTES (e.g. one 4096^2 pair up to m = 27, or four at m = 19, fit; sixteen do not);
 * INVALID_ARG / UNSUPPORTED / CUDA as for dia_create and dia_eval_loss_grad (text: dia_last_error(NULL)).
 * ALL CALLS ON A DEVICE SHARE THE ARRAY: two calls whose kernels can overlap on the GPU (different streams without an
 * ordering between them, or two host threads) race on it and both results are garbage; calls on one stream are ordered
 * and safe.  The array keeps the last call's partial sums; the kernel overwrites every element the reduction reads
 * before it reads it, so nothing has to be cleared between calls (tests/test_zz_no_alloc.py runs two in a row). */
#define DIA_STATIC_SCRATCH_BYTES (4u << 20)
int dia_eval_loss_grad_static(const dia_config* cfg, const float* d_R, int n_epochs,
                              const float* d_I, const unsigned char* d_mask, const float* d_var,
                              const float* d_theta, double* d_loss, double* d_grad);

/* Frees the handle's workspace (synchronises the handle's stream first). */
int dia_destroy(dia_handle* h);

const char* dia_status_string(int code);
/* Last error text recorded on this handle (or on the creating thread when h == NULL). */
const char* dia_last_error(const dia_handle* h);

/* Introspection used by bench.py / tests: number of kernels the last eval or fit call
 * enqueued per iteration, and the persistent grid size. */
int dia_get_info(const dia_handle* h, int* grid_blocks, int* threads_per_block,
                 int* smem_bytes, int* launches_per_eval);

/* Register-only FMA microbenchmarks on the current device (no memory traffic; SURVEY.md section 7 hard part 2 asks for
 * the measured FP32 peak that MEASURED_PEAKS.json lacks).  Each writes thread-level fused multiply-adds per second to
 * *fma_per_second (HOST pointer) and synchronises.
 *   dia_measure_fp32_peak: the FMA pipe's peak, FFMAs that read one vector register (pattern 0) -- 97 % of the
 *     nominal SMs x 128 lanes x SM clock on B200, i.e. the nominal peak is attainable and is what the roofline uses;
 *   dia_measure_fp32_pattern: 0 = that; 1 = the forward stencil's packed FFMA2 with the kernel pixel in a uniform
 *     register; 2 = the gradient correlation's packed FFMA2 with all operands in vector registers; 3 = scalar FFMA with
 *     three vector registers (the loops before packing).  1-3 show what the register file's operand bandwidth allows
 *     the kernel's own inner loops (profiles/r02_fp32_peak_sass.md). */
int dia_measure_fp32_peak(void* stream, double* fma_per_second);
int dia_measure_fp32_pattern(void* stream, int pattern, double* fma_per_second);

/* Tensor-core probe (measurement only; csrc/dia_tc_probe.cuh): D [128][N] = sum_k A[r][k] B[n][k] on ONE CTA with
 * tcgen05.mma, the operands built in shared memory from the float32 DEVICE arrays d_A [128][K] and d_B [N][K] exactly as
 * dia_hessian's tensor-core kernel builds its own (same layout, descriptors and hi / lo split), one accumulation chain
 * over all of K in TMEM.  mode: 0 = float16 operands, 1 = float16 hi + lo split (four terms), 2 = tf32 operands,
 * 3 = tf32 big + small split (three terms).  K a positive multiple of 64, N a multiple of 32 up to 256; d_D [128][N]
 * float32 DEVICE.  Asynchronous on `stream`.  Shows how the tensor core rounds when it accumulates. */
int dia_tc_probe_gemm(void* stream, const float* d_A, const float* d_B, float* d_D, int K, int N, int mode);

/* The work plan of dia_hessian's tensor-core kernel for kernel size m and background degree d (host arithmetic only, no
 * device needed; exported for tests): the np = m*m + (d+1)(d+2)/2 parameters fill n_groups = ceil(np / 128) groups of 128
 * operand slots, perm[slot] is the parameter of a slot (-1: empty; 128 n_groups entries), and every CTA type t is the
 * five bytes types[5 t ..] = { g0, g1 (255: none), a_sel, b_start, b_groups }: an operand tile [g0 | g1], the A operand
 * (rows of the result block) group (a_sel ? g1 : g0), the B operand b_groups groups starting at tile position b_start.
 * Every block (gi <= gj) of H is computed by exactly one type.  Returns INVALID_ARG when the outputs are too small
 * (max_types, max_slots), UNSUPPORTED when the table does not fit the kernel's limits (dia_hessian then runs the
 * CUDA-core path). */
int dia_hess_tc_plan(int m, int bg_degree, int* n_groups, int* n_types, unsigned char* types, int max_types,
                     short* perm, int max_slots);

#ifdef __cplusplus
}
#endif
#endif
