// dia_fit.cuh -- on-device optimiser: Adam (Eq. 9) then L-BFGS (PAPER.md:132-135,
// Eq. 10; two-loop recursion), with the switch / stop rules of PAPER.md:244, 248-255 under the
// readings R5-R9 of DESIGN.md.  One CTA per epoch runs a small state machine after every
// evaluation; the loop itself is a CUDA-graph WHILE node whose condition is cleared by the last
// epoch to finish, so the host enqueues one graph launch per fit and never reads a per-iteration value.
// All optimiser state is FP64; theta is rounded to float32 only where it enters the stencil (R9).
#pragma once
#include <cuda_runtime.h>

#include <cstring>
#include <string>

#include "../../include/dia.h"
#include "dia_eval.cuh"

struct dia_handle;

namespace dia {

constexpr int kMaxHistory = 128;
constexpr int kFitThreads = 256;
constexpr int kPerThreadSmall = 4;    // parameters per thread of the optimiser kernel: ceil((31*31+10) / 256) ...
constexpr int kPerThreadLarge = 9;    // ... and ceil((47*47+10) / 256) for 33 <= m <= 47
constexpr int kMaxPerThread = kPerThreadLarge;

inline bool eval_is_aux(const EvalParams& p) { return p.mask || p.flat || p.var || p.noise_kind != 0 || p.hess_q0 >= 0; }
cudaError_t launch_eval(const dia_handle* h, const EvalParams& p, const TensorMaps& tm, bool diff = false);
const void* eval_kernel_ptr(const dia_handle* h, bool aux);
bool eval_uses_const(const dia_handle* h, const EvalParams& p, bool diff);
size_t const_block_bytes(const dia_handle* h, int n_epochs);
const void* eval_kernel_ptr_kc(const dia_handle* h, const EvalParams& p);
ConstBlock* const_stage(const dia_handle* h);
const void* const_symbol(const dia_handle* h);
size_t eval_smem_bytes(const dia_handle* h);
const void* eval_kernel_ptr_p(const dia_handle* h, const EvalParams& p);
size_t eval_smem_bytes_p(const dia_handle* h, const EvalParams& p);
int eval_threads_p(const dia_handle* h, const EvalParams& p);

enum { PH_ADAM = 0, PH_LBFGS = 1, PH_DONE = 2 };

struct FitState {
  int phase, t, n_adam, n_lbfgs, n_evals, status;
  int k, n_pairs, head, nbt;
  double L, Lprev, b1t, b2t, g_switch, alpha, gtd;
};

struct FitBuffers {
  double* theta64;   // [E][np]
  double* g;         // [E][np]  gradient at the current iterate (L-BFGS)
  double* m1;        // [E][np]
  double* m2;        // [E][np]
  double* d;         // [E][np]  search direction
  double* S;         // [E][hist_cap][np]
  double* Y;         // [E][hist_cap][np]
  double* rho;       // [E][hist_cap]
  double* yy;        // [E][hist_cap]
  FitState* st;      // [E]
  float* theta32;    // [E][np]  evaluation point
  int* done;         // [E]
  int* remaining;    // [1]
};

struct FitWorkspace {
  FitBuffers b;
  float* d_theta32;  // alias of b.theta32 (what the eval kernel reads)
  int* d_done;
  int max_epochs, np, hist_cap;
  // instantiated fit graphs, keyed by (pointers, epoch count, options); least recently used entry is replaced
  struct CachedGraph {
    cudaGraph_t graph;
    cudaGraphExec_t exec;
    unsigned char key[256];
    int key_len;
    unsigned long long last_use;
  };
  static constexpr int kGraphCache = 8;
  CachedGraph cache[kGraphCache];
  unsigned long long use_counter;
};

struct StepArgs {
  FitBuffers b;
  const double* partials;
  int n_blocks, np, hist_cap;
  dia_fit_opts o;
  float* theta_out;          // caller's theta [E][np]
  dia_fit_result* result;    // caller's results [E]
  cudaGraphConditionalHandle cond;
  int m;                     // kernel size
  double lamN;               // lambda * N_data of Eq. 20, 0 = no penalty
  int use_graph;             // 1: the last epoch to stop clears the WHILE condition `cond` of the fit graph
};

// Shared-memory scratch of one optimiser transition (fit_step_body): the step kernel declares it statically, the
// cluster kernel (dia_fit_cluster.cuh) carves it out of its dynamic shared memory.
struct StepScratch {
  double (*sh_rows)[kFitThreads / 32];   // [2][8]   block reductions
  double* s_alpha;                       // [kMaxHistory]
  double* gsum;                          // [kFitThreads * PER]
  double* xs;                            // [kFitThreads * PER]  (penalty; the vector of the two-loop recursion)
  // cluster loop only (null in the graph loop): the partial column of every CTA of the epoch in that CTA's shared
  // memory (distributed shared memory) instead of the global partials; a shared-memory copy of the next evaluation
  // point and of the done flag, which the caller hands to the other CTAs of the cluster
  const double* const* peer_cols;        // [n_blocks] -> double [np + 1]
  float* th_local;                       // [np]
  int* done_local;                       // [1]
};
template <int PER>
constexpr size_t step_scratch_bytes() { return 8 * (2 * (kFitThreads / 32) + kMaxHistory + 2 * kFitThreads * PER); }

// ---------------------------------------------------------------- block-wide FP64 reductions
// One barrier per reduction: two scratch rows are used alternately (`par` toggles on every call, and every
// call is made by the whole block), so a row is rewritten only after a later barrier that all of its
// readers have passed.
struct BlockRed {
  double (*sh)[kFitThreads / 32];
  int par;
};
__device__ __forceinline__ double block_sum(double v, BlockRed& br) {
  v = warp_sum_f64(v);
  double* row = br.sh[br.par];
  br.par ^= 1;
  if ((threadIdx.x & 31) == 0) row[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0.0;
#pragma unroll
  for (int w = 0; w < kFitThreads / 32; ++w) s += row[w];
  return s;
}
__device__ __forceinline__ double block_max(double v, BlockRed& br) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { double u = __shfl_xor_sync(0xffffffffu, v, o); v = (u > v || u != u) ? u : v; }
  double* row = br.sh[br.par];
  br.par ^= 1;
  if ((threadIdx.x & 31) == 0) row[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0.0;
#pragma unroll
  for (int w = 0; w < kFitThreads / 32; ++w) { double u = row[w]; s = (u > s || u != u) ? u : s; }
  return s;
}

// (L x)_k for the graph Laplacian of the m x m kernel grid (Eq. 21; 4 edge neighbours)
__device__ __forceinline__ double laplacian_row(const double* __restrict__ x, int m, int k) {
  const int a = k / m, b = k - a * m;
  int nadj = 0;
  double s = 0.0;
  if (a > 0)     { ++nadj; s += x[k - m]; }
  if (a < m - 1) { ++nadj; s += x[k + m]; }
  if (b > 0)     { ++nadj; s += x[k - 1]; }
  if (b < m - 1) { ++nadj; s += x[k + 1]; }
  return nadj * x[k] - s;
}

#ifndef DIA_INST_M      // the stand-alone kernels and the host side belong to the API translation unit only
// Eq. 20: adds lamN |L theta|^2 to loss[e] and 2 lamN L (L theta) to grad[e][0..m*m) for the
// stand-alone evaluation path (one CTA per epoch, launched after reduce_partials_kernel).
__global__ void __launch_bounds__(kFitThreads) penalty_kernel(const float* __restrict__ theta, int m, int np, double lamN,
                                                              double* __restrict__ loss, double* __restrict__ grad) {
  __shared__ double xs[kFitThreads * kMaxPerThread], us[kFitThreads * kMaxPerThread];
  __shared__ double sh_rows[2][kFitThreads / 32];
  BlockRed br{sh_rows, 0};
  const int e = blockIdx.x, nk = m * m, tid = threadIdx.x;
  for (int k = tid; k < nk; k += kFitThreads) xs[k] = (double)theta[(size_t)e * np + k];
  __syncthreads();
  double pen = 0.0;
  for (int k = tid; k < nk; k += kFitThreads) { const double u = laplacian_row(xs, m, k); us[k] = u; pen += u * u; }
  pen = block_sum(pen, br);                    // the barrier inside also publishes us[]
  for (int k = tid; k < nk; k += kFitThreads) grad[(size_t)e * np + k] += 2.0 * lamN * laplacian_row(us, m, k);
  if (tid == 0) loss[e] += lamN * pen;
}

__global__ void fit_init_kernel(FitBuffers b, const float* __restrict__ theta_in, int np, int n_epochs) {
  const int e = blockIdx.x;
  for (int k = threadIdx.x; k < np; k += blockDim.x) {
    const float v = theta_in[(size_t)e * np + k];
    b.theta64[(size_t)e * np + k] = (double)v;
    b.theta32[(size_t)e * np + k] = v;
    b.m1[(size_t)e * np + k] = 0.0;
    b.m2[(size_t)e * np + k] = 0.0;
  }
  if (threadIdx.x == 0) {
    FitState s;
    s.phase = PH_ADAM; s.t = 0; s.n_adam = 0; s.n_lbfgs = 0; s.n_evals = 0; s.status = DIA_FIT_MAX_ITERS;
    s.k = 0; s.n_pairs = 0; s.head = 0; s.nbt = 0;
    s.L = 0.0; s.Lprev = 0.0; s.b1t = 1.0; s.b2t = 1.0; s.g_switch = 0.0; s.alpha = 0.0; s.gtd = 0.0;
    b.st[e] = s;
    b.done[e] = 0;
    if (e == 0) *b.remaining = n_epochs;
  }
}

#endif  // DIA_INST_M

// The two-loop recursion (N&W Alg. 7.4) run by ONE warp: x [np] in shared memory holds q on entry and H q on exit
// (np <= 32 JW <= 256; lane l owns elements l, l + 32, ...).  The 2 n_pairs steps depend on each other through a dot
// product each: a lane-strided partial sum and a warp butterfly, with the history rows of the next D steps already in
// flight in a ring of D register slots, instead of a block-wide sum (two barriers) and rows loaded when needed.
// The warp runs alone (the rest of the block waits at a barrier), so the latency of EVERY instruction of a step adds
// up: the history slot is stepped instead of computed with a modulo, a row address is one multiply-add, the dot
// product is split into independent chains (a dependent FP64 operation costs ~40 cycles on this part).
// Measured (128^2, m = 7, full history of 100 pairs): 65 us per L-BFGS iteration against 102 us for the block-wide
// form (clock64: 110 000 of its 121 000 step cycles were this loop); a step is now ~0.25 us, its dependent chain
// (dot, five shuffle + add levels, scale, update) ~0.2 us.
// Not inlined: its registers must not count against the caller (fit_cluster_kernel runs under a 128-register cap;
// inlined, a first version cost it 5 KB of spills and 15 % of its Adam rate).
template <int JW, int D>
__device__ __noinline__ void two_loop_warp(double* __restrict__ x, int np, const double* __restrict__ Sm,
                                           const double* __restrict__ Ym, const double* __restrict__ rho,
                                           const double* __restrict__ yy, int head, int n_pairs, int hist,
                                           double* __restrict__ s_alpha) {
  const int lane = threadIdx.x & 31;
  double v[JW], a[D][JW], b[D][JW], r[D];
  bool ok[JW];
#pragma unroll
  for (int j = 0; j < JW; ++j) { ok[j] = lane + 32 * j < np; v[j] = ok[j] ? x[lane + 32 * j] : 0.0; }
  // one warp runs alone here, so every instruction's latency counts: the history slot of a step is stepped, not
  // computed with a modulo, and a row's address is one multiply-add
  auto load_rows = [&](int id, double* sr, double* yr, double& rh) {      // history pair in slot id
    const double* sp = Sm + (size_t)id * np + lane;
    const double* yp = Ym + (size_t)id * np + lane;
#pragma unroll
    for (int j = 0; j < JW; ++j) { sr[j] = ok[j] ? sp[32 * j] : 0.0; yr[j] = ok[j] ? yp[32 * j] : 0.0; }
    rh = rho[id];
  };
  auto dot = [](const double* p, const double* q) {     // up to four independent chains: a dependent FP64 FMA costs ~40 cycles
    double c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0;
#pragma unroll
    for (int j = 0; j < JW; j += 4) {
      c0 = fma(p[j], q[j], c0);
      if (j + 1 < JW) c1 = fma(p[j + 1], q[j + 1], c1);
      if (j + 2 < JW) c2 = fma(p[j + 2], q[j + 2], c2);
      if (j + 3 < JW) c3 = fma(p[j + 3], q[j + 3], c3);
    }
    return (c0 + c1) + (c2 + c3);
  };
  auto dec = [&](int id) { return id == 0 ? hist - 1 : id - 1; };
  auto inc = [&](int id) { return id + 1 == hist ? 0 : id + 1; };
  const int id_last = n_pairs > 0 ? (head + n_pairs - 1) % hist : 0;
  int idp = id_last;                                                      // slot of the next row to request
#pragma unroll
  for (int u = 0; u < D; ++u) {
    r[u] = 0.0;
#pragma unroll
    for (int j = 0; j < JW; ++j) { a[u][j] = 0.0; b[u][j] = 0.0; }
    if (u < n_pairs) { load_rows(idp, a[u], b[u], r[u]); idp = dec(idp); }
  }
  for (int base = n_pairs - 1; base >= 0; base -= D) {
#pragma unroll
    for (int u = 0; u < D; ++u) {
      const int i = base - u;                          // slot u holds step i
      if (i >= 0) {
        const double al = r[u] * warp_sum_f64(dot(a[u], v));
        if (lane == 0) s_alpha[i] = al;
#pragma unroll
        for (int j = 0; j < JW; ++j) v[j] -= al * b[u][j];
        if (i - D >= 0) { load_rows(idp, a[u], b[u], r[u]); idp = dec(idp); }
      }
    }
  }
  double gamma = 1.0;
  if (n_pairs > 0) gamma = (1.0 / rho[id_last]) / yy[id_last];
#pragma unroll
  for (int j = 0; j < JW; ++j) v[j] *= gamma;
  __syncwarp();
  idp = head;
#pragma unroll
  for (int u = 0; u < D; ++u)
    if (u < n_pairs) { load_rows(idp, a[u], b[u], r[u]); idp = inc(idp); }
  for (int base = 0; base < n_pairs; base += D) {
#pragma unroll
    for (int u = 0; u < D; ++u) {
      const int i = base + u;
      if (i < n_pairs) {
        const double c = s_alpha[i] - r[u] * warp_sum_f64(dot(b[u], v));
#pragma unroll
        for (int j = 0; j < JW; ++j) v[j] += c * a[u][j];
        if (i + D < n_pairs) { load_rows(idp, a[u], b[u], r[u]); idp = inc(idp); }
      }
    }
  }
#pragma unroll
  for (int j = 0; j < JW; ++j) if (ok[j]) x[lane + 32 * j] = v[j];
}

// The same recursion for 256 < np <= 32 JW <= 512 (m = 17 .. 21: the paper's stamp fits): the register ring does not
// fit beside v there, so a row is reloaded IN PLACE as soon as its last use of the step is over -- the S row right
// after the dot product, the Y row right after the update (the other way round in the second loop) -- and is in flight
// during the butterfly and the rest of the step.
template <int JW>
__device__ __noinline__ void two_loop_warp_inplace(double* __restrict__ x, int np, const double* __restrict__ Sm,
                                                   const double* __restrict__ Ym, const double* __restrict__ rho,
                                                   const double* __restrict__ yy, int head, int n_pairs, int hist,
                                                   double* __restrict__ s_alpha) {
  const int lane = threadIdx.x & 31;
  double v[JW], a[JW], b[JW];
  bool ok[JW];
#pragma unroll
  for (int j = 0; j < JW; ++j) { ok[j] = lane + 32 * j < np; v[j] = ok[j] ? x[lane + 32 * j] : 0.0; a[j] = 0.0; b[j] = 0.0; }
  auto load = [&](const double* M, int id, double* dst) {
    const double* p = M + (size_t)id * np + lane;
#pragma unroll
    for (int j = 0; j < JW; ++j) dst[j] = ok[j] ? p[32 * j] : 0.0;
  };
  auto dot = [](const double* p, const double* q) {
    double c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0;
#pragma unroll
    for (int j = 0; j < JW; j += 4) {
      c0 = fma(p[j], q[j], c0);
      if (j + 1 < JW) c1 = fma(p[j + 1], q[j + 1], c1);
      if (j + 2 < JW) c2 = fma(p[j + 2], q[j + 2], c2);
      if (j + 3 < JW) c3 = fma(p[j + 3], q[j + 3], c3);
    }
    return (c0 + c1) + (c2 + c3);
  };
  auto dec = [&](int id) { return id == 0 ? hist - 1 : id - 1; };
  auto inc = [&](int id) { return id + 1 == hist ? 0 : id + 1; };
  const int id_last = n_pairs > 0 ? (head + n_pairs - 1) % hist : 0;
  int id = id_last;
  double r = 0.0;
  if (n_pairs > 0) { load(Sm, id, a); load(Ym, id, b); r = rho[id]; }
  for (int i = n_pairs - 1; i >= 0; --i) {
    const int idn = dec(id);
    const double part = dot(a, v);
    if (i > 0) load(Sm, idn, a);                       // S of the next step: in flight during the butterfly
    const double al = r * warp_sum_f64(part);
    if (lane == 0) s_alpha[i] = al;
#pragma unroll
    for (int j = 0; j < JW; ++j) v[j] -= al * b[j];
    if (i > 0) { load(Ym, idn, b); r = rho[idn]; }
    id = idn;
  }
  double gamma = 1.0;
  if (n_pairs > 0) gamma = (1.0 / rho[id_last]) / yy[id_last];
#pragma unroll
  for (int j = 0; j < JW; ++j) v[j] *= gamma;
  __syncwarp();
  id = head;
  if (n_pairs > 0) { load(Sm, id, a); load(Ym, id, b); r = rho[id]; }
  for (int i = 0; i < n_pairs; ++i) {
    const int idn = inc(id);
    const double part = dot(b, v);
    if (i + 1 < n_pairs) load(Ym, idn, b);
    const double c = s_alpha[i] - r * warp_sum_f64(part);
#pragma unroll
    for (int j = 0; j < JW; ++j) v[j] += c * a[j];
    if (i + 1 < n_pairs) { load(Sm, idn, a); r = rho[idn]; }
    id = idn;
  }
#pragma unroll
  for (int j = 0; j < JW; ++j) if (ok[j]) x[lane + 32 * j] = v[j];
}

// One optimiser transition for epoch e, run by one CTA of kFitThreads threads after every evaluation of that epoch.
template <int PER>
__device__ __forceinline__ void fit_step_body(const StepArgs& a, const int e, const StepScratch& sc) {
  BlockRed sh{sc.sh_rows, 0};
  double* const s_alpha = sc.s_alpha;
  const int np = a.np, nk = a.m * a.m, tid = threadIdx.x;   // nk kernel pixels, np - nk background coefficients
  const dia_fit_opts& o = a.o;
  FitState st = a.b.st[e];                       // every thread holds a private copy; thread 0 writes back

  double* theta = a.b.theta64 + (size_t)e * np;
  double* gcur = a.b.g + (size_t)e * np;
  double* dvec = a.b.d + (size_t)e * np;
  double* Sm = a.b.S + (size_t)e * a.hist_cap * np;
  double* Ym = a.b.Y + (size_t)e * a.hist_cap * np;
  double* rho = a.b.rho + (size_t)e * a.hist_cap;
  double* yy = a.b.yy + (size_t)e * a.hist_cap;
  float* th32 = a.b.theta32 + (size_t)e * np;
  const int hist = o.lbfgs_history;

  // ---- second-level reduction of the evaluation's block partials: one warp per output, fixed order
  double* const gsum = sc.gsum;
  double gn[PER];
  double Ln = 0.0;
  {
    const double* src = a.partials + (size_t)e * (np + 1) * a.n_blocks;
    const int lane = tid & 31, wid = tid >> 5;
    if (a.n_blocks <= 8) {
      // few columns (a small image; always in the cluster loop): one thread per output adds its <= 8 values in the
      // association order of the warp butterfly below -- ((v0+v4)+(v2+v6)) + ((v1+v5)+(v3+v7)), absent columns 0 -- so
      // the bits are those of the general path, without its four butterflies per warp in the chain (3800 -> ~800
      // cycles of a 20 000-cycle Adam iteration at 128^2)
      for (int k = tid; k < np + 1; k += kFitThreads) {
        double v[8];
#pragma unroll
        for (int b = 0; b < 8; ++b)
          v[b] = b < a.n_blocks ? (sc.peer_cols ? sc.peer_cols[b][k] : src[(size_t)k * a.n_blocks + b]) : 0.0;
        gsum[k] = ((v[0] + v[4]) + (v[2] + v[6])) + ((v[1] + v[5]) + (v[3] + v[7]));
      }
    } else
    // four rows per warp at a time, so that enough loads are in flight to hide the L2 latency
    for (int k = wid * 4; k < np + 1; k += (kFitThreads / 32) * 4) {
      double s4[4] = {0.0, 0.0, 0.0, 0.0};
      for (int b = lane; b < a.n_blocks; b += 32) {
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if (k + j < np + 1) s4[j] += sc.peer_cols ? sc.peer_cols[b][k + j] : src[(size_t)(k + j) * a.n_blocks + b];
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const double s = warp_sum_f64(s4[j]);
        if (lane == 0 && k + j < np + 1) gsum[k + j] = s;
      }
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      const int k = tid + q * kFitThreads;
      gn[q] = (k < np) ? gsum[k] : 0.0;
    }
    Ln = gsum[np];                               // loss lives in row np
    __syncthreads();
  }
  if (a.lamN > 0.0) {                            // Eq. 20 penalty at the evaluation point (uniform branch)
    double* const xs = sc.xs;
    double* const us = gsum;                     // gsum is dead: gn / Ln hold its content (keeps static shared memory < 48 KB)
    for (int k = tid; k < nk; k += kFitThreads) xs[k] = (double)th32[k];
    __syncthreads();
    double pen = 0.0;
    for (int k = tid; k < nk; k += kFitThreads) { const double u = laplacian_row(xs, a.m, k); us[k] = u; pen += u * u; }
    pen = block_sum(pen, sh);
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      const int k = tid + q * kFitThreads;
      if (k < nk) gn[q] += 2.0 * a.lamN * laplacian_row(us, a.m, k);
    }
    Ln += a.lamN * pen;
  }
  st.n_evals += 1;
  bool finished = false;
  bool at_top = false;                           // enter the L-BFGS loop head with (st.L, gcur) current

  if (st.phase == PH_ADAM) {
    const int t = st.t + 1;
    if (!isfinite(Ln)) {
      st.status = DIA_FIT_NONFINITE; st.L = Ln; finished = true;
#pragma unroll
      for (int q = 0; q < PER; ++q) { const int k = tid + q * kFitThreads; if (k < np) gcur[k] = gn[q]; }
    } else {
      bool sw;
      if (o.force_adam_iters >= 0) sw = t > o.force_adam_iters;
      else sw = (t >= 2 && fabs(Ln - st.Lprev) < o.tol_switch * fabs(st.Lprev)) || (t > o.max_adam_iters);
      if (!sw) {
        st.b1t *= o.adam_beta1; st.b2t *= o.adam_beta2;
#pragma unroll
        for (int q = 0; q < PER; ++q) {
          const int k = tid + q * kFitThreads;
          if (k < np) {
            double* m1 = a.b.m1 + (size_t)e * np; double* m2 = a.b.m2 + (size_t)e * np;
            const double g = gn[q];
            const double v1 = o.adam_beta1 * m1[k] + (1.0 - o.adam_beta1) * g;
            const double v2 = o.adam_beta2 * m2[k] + (1.0 - o.adam_beta2) * g * g;
            m1[k] = v1; m2[k] = v2;
            const double mh = v1 / (1.0 - st.b1t), vh = v2 / (1.0 - st.b2t);
            const double lr = (k < nk) ? (double)o.lr_kernel : (double)o.lr_b0;
            const double th = theta[k] - lr * mh / (sqrt(vh) + o.adam_eps);
            theta[k] = th;
            th32[k] = (float)th;
            if (sc.th_local) sc.th_local[k] = (float)th;
          }
        }
        st.n_adam += 1; st.Lprev = Ln; st.t = t; st.L = Ln;
      } else {
        // switch: L-BFGS starts from this iterate and reuses this evaluation (R6)
        double gi = 0.0;
#pragma unroll
        for (int q = 0; q < PER; ++q) {
          const int k = tid + q * kFitThreads;
          if (k < np) { gcur[k] = gn[q]; const double ag = fabs(gn[q]); gi = (ag > gi || ag != ag) ? ag : gi; }
        }
        st.g_switch = block_max(gi, sh);
        st.L = Ln; st.phase = PH_LBFGS; st.k = 1; st.n_pairs = 0; st.head = 0; st.t = t;
        at_top = true;
      }
    }
  } else {  // PH_LBFGS: (Ln, gn) is the trial point theta + alpha d
    const bool bad = !isfinite(Ln);
    if (o.lbfgs_backtrack && (bad || Ln > st.L + 1e-4 * st.alpha * st.gtd) && st.nbt < 20) {
      st.alpha *= 0.5; st.nbt += 1;
#pragma unroll
      for (int q = 0; q < PER; ++q) {
        const int k = tid + q * kFitThreads;
        if (k < np) {
          th32[k] = (float)(theta[k] + st.alpha * dvec[k]);
          if (sc.th_local) sc.th_local[k] = th32[k];
        }
      }
    } else if (bad) {
      st.status = DIA_FIT_NONFINITE; finished = true;
    } else {
      double sty = 0.0, yty = 0.0;
      double sv[PER], yv[PER];
#pragma unroll
      for (int q = 0; q < PER; ++q) {
        const int k = tid + q * kFitThreads;
        sv[q] = 0.0; yv[q] = 0.0;
        if (k < np) { sv[q] = st.alpha * dvec[k]; yv[q] = gn[q] - gcur[k]; sty += sv[q] * yv[q]; yty += yv[q] * yv[q]; }
      }
      sty = block_sum(sty, sh);
      yty = block_sum(yty, sh);
      if (sty > 1e-10) {                                 // R7 curvature guard, FIFO eviction
        int id;
        if (st.n_pairs < hist) { id = (st.head + st.n_pairs) % hist; st.n_pairs += 1; }
        else { id = st.head; st.head = (st.head + 1) % hist; }
#pragma unroll
        for (int q = 0; q < PER; ++q) {
          const int k = tid + q * kFitThreads;
          if (k < np) { Sm[(size_t)id * np + k] = sv[q]; Ym[(size_t)id * np + k] = yv[q]; }
        }
        if (tid == 0) { rho[id] = 1.0 / sty; yy[id] = yty; }
      }
      const double dL = fabs(Ln - st.L);
#pragma unroll
      for (int q = 0; q < PER; ++q) {
        const int k = tid + q * kFitThreads;
        if (k < np) { theta[k] += sv[q]; gcur[k] = gn[q]; }
      }
      st.L = Ln; st.n_lbfgs += 1;
      if (o.force_lbfgs_iters < 0) {
        if (dL <= o.tol_change_rel * fabs(st.L)) { st.status = DIA_FIT_CONVERGED_CHANGE; finished = true; }   // R8
        else if (st.k >= o.max_lbfgs_iters) { st.status = DIA_FIT_MAX_ITERS; finished = true; }
      }
      if (!finished) { st.k += 1; at_top = true; }
      __syncthreads();                                   // rho / yy / S / Y visible to the block
    }
  }

  if (at_top && !finished) {
    // ---- L-BFGS loop head: stop test, two-loop recursion, first trial point
    double q4[PER];
    double gi = 0.0, g1 = 0.0;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      const int k = tid + q * kFitThreads;
      q4[q] = (k < np) ? gcur[k] : 0.0;
      const double ag = fabs(q4[q]);
      gi = (ag > gi || ag != ag) ? ag : gi;
      g1 += ag;
    }
    gi = block_max(gi, sh);
    g1 = block_sum(g1, sh);
    bool stop = false;
    if (o.force_lbfgs_iters >= 0) { if (st.k > o.force_lbfgs_iters) { st.status = DIA_FIT_MAX_ITERS; stop = true; } }
    else if (gi < o.tol_grad_abs || gi < o.tol_grad_rel * st.g_switch) { st.status = DIA_FIT_CONVERGED_GRAD; stop = true; }
    if (stop) {
      finished = true;
    } else {
      double gq[PER];
#pragma unroll
      for (int q = 0; q < PER; ++q) gq[q] = q4[q];
      // two-loop recursion (N&W Alg. 7.4)
      if (np <= 512) {                                    // one warp, history rows prefetched (two_loop_warp)
#pragma unroll
        for (int q = 0; q < PER; ++q) { const int k = tid + q * kFitThreads; if (k < np) sc.xs[k] = q4[q]; }
        __syncthreads();
        if (tid < 32) {
          if (np <= 64) two_loop_warp<2, 6>(sc.xs, np, Sm, Ym, rho, yy, st.head, st.n_pairs, hist, s_alpha);
          else if (np <= 128) two_loop_warp<4, 4>(sc.xs, np, Sm, Ym, rho, yy, st.head, st.n_pairs, hist, s_alpha);
          else if (np <= 256) two_loop_warp<8, 2>(sc.xs, np, Sm, Ym, rho, yy, st.head, st.n_pairs, hist, s_alpha);
          else if (np <= 384) two_loop_warp_inplace<12>(sc.xs, np, Sm, Ym, rho, yy, st.head, st.n_pairs, hist, s_alpha);
          else two_loop_warp_inplace<16>(sc.xs, np, Sm, Ym, rho, yy, st.head, st.n_pairs, hist, s_alpha);
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < PER; ++q) { const int k = tid + q * kFitThreads; q4[q] = (k < np) ? sc.xs[k] : 0.0; }
      } else {
        for (int i = st.n_pairs - 1; i >= 0; --i) {
          const int id = (st.head + i) % hist;
          double part = 0.0;
#pragma unroll
          for (int q = 0; q < PER; ++q) { const int k = tid + q * kFitThreads; if (k < np) part += Sm[(size_t)id * np + k] * q4[q]; }
          const double al = rho[id] * block_sum(part, sh);
          if (tid == 0) s_alpha[i] = al;
#pragma unroll
          for (int q = 0; q < PER; ++q) { const int k = tid + q * kFitThreads; if (k < np) q4[q] -= al * Ym[(size_t)id * np + k]; }
        }
        __syncthreads();
        double gamma = 1.0;
        if (st.n_pairs > 0) { const int id = (st.head + st.n_pairs - 1) % hist; gamma = (1.0 / rho[id]) / yy[id]; }
#pragma unroll
        for (int q = 0; q < PER; ++q) q4[q] *= gamma;
        for (int i = 0; i < st.n_pairs; ++i) {
          const int id = (st.head + i) % hist;
          double part = 0.0;
#pragma unroll
          for (int q = 0; q < PER; ++q) { const int k = tid + q * kFitThreads; if (k < np) part += Ym[(size_t)id * np + k] * q4[q]; }
          const double beta = rho[id] * block_sum(part, sh);
          const double c = s_alpha[i] - beta;
#pragma unroll
          for (int q = 0; q < PER; ++q) { const int k = tid + q * kFitThreads; if (k < np) q4[q] += c * Sm[(size_t)id * np + k]; }
        }
      }
      double part = 0.0;
#pragma unroll
      for (int q = 0; q < PER; ++q) { q4[q] = -q4[q]; part += gq[q] * q4[q]; }
      double gtd = block_sum(part, sh);
      if (!(gtd < 0.0)) {                                 // not a descent direction: drop the history
        st.n_pairs = 0; st.head = 0;
        part = 0.0;
#pragma unroll
        for (int q = 0; q < PER; ++q) { q4[q] = -gq[q]; part += gq[q] * q4[q]; }
        gtd = block_sum(part, sh);
      }
      double alpha = o.lbfgs_lr;
      if (st.n_pairs == 0) alpha *= (g1 > 1.0) ? 1.0 / g1 : 1.0;     // R7 first-step scaling
      st.alpha = alpha; st.gtd = gtd; st.nbt = 0;
#pragma unroll
      for (int q = 0; q < PER; ++q) {
        const int k = tid + q * kFitThreads;
        if (k < np) {
          dvec[k] = q4[q]; th32[k] = (float)(theta[k] + alpha * q4[q]);
          if (sc.th_local) sc.th_local[k] = th32[k];
        }
      }
    }
  }

  if (finished) {
    double gi = 0.0, P = 0.0;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      const int k = tid + q * kFitThreads;
      if (k < np) {
        const double ag = fabs(gcur[k]);
        gi = (ag > gi || ag != ag) ? ag : gi;
        if (k < nk) P += theta[k];
        a.theta_out[(size_t)e * np + k] = (float)theta[k];
      }
    }
    gi = block_max(gi, sh);
    P = block_sum(P, sh);                                  // Eq. 3
    st.phase = PH_DONE;
    if (tid == 0) {
      dia_fit_result r;
      r.loss = st.L; r.grad_inf_norm = gi; r.photometric_scale = P;
      r.n_adam = st.n_adam; r.n_lbfgs = st.n_lbfgs; r.n_evals = st.n_evals; r.status = st.status;
      a.result[e] = r;
      a.b.done[e] = 1;
      if (sc.done_local) *sc.done_local = 1;
      __threadfence();
      if (atomicSub(a.b.remaining, 1) == 1 && a.use_graph) cudaGraphSetConditional(a.cond, 0);
    }
  }
  if (tid == 0) a.b.st[e] = st;
}

#ifndef DIA_INST_M
// Two CTAs per SM in the launch bounds = a cap of 128 registers: the one-warp recursions above would otherwise raise the
// kernel's allocation to 178 registers per thread for all 256 threads, and the step kernel's place in the graph loop is
// sensitive to its footprint -- measured per Adam iteration at c2 (1024^2, m = 19: eval 45 us): 54.6 us with the cap,
// 65.4 us without, 62.1 us for the 88-register kernel before the recursions were added.
template <int PER>
__global__ void __launch_bounds__(kFitThreads, 2) fit_step_kernel(const StepArgs a) {
  const int e = blockIdx.x;
  if (a.b.done[e]) return;
  __shared__ double sh_rows[2][kFitThreads / 32];
  __shared__ double s_alpha[kMaxHistory];
  __shared__ double gsum[kFitThreads * PER];
  __shared__ double xs[kFitThreads * PER];
  const StepScratch sc{sh_rows, s_alpha, gsum, xs, nullptr, nullptr, nullptr};
  fit_step_body<PER>(a, e, sc);
}

// ---------------------------------------------------------------- host side
inline int fit_workspace_create(FitWorkspace* w, int max_epochs, int np) {
  std::memset(w, 0, sizeof(*w));
  w->max_epochs = max_epochs; w->np = np; w->hist_cap = kMaxHistory;
  const size_t E = (size_t)max_epochs, n = E * np;
  auto A = [&](void** p, size_t bytes) { return cudaMalloc(p, bytes) == cudaSuccess; };
  bool ok = A((void**)&w->b.theta64, 8 * n) && A((void**)&w->b.g, 8 * n) && A((void**)&w->b.m1, 8 * n) &&
            A((void**)&w->b.m2, 8 * n) && A((void**)&w->b.d, 8 * n) &&
            A((void**)&w->b.S, 8 * n * kMaxHistory) && A((void**)&w->b.Y, 8 * n * kMaxHistory) &&
            A((void**)&w->b.rho, 8 * E * kMaxHistory) && A((void**)&w->b.yy, 8 * E * kMaxHistory) &&
            A((void**)&w->b.st, sizeof(FitState) * E) && A((void**)&w->b.theta32, 4 * n) &&
            A((void**)&w->b.done, 4 * E) && A((void**)&w->b.remaining, 4);
  if (!ok) { cudaGetLastError(); return DIA_ERR_ALLOC; }
  w->d_theta32 = w->b.theta32; w->d_done = w->b.done;
  return DIA_OK;
}

inline void fit_workspace_destroy(FitWorkspace* w) {
  for (auto& c : w->cache) {
    if (c.exec) cudaGraphExecDestroy(c.exec);
    if (c.graph) cudaGraphDestroy(c.graph);
  }
  void* ptrs[] = {w->b.theta64, w->b.g, w->b.m1, w->b.m2, w->b.d, w->b.S, w->b.Y, w->b.rho, w->b.yy,
                  w->b.st, w->b.theta32, w->b.done, w->b.remaining};
  for (void* p : ptrs) cudaFree(p);
  std::memset(w, 0, sizeof(*w));
}

#define DIA_CU(x) do { cudaError_t _e = (x); if (_e != cudaSuccess) { *err = std::string(#x) + ": " + cudaGetErrorString(_e); return DIA_ERR_CUDA; } } while (0)

// Builds (or reuses) the fit graph  init -> WHILE { eval ; step }  and launches it once.
inline int fit_run(FitWorkspace* w, const dia_handle* h, const EvalParams& p, const TensorMaps& tm,
                   const dia_fit_opts& o,
                   int n_epochs, float* d_theta, dia_fit_result* d_result, int grid, int part_cols, int unroll,
                   int m, double lamN,
                   cudaStream_t stream, std::string* err) {
  unsigned char key[256];
  int len = 0;
  auto put = [&](const void* src, size_t n) { std::memcpy(key + len, src, n); len += (int)n; };
  put(&n_epochs, sizeof(int)); put(&p.I, sizeof(void*)); put(&p.mask, sizeof(void*)); put(&p.var, sizeof(void*));
  put(&d_theta, sizeof(void*)); put(&d_result, sizeof(void*)); put(&o, sizeof(o)); put(&unroll, sizeof(int)); put(&lamN, sizeof(double));
  FitWorkspace::CachedGraph* slot = nullptr;
  for (auto& c : w->cache)
    if (c.exec && c.key_len == len && std::memcmp(key, c.key, len) == 0) slot = &c;
  if (!slot) {
    slot = &w->cache[0];
    for (auto& c : w->cache)
      if (!c.exec) { slot = &c; break; } else if (c.last_use < slot->last_use) slot = &c;
    if (slot->exec) { cudaGraphExecDestroy(slot->exec); slot->exec = nullptr; }
    if (slot->graph) { cudaGraphDestroy(slot->graph); slot->graph = nullptr; }
    DIA_CU(cudaGraphCreate(&slot->graph, 0));
    // node 1: init
    const float* theta_in = d_theta;
    int np = w->np, ne = n_epochs;
    void* init_args[] = {(void*)&w->b, (void*)&theta_in, (void*)&np, (void*)&ne};
    cudaKernelNodeParams kp = {};
    kp.func = (void*)fit_init_kernel; kp.gridDim = dim3(n_epochs); kp.blockDim = dim3(256);
    kp.sharedMemBytes = 0; kp.kernelParams = init_args; kp.extra = nullptr;
    cudaGraphNode_t n_init;
    DIA_CU(cudaGraphAddKernelNode(&n_init, slot->graph, nullptr, 0, &kp));
    // node 2: WHILE
    cudaGraphConditionalHandle cond;
    DIA_CU(cudaGraphConditionalHandleCreate(&cond, slot->graph, 1, cudaGraphCondAssignDefault));
    cudaGraphNodeParams cp = {};
    cp.type = cudaGraphNodeTypeConditional;
    cp.conditional.handle = cond; cp.conditional.type = cudaGraphCondTypeWhile; cp.conditional.size = 1;
    cudaGraphNode_t n_while;
    DIA_CU(cudaGraphAddNode(&n_while, slot->graph, &n_init, 1, &cp));
    cudaGraph_t body = cp.conditional.phGraph_out[0];
    // body: eval -> step
    EvalParams pe = p;
    TensorMaps tme = tm;
    void* eval_args[] = {(void*)&pe, (void*)&tme};
    cudaKernelNodeParams ke = {};
    const bool kc = eval_uses_const(h, p, false);
    ke.func = kc ? (void*)eval_kernel_ptr_kc(h, p) : (void*)eval_kernel_ptr_p(h, p);
    ke.gridDim = dim3(grid); ke.blockDim = dim3(eval_threads_p(h, p));
    ke.sharedMemBytes = (unsigned)eval_smem_bytes_p(h, p); ke.kernelParams = eval_args; ke.extra = nullptr;
    StepArgs sa;
    sa.b = w->b; sa.partials = p.partials; sa.n_blocks = part_cols; sa.np = w->np; sa.hist_cap = w->hist_cap;
    sa.o = o; sa.theta_out = d_theta; sa.result = d_result; sa.cond = cond;
    sa.m = m; sa.lamN = lamN; sa.use_graph = 1;
    void* step_args[] = {(void*)&sa};
    cudaKernelNodeParams ks = {};
    ks.func = w->np <= kFitThreads * kPerThreadSmall ? (void*)fit_step_kernel<kPerThreadSmall>
                                                      : (void*)fit_step_kernel<kPerThreadLarge>;
    ks.gridDim = dim3(n_epochs); ks.blockDim = dim3(kFitThreads);
    ks.sharedMemBytes = 0; ks.kernelParams = step_args; ks.extra = nullptr;
    // The body holds `unroll` (eval ; step) pairs: re-evaluating the WHILE condition costs several
    // microseconds, which matters when an evaluation takes ~10 us (small images).  Pairs that run after
    // every epoch has stopped find done[e] set and return at once.
    // constant-bank variant: refresh the constant block (active epochs, kernel pixels) before every evaluation
    const float* pk_theta = p.theta;  const int* pk_done = p.done;
    int pk_ne = n_epochs, pk_np = w->np, pk_m = m, pk_kp = (m + 3) / 4 * 4;
    ConstBlock* pk_dst = const_stage(h);
    void* pack_args[] = {(void*)&pk_theta, (void*)&pk_done, (void*)&pk_ne, (void*)&pk_np, (void*)&pk_m, (void*)&pk_kp,
                         (void*)&pk_dst};
    cudaKernelNodeParams kpk = {};
    kpk.func = (void*)pack_const_kernel; kpk.gridDim = dim3(1); kpk.blockDim = dim3(256);
    kpk.sharedMemBytes = 0; kpk.kernelParams = pack_args; kpk.extra = nullptr;
    cudaGraphNode_t prev = nullptr;
    for (int u = 0; u < unroll; ++u) {
      cudaGraphNode_t n_eval, n_step;
      if (kc) {
        cudaGraphNode_t n_pack, n_copy;
        DIA_CU(cudaGraphAddKernelNode(&n_pack, body, prev ? &prev : nullptr, prev ? 1 : 0, &kpk));
        DIA_CU(cudaGraphAddMemcpyNodeToSymbol(&n_copy, body, &n_pack, 1, const_symbol(h), pk_dst, const_block_bytes(h, n_epochs), 0,
                                              cudaMemcpyDeviceToDevice));
        prev = n_copy;
      }
      DIA_CU(cudaGraphAddKernelNode(&n_eval, body, prev ? &prev : nullptr, prev ? 1 : 0, &ke));
      DIA_CU(cudaGraphAddKernelNode(&n_step, body, &n_eval, 1, &ks));
      prev = n_step;
    }
    DIA_CU(cudaGraphInstantiate(&slot->exec, slot->graph, 0));
    std::memcpy(slot->key, key, len); slot->key_len = len;
  }
  slot->last_use = ++w->use_counter;
  DIA_CU(cudaGraphLaunch(slot->exec, stream));
  return DIA_OK;
}

#endif  // DIA_INST_M

}  // namespace dia
