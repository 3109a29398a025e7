// dia_api.cu -- host side of the C ABI declared in include/dia.h.
#include "../../include/dia.h"

#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <atomic>
#include <cstddef>
#include <cstring>
#include <new>
#include <mutex>
#include <string>
#include <vector>

#include "dia_eval.cuh"
#include "dia_eval_small.cuh"
#include "dia_fit.cuh"
#include "dia_fit_cluster.cuh"
#include "dia_hess.cuh"
#include "dia_hess_tc.cuh"
#include "dia_cov.cuh"
#include "dia_probe.cuh"
#include "dia_tc_probe.cuh"

struct dia_handle {
  dia_config cfg;
  const float* d_R;
  cudaStream_t stream;
  int grid, np, sms;       // grid: resident CTAs (SMs x occupancy), capped by max_epochs x tiles
  int tiles, n_refs;
  int small_grid;          // > 0: the plain objective of this handle (m <= 5) runs eval_small_kernel on at most this many CTAs
  int grid_limit;          // test hook DIA_GRID_LIMIT (0 = none)
  int cluster_fit;         // 1: dia_fit may run small image pairs in fit_cluster_kernel (0: test hook DIA_DISABLE_CLUSTER, or
                           // the kernel does not fit); -1: not decided yet
  int flush_tiles;         // tiles between two FP64 folds of the FP32 gradient strips (kFlushTiles; test hook DIA_FLUSH_TILES)
  dia::ConstBlock* d_const_stage;   // staging copy of the constant block; non-null iff this handle may use the bank
  size_t smem;
  int use_tma;             // rows 16-byte aligned: R / I tiles are staged with TMA tensor copies
  CUtensorMap tmR;         // valid iff use_tma
  double* d_partials;      // [max_epochs][np+1][min(tiles, grid)]
  dia::FitWorkspace fit;   // device optimiser state + cached graph
  dia::HessWorkspace hess; // dia_hessian scratch, allocated on first use
  struct HostPath {        // device staging of the host-buffer entry points (dia_*_host), allocated on first use
    float* dI = nullptr;  float* dth = nullptr;  unsigned char* dmask = nullptr;  dia_fit_result* dres = nullptr;
    double* dloss = nullptr;  double* dgrad = nullptr;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ready[16] = {};          // chunk k has arrived
    cudaEvent_t free_ev = nullptr;       // the staging buffers are free again
  } host;
  std::string err;
};

static thread_local std::string g_create_err;
// There is one constant block (dia::c_blk) per kernel size and device.  Every evaluation that uses it refreshes it
// on the handle's stream right before its launch, so handles that share a stream can share the block; the first
// stream to claim the block of a kernel size keeps it until its last handle is destroyed, and handles on other
// streams (or devices) run the shared-memory variant of the kernel.
struct ConstSlot { void* stream = nullptr; int device = -1; int refs = 0; };
static std::mutex g_const_mutex;
static ConstSlot g_const_slot[DIA_MAX_KERNEL_SIZE + 1];
static std::mutex g_const_launch_mutex[DIA_MAX_KERNEL_SIZE + 1];   // (pack, copy, launch) of one evaluation is atomic per kernel size
static bool const_slot_acquire(int m, void* stream, int device) {
  std::lock_guard<std::mutex> lock(g_const_mutex);
  ConstSlot& sl = g_const_slot[m];
  if (sl.refs > 0 && (sl.stream != stream || sl.device != device)) return false;
  sl.stream = stream;  sl.device = device;  ++sl.refs;
  return true;
}
static void const_slot_release(int m) {
  std::lock_guard<std::mutex> lock(g_const_mutex);
  if (g_const_slot[m].refs > 0) --g_const_slot[m].refs;
}

static int fail(dia_handle* h, int code, const std::string& msg) {
  if (h) h->err = msg; else g_create_err = msg;
  return code;
}
static int cuda_fail(dia_handle* h, cudaError_t e, const char* what) {
  return fail(h, DIA_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

extern "C" const char* dia_status_string(int code) {
  switch (code) {
    case DIA_OK: return "ok";
    case DIA_ERR_INVALID_ARG: return "invalid argument";
    case DIA_ERR_CUDA: return "CUDA error";
    case DIA_ERR_ALLOC: return "allocation failed";
    case DIA_ERR_UNSUPPORTED: return "unsupported configuration";
    default: return "unknown status";
  }
}
extern "C" const char* dia_last_error(const dia_handle* h) { return h ? h->err.c_str() : g_create_err.c_str(); }

extern "C" void dia_default_fit_opts(dia_fit_opts* o) {
  if (!o) return;
  o->lr_kernel = 1e-3f;  o->lr_b0 = 10.0f;
  o->adam_beta1 = 0.9;  o->adam_beta2 = 0.999;  o->adam_eps = 1e-8;
  o->tol_switch = 1e-6;  o->lbfgs_lr = 1.0;
  o->lbfgs_history = 100;  o->lbfgs_backtrack = 0;
  o->tol_change_rel = 1e-8;  o->tol_grad_abs = 1e-7;  o->tol_grad_rel = 0.0;
  o->max_adam_iters = 20000;  o->max_lbfgs_iters = 500;
  o->force_adam_iters = -1;  o->force_lbfgs_iters = -1;
}

// ---------------------------------------------------------------------------------------------
// kernel-size dispatch: one instantiation per odd m
// ---------------------------------------------------------------------------------------------
#ifndef DIA_FOR_EACH_M
#define DIA_FOR_EACH_M(X) X(1) X(3) X(5) X(7) X(9) X(11) X(13) X(15) X(17) X(19) X(21) X(23) X(25) X(27) X(29) X(31) \
  X(33) X(35) X(37) X(39) X(41) X(43) X(45) X(47)
#endif

static size_t smem_for(int m) {
  switch (m) {
#define X(MM) case MM: return dia::Geo<MM>::SMEM;
    DIA_FOR_EACH_M(X)
#undef X
  }
  return 0;
}
static void geometry_for(int m, int* rpitch, int* rh) {
  switch (m) {
#define X(MM) case MM: *rpitch = dia::Geo<MM>::RPITCH; *rh = dia::Geo<MM>::RH; return;
    DIA_FOR_EACH_M(X)
#undef X
  }
}
// The kernel instantiations live in one translation unit per m (dia_eval_inst.cu); each exports its kernels and
// the host shadow of its own constant block.
namespace dia {
#define X(MM) const void* eval_kernel_ptr_m##MM(int variant); const void* const_symbol_m##MM(); size_t cluster_smem_m##MM(); \
  size_t hess_tc_smem_m##MM();
DIA_FOR_EACH_M(X)
#undef X
}  // namespace dia

// aux = true: mask / flat field / caller variance map present (read from global memory per pixel);
// diff = true: difference-image instantiation; kc = true: kernel pixels in the constant bank
static const void* kernel_for(int m, bool aux, bool diff = false, bool kc = false) {
  const int variant = diff ? 2 : aux ? (kc ? 5 : 1) : kc ? 3 : 0;
  switch (m) {
#define X(MM) case MM: return dia::eval_kernel_ptr_m##MM(variant);
    DIA_FOR_EACH_M(X)
#undef X
  }
  return nullptr;
}
static const void* hess_kernel_for(int m) {
  switch (m) {
#define X(MM) case MM: return dia::eval_kernel_ptr_m##MM(4);
    DIA_FOR_EACH_M(X)
#undef X
  }
  return nullptr;
}
static const void* cluster_kernel_for(int m) {
  switch (m) {
#define X(MM) case MM: return dia::eval_kernel_ptr_m##MM(6);
    DIA_FOR_EACH_M(X)
#undef X
  }
  return nullptr;
}
static const void* hess_tc_kernel_for(int m) {
  switch (m) {
#define X(MM) case MM: return dia::eval_kernel_ptr_m##MM(7);
    DIA_FOR_EACH_M(X)
#undef X
  }
  return nullptr;
}
static size_t hess_tc_smem_for(int m) {
  switch (m) {
#define X(MM) case MM: return dia::hess_tc_smem_m##MM();
    DIA_FOR_EACH_M(X)
#undef X
  }
  return 0;
}
static size_t cluster_smem_for(int m) {
  switch (m) {
#define X(MM) case MM: return dia::cluster_smem_m##MM();
    DIA_FOR_EACH_M(X)
#undef X
  }
  return 0;
}
static const void* const_symbol_for(int m) {
  switch (m) {
#define X(MM) case MM: return dia::const_symbol_m##MM();
    DIA_FOR_EACH_M(X)
#undef X
  }
  return nullptr;
}

// ---------------------------------------------------------------------------------------------
// TMA tensor maps (driver entry point fetched through the runtime: no link against libcuda)
// ---------------------------------------------------------------------------------------------
typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static encode_tiled_fn get_encode() {
  static encode_tiled_fn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (encode_tiled_fn)ptr;
    else
      cudaGetLastError();
  }
  return fn;
}
// float32 tensor {n_cols, n_rows[, n_img]} with box {box_w, box_h[, 1]}; out-of-bounds elements read as 0
static bool make_tensor_map(CUtensorMap* tm, const float* base, int n_cols, int n_rows, int n_img, int box_w,
                            int box_h) {
  encode_tiled_fn enc = get_encode();
  if (!enc) return false;
  const cuuint32_t rank = n_img > 0 ? 3 : 2;
  cuuint64_t dims[3] = {(cuuint64_t)n_cols, (cuuint64_t)n_rows, (cuuint64_t)(n_img > 0 ? n_img : 1)};
  cuuint64_t strides[2] = {(cuuint64_t)n_cols * 4, (cuuint64_t)n_cols * 4 * (cuuint64_t)n_rows};
  cuuint32_t box[3] = {(cuuint32_t)box_w, (cuuint32_t)box_h, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, rank, (void*)base, dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

static const void* small_kernel_for(int m, int loss = DIA_LOSS_GAUSSIAN) {
  const bool hub = loss == DIA_LOSS_HUBER;
  switch (m) {
    case 1: return hub ? (const void*)dia::eval_small_kernel<1, true> : (const void*)dia::eval_small_kernel<1, false>;
    case 3: return hub ? (const void*)dia::eval_small_kernel<3, true> : (const void*)dia::eval_small_kernel<3, false>;
    case 5: return hub ? (const void*)dia::eval_small_kernel<5, true> : (const void*)dia::eval_small_kernel<5, false>;
    // m = 5: 240 registers, one CTA of eight warps per SM -- 63.3 against the generic kernel's 73.1 us per 4096^2 epoch
    // since the edge fix (12 % slower than the generic kernel before it)
  }
  return nullptr;
}
static size_t small_smem_for(int) { return 0; }   // static shared memory only
static int small_threads_for(int m) { return m == 1 ? dia::SmallGeo<1>::THREADS : (m == 3 ? dia::SmallGeo<3>::THREADS : dia::SmallGeo<5>::THREADS); }
// Geometry of an eval_small_kernel launch (dia_eval_small.cuh): lanes side by side until they span the valid width,
// and the largest number of rows per thread that still leaves three tiles per resident CTA.
namespace dia { int eval_grid(const dia_handle* h, int n_epochs); int eval_part_cols(const dia_handle* h, int n_epochs); }
struct SmallPlan { int rpt, lxlog, tiles, grid; };
static SmallPlan small_plan(const dia_handle* h, int n_epochs) {
  const int vc = h->cfg.n_cols - h->cfg.m + 1, vr = h->cfg.n_rows - h->cfg.m + 1;
  SmallPlan sp;
  sp.lxlog = 0;
  while (sp.lxlog < 5 && (dia::kSmallPx << sp.lxlog) < vc) ++sp.lxlog;
  const int tw = dia::kSmallPx << sp.lxlog, tx = (vc + tw - 1) / tw;
  for (sp.rpt = 16; ; sp.rpt /= 2) {
    const int th = (small_threads_for(h->cfg.m) / 32) * (32 >> sp.lxlog) * sp.rpt;
    sp.tiles = tx * ((vr + th - 1) / th);
    // (a full batch decides, so that every call on this handle cuts the image the same way: batched == singles)
    if (sp.rpt == 2 || (long long)sp.tiles * h->cfg.max_epochs >= 3LL * h->small_grid) break;
  }
  const long long items = (long long)sp.tiles * n_epochs;
  sp.grid = items < h->small_grid ? (int)items : h->small_grid;
  return sp;
}

namespace dia {
const void* eval_kernel_ptr(const dia_handle* h, bool aux) { return kernel_for(h->cfg.m, aux); }
size_t eval_smem_bytes(const dia_handle* h) { return h->smem; }
// the launch that evaluates p: kernel, grid, dynamic shared memory and the number of partial columns per epoch
const void* eval_kernel_ptr_p(const dia_handle* h, const EvalParams& p) {
  return p.small_rpt > 0 ? small_kernel_for(h->cfg.m, h->cfg.loss) : kernel_for(h->cfg.m, eval_is_aux(p));
}
int eval_threads_p(const dia_handle* h, const EvalParams& p) { return p.small_rpt > 0 ? small_threads_for(h->cfg.m) : kThreads; }
size_t eval_smem_bytes_p(const dia_handle* h, const EvalParams& p) { return p.small_rpt > 0 ? small_smem_for(h->cfg.m) : h->smem; }
int eval_grid_p(const dia_handle* h, const EvalParams& p) {
  return p.small_rpt > 0 ? small_plan(h, p.n_epochs).grid : eval_grid(h, p.n_epochs);
}
int eval_part_cols_p(const dia_handle* h, const EvalParams& p) {
  if (p.small_rpt > 0) {
    const SmallPlan sp = small_plan(h, p.n_epochs);
    return sp.tiles < sp.grid ? sp.tiles : sp.grid;
  }
  return eval_part_cols(h, p.n_epochs);
}
// Many small images (at least one epoch per resident CTA): each CTA takes whole epochs, unless that balances the
// CTAs more than 3 % worse than dealing the (epoch, tile) items out one by one.
bool eval_by_epoch(const dia_handle* h, int n_epochs) {
  const long long g = h->grid, items = (long long)n_epochs * h->tiles;
  if (n_epochs < g || h->tiles < 2) return false;
  const long long by_epoch = (n_epochs + g - 1) / g * h->tiles, by_item = (items + g - 1) / g;
  return 100 * by_epoch <= 103 * by_item;
}
int eval_grid(const dia_handle* h, int n_epochs) {
  const long long items = (long long)n_epochs * h->tiles;
  return items < h->grid ? (int)items : h->grid;
}
int eval_part_cols(const dia_handle* h, int n_epochs) {
  if (eval_by_epoch(h, n_epochs)) return 1;
  const int g = eval_grid(h, n_epochs);
  return h->tiles < g ? h->tiles : g;
}
// Constant-bank variant: loss and gradient (plain or with mask / flat / variance map; not the Hessian rows, whose
// "epochs" share one theta), few enough epochs, and enough work per
// launch: refreshing the bank costs ~5.5 us (pack kernel + copy to the symbol) and buys ~9 % of the kernel time,
// which pays from about 60 us on -- two or more tiles per resident CTA at m = 19 (bench.py --sweep).
bool eval_uses_const(const dia_handle* h, const EvalParams& p, bool diff) {
  const int m = h->cfg.m, kp = (m + 3) / 4 * 4;
  const long long items = (long long)p.n_epochs * h->tiles;
  const long long waves = (items + h->grid - 1) / h->grid;
  return h->d_const_stage && !diff && p.small_rpt == 0 && p.hess_q0 < 0 && !eval_by_epoch(h, p.n_epochs) && waves * m * m >= 2 * 19 * 19 &&
         p.n_epochs <= kConstEpochs &&
         (long long)p.n_epochs * m * kp <= kConstK;
}
size_t const_block_bytes(const dia_handle* h, int n_epochs) {
  const int kp = (h->cfg.m + 3) / 4 * 4;
  return offsetof(ConstBlock, K) + sizeof(float) * (size_t)n_epochs * h->cfg.m * kp;
}
const void* eval_kernel_ptr_kc(const dia_handle* h, const EvalParams& p) { return kernel_for(h->cfg.m, eval_is_aux(p), false, true); }
ConstBlock* const_stage(const dia_handle* h) { return h->d_const_stage; }
const void* const_symbol(const dia_handle* h) { return const_symbol_for(h->cfg.m); }
cudaError_t launch_eval(const dia_handle* h, const EvalParams& p, const TensorMaps& tm, bool diff) {
  void* args[] = {(void*)&p, (void*)&tm};
  const bool kc = eval_uses_const(h, p, diff);
  if (kc) {      // refresh the constant block from theta (and the done flags) first, stream-ordered
    // The block is shared by every handle of this kernel size on this stream: the three enqueues (pack, copy, launch)
    // must not interleave with those of another host thread driving such a handle, or the other handle's kernel
    // pixels would be in the bank when this launch runs.  (A dia_fit graph launch is one enqueue and needs no lock.)
    std::lock_guard<std::mutex> lock(g_const_launch_mutex[h->cfg.m]);
    const int kp = (h->cfg.m + 3) / 4 * 4;
    pack_const_kernel<<<1, 256, 0, h->stream>>>(p.theta, p.done, p.n_epochs, p.np, h->cfg.m, kp, h->d_const_stage);
    cudaError_t ce = cudaMemcpyToSymbolAsync(const_symbol_for(h->cfg.m), h->d_const_stage, const_block_bytes(h, p.n_epochs), 0,
                                             cudaMemcpyDeviceToDevice, h->stream);
    if (ce != cudaSuccess) return ce;
    return cudaLaunchKernel(kernel_for(h->cfg.m, eval_is_aux(p), false, true), dim3(eval_grid(h, p.n_epochs)), dim3(kThreads), args,
                            h->smem, h->stream);
  }
  if (p.small_rpt > 0 && !diff) {
    void* sargs[] = {(void*)&p};
    return cudaLaunchKernel(small_kernel_for(h->cfg.m, h->cfg.loss), dim3(eval_grid_p(h, p)), dim3(small_threads_for(h->cfg.m)), sargs,
                            small_smem_for(h->cfg.m), h->stream);
  }
  return cudaLaunchKernel(kernel_for(h->cfg.m, eval_is_aux(p), diff, kc), dim3(eval_grid(h, p.n_epochs)), dim3(kThreads), args,
                          h->smem, h->stream);
}
}  // namespace dia

// lambda * N_data of Eq. 20 (N_data = valid-region pixels)
static double lambda_n(const dia_handle* h) {
  const dia_config& c = h->cfg;
  return (double)c.lambda_reg * (double)(c.n_rows - c.m + 1) * (double)(c.n_cols - c.m + 1);
}

static void fill_params(const dia_handle* h, int n_epochs, const float* d_I, const unsigned char* d_mask,
                        const float* d_var, const float* d_theta, const int* d_done, dia::EvalParams* p,
                        dia::TensorMaps* tm, int hess_q0 = -1) {
  const dia_config& c = h->cfg;
  p->R = h->d_R;  p->I = d_I;  p->mask = d_mask;  p->var = d_var;  p->flat = c.d_flat;
  p->theta = d_theta;  p->done = d_done;  p->partials = h->d_partials;
  p->n_rows = c.n_rows;  p->n_cols = c.n_cols;  p->n_epochs = n_epochs;  p->n_refs = h->n_refs;
  p->hess_q0 = hess_q0;
  p->np = h->np;  p->part_rows = h->np + 1;  p->diff = nullptr;  p->bg_degree = c.bg_degree;
  // Eq. 19: centre ((N-1)/2), normalisation N (R18)
  p->bg_xc = 0.5f * (float)(c.n_cols - 1);  p->bg_yc = 0.5f * (float)(c.n_rows - 1);
  p->bg_inv_nx = 1.0f / (float)c.n_cols;  p->bg_inv_ny = 1.0f / (float)c.n_rows;
  p->tiles_x = (c.n_cols - c.m + 1 + dia::kTW - 1) / dia::kTW;
  p->tiles_y = (c.n_rows - c.m + 1 + dia::kTH - 1) / dia::kTH;
  p->loss_kind = c.loss;  p->noise_kind = c.noise;
  p->huber_c = c.huber_c;  p->sigma0_sq = c.sigma0 * c.sigma0;
  p->inv_gain = c.noise == DIA_NOISE_MODEL ? 1.0f / c.gain : 0.f;
  p->use_tma = 0;
  p->flush_tiles = h->flush_tiles;
  p->epoch_per_cta = dia::eval_by_epoch(h, n_epochs) ? 1 : 0;
  // plain objective with a small kernel: the register-resident kernel of dia_eval_small.cuh
  p->small_rpt = 0;  p->small_lxlog = 0;  p->small_vec = 0;
  if (h->small_grid > 0 && !d_mask && !d_var && hess_q0 < 0) {
    const SmallPlan sp = small_plan(h, n_epochs);
    p->small_rpt = sp.rpt;  p->small_lxlog = sp.lxlog;  p->epoch_per_cta = 0;
    p->small_vec = (c.n_cols % 4 == 0 && aligned16(h->d_R) && aligned16(d_I)) ? 1 : 0;
  }
  p->cp8 = (c.n_cols % 2 == 0) && (reinterpret_cast<uintptr_t>(h->d_R) & 7) == 0 && (reinterpret_cast<uintptr_t>(d_I) & 7) == 0;
  std::memset(tm, 0, sizeof(*tm));
  if (h->use_tma && aligned16(d_I) &&
      make_tensor_map(&tm->I, d_I, c.n_cols, c.n_rows, hess_q0 >= 0 ? 1 : n_epochs, dia::kIPitch, dia::kTH)) {
    tm->R = h->tmR;
    p->use_tma = 1;
  }
}

extern "C" int dia_create(const dia_config* cfg, const float* d_R, dia_handle** out) {
  if (!cfg || !d_R || !out) return fail(nullptr, DIA_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  if (cfg->m < 1 || cfg->m % 2 == 0) return fail(nullptr, DIA_ERR_INVALID_ARG, "m must be odd and >= 1");
  if (cfg->n_rows < cfg->m || cfg->n_cols < cfg->m) return fail(nullptr, DIA_ERR_INVALID_ARG, "image smaller than kernel");
  if (cfg->max_epochs < 1) return fail(nullptr, DIA_ERR_INVALID_ARG, "max_epochs must be >= 1");
  if (!(cfg->lambda_reg >= 0.f)) return fail(nullptr, DIA_ERR_INVALID_ARG, "lambda_reg must be >= 0");
  if (cfg->bg_degree < 0) return fail(nullptr, DIA_ERR_INVALID_ARG, "bg_degree must be >= 0");
  if (cfg->bg_degree > DIA_MAX_BG_DEGREE) return fail(nullptr, DIA_ERR_UNSUPPORTED, "bg_degree exceeds DIA_MAX_BG_DEGREE");
  if (cfg->n_refs > 1 && cfg->n_refs != cfg->max_epochs)
    return fail(nullptr, DIA_ERR_INVALID_ARG, "n_refs must be 0, 1 or max_epochs");
  if (cfg->loss != DIA_LOSS_GAUSSIAN && cfg->loss != DIA_LOSS_HUBER) return fail(nullptr, DIA_ERR_INVALID_ARG, "bad loss");
  if (cfg->noise != DIA_NOISE_MODEL && cfg->noise != DIA_NOISE_FIXED) return fail(nullptr, DIA_ERR_INVALID_ARG, "bad noise mode");
  if (cfg->loss == DIA_LOSS_HUBER && !(cfg->huber_c > 0.f)) return fail(nullptr, DIA_ERR_INVALID_ARG, "huber_c must be > 0");
  if (cfg->noise == DIA_NOISE_MODEL && !(cfg->gain > 0.f && cfg->sigma0 >= 0.f))
    return fail(nullptr, DIA_ERR_INVALID_ARG, "need gain > 0 and sigma0 >= 0");
  if (cfg->m > DIA_MAX_KERNEL_SIZE) return fail(nullptr, DIA_ERR_UNSUPPORTED, "m exceeds DIA_MAX_KERNEL_SIZE");

  int dev = 0, sms = 0;
  cudaError_t ce = cudaGetDevice(&dev);
  if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaGetDevice (no CUDA device: there is no CPU fallback)");
  ce = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaDeviceGetAttribute");

  dia_handle* h = new (std::nothrow) dia_handle();
  if (!h) return fail(nullptr, DIA_ERR_ALLOC, "host allocation failed");
  h->n_refs = cfg->n_refs > 1 ? cfg->n_refs : 1;
  h->cfg = *cfg;  h->d_R = d_R;  h->stream = (cudaStream_t)cfg->stream;  h->sms = sms;
  h->np = cfg->m * cfg->m + (cfg->bg_degree + 1) * (cfg->bg_degree + 2) / 2;  h->smem = smem_for(cfg->m);  h->d_partials = nullptr;
  h->d_const_stage = nullptr;

  int occ = 0;
  for (int aux = 0; aux < 5; ++aux) {        // evaluation (plain, generic), difference image, constant-bank variants
    const void* k = kernel_for(cfg->m, aux == 1 || aux == 2 || aux == 4, aux == 2, aux >= 3);
    ce = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem);
    if (ce != cudaSuccess) { int rc = cuda_fail(nullptr, ce, "cudaFuncSetAttribute(smem)"); delete h; return rc; }
    int o = 0;
    ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, k, dia::kThreads, h->smem);
    if (ce != cudaSuccess) { int rc = cuda_fail(nullptr, ce, "occupancy query"); delete h; return rc; }
    if (o < 1) { int rc = fail(nullptr, DIA_ERR_UNSUPPORTED, "the evaluation kernel of this kernel size does not fit on an SM of this device"); delete h; return rc; }
    occ = (aux == 0 || o < occ) ? o : occ;   // one grid size for all variants
  }
  h->use_tma = 0;
  const char* no_tma = std::getenv("DIA_DISABLE_TMA");   // test hook: force the cp.async staging path
  if (cfg->n_cols % 4 == 0 && aligned16(d_R) && !(no_tma && no_tma[0] == '1')) {
    int rpitch = 0, rh = 0;
    geometry_for(cfg->m, &rpitch, &rh);
    h->use_tma = make_tensor_map(&h->tmR, d_R, cfg->n_cols, cfg->n_rows, h->n_refs, rpitch, rh) ? 1 : 0;
  }
  const int tiles = ((cfg->n_cols - cfg->m + 1 + dia::kTW - 1) / dia::kTW) * ((cfg->n_rows - cfg->m + 1 + dia::kTH - 1) / dia::kTH);
  h->tiles = tiles;
  h->grid = sms * occ;                       // persistent grid: every CTA resident
  if ((long long)h->grid > (long long)tiles * cfg->max_epochs) h->grid = tiles * cfg->max_epochs;
  h->grid_limit = 0;
  if (const char* lim = std::getenv("DIA_GRID_LIMIT")) {   // test hook: few CTAs => many tiles per CTA
    const int g = std::atoi(lim);
    if (g >= 1) h->grid_limit = g;
    if (g >= 1 && g < h->grid) h->grid = g;
  }
  h->cluster_fit = -1;
  if (const char* nc = std::getenv("DIA_DISABLE_CLUSTER")) { if (nc[0] == '1') h->cluster_fit = 0; }   // test hook: graph loop
  h->flush_tiles = dia::kFlushTiles;
  if (const char* ft = std::getenv("DIA_FLUSH_TILES")) {   // test hook: how often the FP32 strips are folded
    const int f = std::atoi(ft);
    if (f >= 1) h->flush_tiles = f;
  }
  // m <= 5, no flat field, no background polynomial: eval_small_kernel evaluates the plain objective
  h->small_grid = 0;
  const char* no_small = std::getenv("DIA_DISABLE_SMALL");   // test hook: force the generic kernel
  if (small_kernel_for(cfg->m) && !cfg->d_flat && cfg->bg_degree == 0 && cfg->noise == DIA_NOISE_MODEL &&
      !(no_small && no_small[0] == '1')) {
    int o = 0;
    const void* ks = small_kernel_for(cfg->m, cfg->loss);
    if (cudaFuncSetAttribute(ks, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)small_smem_for(cfg->m)) == cudaSuccess &&
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, ks, small_threads_for(cfg->m), small_smem_for(cfg->m)) == cudaSuccess && o >= 1) {
      h->small_grid = sms * o;
      if (h->grid_limit > 0 && h->grid_limit < h->small_grid) h->small_grid = h->grid_limit;
    } else {
      cudaGetLastError();
    }
  }
  size_t part_cols = (size_t)(tiles < h->grid ? tiles : h->grid);
  if ((size_t)h->small_grid > part_cols) part_cols = (size_t)h->small_grid;
  ce = cudaMalloc(&h->d_partials, sizeof(double) * (size_t)cfg->max_epochs * part_cols * (h->np + 1));
  if (ce != cudaSuccess) { int rc = fail(nullptr, DIA_ERR_ALLOC, "workspace allocation failed"); cudaGetLastError(); delete h; return rc; }
  const char* no_const = std::getenv("DIA_DISABLE_CONST");   // test hook: force the shared-memory variant
  // a full batch would be a long enough launch (eval_uses_const): try to claim the constant block of this kernel size
  const long long full_waves = ((long long)tiles * cfg->max_epochs + h->grid - 1) / h->grid;
  if (full_waves * cfg->m * cfg->m >= 2 * 19 * 19 && !(no_const && no_const[0] == '1')) {
    int device = -1;
    cudaGetDevice(&device);
    if (const_slot_acquire(cfg->m, cfg->stream, device)) {
      if (cudaMalloc(&h->d_const_stage, sizeof(dia::ConstBlock)) != cudaSuccess) {
        cudaGetLastError();  h->d_const_stage = nullptr;  const_slot_release(cfg->m);
      }
    }
  }
  int rc = dia::fit_workspace_create(&h->fit, cfg->max_epochs, h->np);
  if (rc != DIA_OK) {
    cudaFree(h->d_partials);
    if (h->d_const_stage) { cudaFree(h->d_const_stage); const_slot_release(cfg->m); }
    fail(nullptr, rc, "fit workspace allocation failed");
    delete h;
    return rc;
  }
  *out = h;
  return DIA_OK;
}

static void host_path_destroy(dia_handle* h) {
  dia_handle::HostPath& hp = h->host;
  cudaFree(hp.dI); cudaFree(hp.dth); cudaFree(hp.dmask); cudaFree(hp.dres); cudaFree(hp.dloss); cudaFree(hp.dgrad);
  for (cudaEvent_t& e : hp.ready) if (e) cudaEventDestroy(e);
  if (hp.free_ev) cudaEventDestroy(hp.free_ev);
  if (hp.copy_stream) cudaStreamDestroy(hp.copy_stream);
  hp = dia_handle::HostPath();
}

extern "C" int dia_destroy(dia_handle* h) {
  if (!h) return DIA_ERR_INVALID_ARG;
  cudaStreamSynchronize(h->stream);
  dia::fit_workspace_destroy(&h->fit);
  dia::hess_workspace_destroy(&h->hess);
  cudaFree(h->d_partials);
  if (h->d_const_stage) {
    cudaFree(h->d_const_stage);
    const_slot_release(h->cfg.m);
  }
  host_path_destroy(h);
  delete h;
  return DIA_OK;
}

static int check_eval_args(dia_handle* h, int n_epochs, const void* d_I, const void* d_var, const void* d_theta) {
  if (!h) return DIA_ERR_INVALID_ARG;
  if (n_epochs < 1 || n_epochs > h->cfg.max_epochs) return fail(h, DIA_ERR_INVALID_ARG, "n_epochs out of range");
  if (!d_I || !d_theta) return fail(h, DIA_ERR_INVALID_ARG, "null image or theta");
  if (h->cfg.noise == DIA_NOISE_FIXED && !d_var) return fail(h, DIA_ERR_INVALID_ARG, "DIA_NOISE_FIXED needs d_var");
  if (h->cfg.noise == DIA_NOISE_MODEL && d_var) return fail(h, DIA_ERR_INVALID_ARG, "d_var must be NULL in DIA_NOISE_MODEL");
  return DIA_OK;
}

// loss and gradient of n_epochs parameter sets; hess_q0 >= 0: rows hess_q0.. of the Hessian of target 0 instead
static int eval_into(dia_handle* h, int n_epochs, const float* d_I, const unsigned char* d_mask, const float* d_var,
                     const float* d_theta, double* d_loss, double* d_grad, int hess_q0) {
  dia::EvalParams p;
  dia::TensorMaps tm;
  fill_params(h, n_epochs, d_I, d_mask, d_var, d_theta, nullptr, &p, &tm, hess_q0);
  cudaError_t ce = dia::launch_eval(h, p, tm);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "eval launch");
  const int np1 = h->np + 1;
  dia::reduce_partials_kernel<<<dim3((np1 + 7) / 8, n_epochs), 256, 0, h->stream>>>(
      h->d_partials, dia::eval_part_cols_p(h, p), np1, nullptr, d_loss, d_grad);
  if (h->cfg.lambda_reg > 0.f && hess_q0 < 0)
    dia::penalty_kernel<<<n_epochs, dia::kFitThreads, 0, h->stream>>>(d_theta, h->cfg.m, h->np, lambda_n(h), d_loss, d_grad);
  ce = cudaGetLastError();
  if (ce != cudaSuccess) return cuda_fail(h, ce, "reduce launch");
  return DIA_OK;
}

extern "C" int dia_eval_loss_grad(dia_handle* h, int n_epochs, const float* d_I, const unsigned char* d_mask,
                                  const float* d_var, const float* d_theta, double* d_loss, double* d_grad) {
  int rc = check_eval_args(h, n_epochs, d_I, d_var, d_theta);
  if (rc != DIA_OK) return rc;
  if (!d_loss || !d_grad) return fail(h, DIA_ERR_INVALID_ARG, "null output");
  return eval_into(h, n_epochs, d_I, d_mask, d_var, d_theta, d_loss, d_grad, -1);
}

extern "C" int dia_hessian(dia_handle* h, const float* d_I, const unsigned char* d_mask, const float* d_var,
                           const float* d_theta, double* d_H) {
  int rc = check_eval_args(h, 1, d_I, d_var, d_theta);
  if (rc != DIA_OK) return rc;
  if (!d_H) return fail(h, DIA_ERR_INVALID_ARG, "null output");
  if (h->n_refs > 1) return fail(h, DIA_ERR_UNSUPPORTED, "dia_hessian needs a handle with one shared reference");
  const int np = h->np;
  dia::HessWorkspace& w = h->hess;
  if (!w.loss) {
    cudaError_t ce = cudaFuncSetAttribute(hess_kernel_for(h->cfg.m), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem);
    if (ce == cudaSuccess) ce = cudaMalloc(&w.loss, sizeof(double) * (size_t)np);
    if (ce == cudaSuccess)
      ce = cudaMalloc(&w.partials, sizeof(double) * (size_t)dia::kHessRows * (np + 1) * (h->grid < h->tiles ? h->grid : h->tiles));
    if (ce == cudaSuccess && h->cfg.lambda_reg > 0.f) {
      ce = cudaMalloc(&w.ident, sizeof(float) * (size_t)np * np);
      if (ce == cudaSuccess) dia::hess_identity_kernel<<<(np * np + 255) / 256, 256, 0, h->stream>>>(w.ident, np);
    }
    if (ce != cudaSuccess) {
      dia::hess_workspace_destroy(&w);
      h->err = std::string("hessian workspace: ") + cudaGetErrorString(ce);
      return DIA_ERR_ALLOC;
    }
  }
  // Kernel-pixel rows (q < m^2), kHessRows rows per launch: hess_block_kernel computes h once per tile and then one
  // gradient pass per row; it delivers the kernel-kernel block, the remaining entries of these rows
  // come from the background rows below by symmetry.
  const int nk = h->cfg.m * h->cfg.m;
  // m >= 5: all of H is one split-float16 tensor-core contraction (hess_tc_kernel); test hook
  // DIA_HESS_TC=0 keeps the CUDA-core row passes below
  const char* tc_env = std::getenv("DIA_HESS_TC");
  const void* ktc = (h->cfg.m >= 5 && !(tc_env && tc_env[0] == '0')) ? hess_tc_kernel_for(h->cfg.m) : nullptr;
  dia::HessTcTypes tct;
  if (ktc && dia::hess_tc_make_types(np, &tct) == 0) ktc = nullptr;
  if (ktc) {
    int per_type = h->sms / tct.n_types;
    if (h->grid_limit > 0 && h->grid_limit / tct.n_types < per_type) per_type = h->grid_limit / tct.n_types;   // test hook: many tiles per CTA
    tct.ctas_per_type = per_type < 1 ? 1 : (per_type > h->tiles ? h->tiles : per_type);
    const int tgrid = tct.n_types * tct.ctas_per_type;
    if (!w.tc_partials || w.tc_grid < tgrid) {
      cudaFree(w.tc_partials);  w.tc_partials = nullptr;  w.tc_grid = 0;
      cudaError_t ce = cudaFuncSetAttribute(ktc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)hess_tc_smem_for(h->cfg.m));
      if (ce == cudaSuccess) ce = cudaMalloc(&w.tc_partials, sizeof(double) * (size_t)tgrid * dia::kTcRows * dia::kTcGroup);
      if (ce != cudaSuccess) { cudaGetLastError(); return fail(h, DIA_ERR_ALLOC, std::string("hessian tensor-core workspace: ") + cudaGetErrorString(ce)); }
      w.tc_grid = tgrid;
    }
    if (!w.tc_perm) {                        // slot -> parameter table (depends on m and the background degree only)
      const int slots = (np + dia::kTcGroup - 1) / dia::kTcGroup * dia::kTcGroup;
      int rpitch = 0, rh = 0;
      geometry_for(h->cfg.m, &rpitch, &rh);
      std::vector<short> perm((size_t)slots);
      dia::hess_tc_make_perm(h->cfg.m, np, rpitch, perm.data());
      cudaError_t ce = cudaMalloc(&w.tc_perm, sizeof(short) * (size_t)slots);
      if (ce == cudaSuccess) ce = cudaMemcpy(w.tc_perm, perm.data(), sizeof(short) * (size_t)slots, cudaMemcpyHostToDevice);
      if (ce != cudaSuccess) { cudaGetLastError(); cudaFree(w.tc_perm); w.tc_perm = nullptr; return fail(h, DIA_ERR_ALLOC, "hessian slot table"); }
    }
    dia::EvalParams p;
    dia::TensorMaps tm;
    fill_params(h, 1, d_I, d_mask, d_var, d_theta, nullptr, &p, &tm, 0);
    void* args[] = {(void*)&p, (void*)&w.tc_partials, (void*)&w.tc_perm, (void*)&tct};
    cudaError_t ce = cudaLaunchKernel(ktc, dim3(tgrid), dim3(dia::kThreads), args, hess_tc_smem_for(h->cfg.m), h->stream);
    if (ce != cudaSuccess) return cuda_fail(h, ce, "hessian tensor-core launch");
    dia::hess_tc_reduce_kernel<<<dim3((dia::kTcRows * dia::kTcGroup + 255) / 256, tct.n_types), 256, 0, h->stream>>>(
        w.tc_partials, w.tc_perm, tct, np, d_H);
  }
  const void* kblock = hess_kernel_for(h->cfg.m);
  const int bgrid = h->grid < h->tiles ? h->grid : h->tiles;
  for (int q0 = 0; q0 < (ktc ? 0 : nk); q0 += dia::kHessRows) {
    const int n = nk - q0 < dia::kHessRows ? nk - q0 : dia::kHessRows;
    dia::EvalParams p;
    dia::TensorMaps tm;
    fill_params(h, 1, d_I, d_mask, d_var, d_theta, nullptr, &p, &tm, q0);
    p.n_epochs = n;  p.partials = w.partials;      // rows of this launch, the Hessian's own partial columns
    void* args[] = {(void*)&p};
    cudaError_t ce = cudaLaunchKernel(kblock, dim3(bgrid), dim3(dia::kThreads), args, h->smem, h->stream);
    if (ce != cudaSuccess) return cuda_fail(h, ce, "hessian block launch");
    const int np1 = np + 1, warps = 8;
    dia::reduce_partials_kernel<<<dim3((np1 + warps - 1) / warps, n), warps * 32, 0, h->stream>>>(
        w.partials, bgrid, np1, nullptr, w.loss + q0, d_H + (size_t)q0 * np);
  }
  // Background rows (B0 and the polynomial terms): the fused kernel with the weight h X_q in place of w (D3)
  for (int q0 = nk; q0 < (ktc ? 0 : np); q0 += h->cfg.max_epochs) {
    const int n = np - q0 < h->cfg.max_epochs ? np - q0 : h->cfg.max_epochs;
    rc = eval_into(h, n, d_I, d_mask, d_var, d_theta, w.loss + q0, d_H + (size_t)q0 * np, q0);
    if (rc != DIA_OK) return rc;
  }
  if (!ktc) dia::hess_fill_columns_kernel<<<(nk * (np - nk) + 255) / 256, 256, 0, h->stream>>>(d_H, np, nk);
  // Eq. 20: the penalty lambda N |L theta|^2 adds 2 lambda N L'L; its gradient is linear in theta, so the
  // gradient at the unit vector e_q is row q
  if (h->cfg.lambda_reg > 0.f)
    dia::penalty_kernel<<<np, dia::kFitThreads, 0, h->stream>>>(w.ident, h->cfg.m, np, lambda_n(h), w.loss, d_H);
  dia::hess_symmetrise_kernel<<<(np * np + 255) / 256, 256, 0, h->stream>>>(d_H, np);
  cudaError_t ce = cudaGetLastError();
  if (ce != cudaSuccess) return cuda_fail(h, ce, "hessian launch");
  return DIA_OK;
}

extern "C" int dia_covariance(dia_handle* h, const double* d_H, double* d_cov, double* d_sigma, double* d_info) {
  if (!h) return DIA_ERR_INVALID_ARG;
  if (!d_H || !d_sigma || !d_info) return fail(h, DIA_ERR_INVALID_ARG, "null Hessian, sigma or info");
  if (d_cov == d_H) return fail(h, DIA_ERR_INVALID_ARG, "d_cov must not alias d_H");
  const int np = h->np;
  dia::HessWorkspace& w = h->hess;
  if (!w.chol) {
    cudaError_t ce = cudaMalloc(&w.chol, sizeof(double) * ((size_t)np * np + dia::kCholPanel * dia::kCholPanel));   // + the panel's diagonal block

    if (ce != cudaSuccess) {
      cudaFree(w.chol);  w.chol = nullptr;
      h->err = std::string("covariance workspace: ") + cudaGetErrorString(ce);
      return DIA_ERR_ALLOC;
    }
  }
  dia::cov_init_kernel<<<1, 1, 0, h->stream>>>(d_info);
  for (int j0 = 0; j0 < np; j0 += dia::kCholPanel) {          // blocked left-looking Cholesky: two launches per panel
    const int nb = np - j0 < dia::kCholPanel ? np - j0 : dia::kCholPanel;
    dia::chol_panel_update_kernel<<<(np - j0 + dia::kCholWarps - 1) / dia::kCholWarps, dia::kCholWarps * 32, 0, h->stream>>>(
        d_H, w.chol, w.chol + (size_t)np * np, np, j0, nb);
    const int below = np - j0 - nb;
    dia::chol_panel_factor_kernel<<<below > 0 ? (below + dia::kCholWarps - 1) / dia::kCholWarps : 1, dia::kCholWarps * 32, 0,
                                    h->stream>>>(w.chol, w.chol + (size_t)np * np, np, j0, nb, d_info);
  }
  {
    const double* Wc = w.chol;
    int np_ = np, nk_ = h->cfg.m * h->cfg.m;
    void* sargs[] = {(void*)&Wc, (void*)&np_, (void*)&nk_, (void*)&d_cov, (void*)&d_sigma, (void*)&d_info};
    size_t ssmem = 0;
    const void* ksolve = dia::cov_solve_kernel_for(np, &ssmem);
    cudaError_t ce = cudaFuncSetAttribute(ksolve, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssmem);
    if (ce == cudaSuccess)
      ce = cudaLaunchKernel(ksolve, dim3((np + 1 + dia::kSolveWarps - 1) / dia::kSolveWarps), dim3(dia::kSolveWarps * 32), sargs, ssmem,
                            h->stream);
    if (ce != cudaSuccess) return cuda_fail(h, ce, "covariance solve launch");
  }
  if (d_cov) dia::hess_symmetrise_kernel<<<(np * np + 255) / 256, 256, 0, h->stream>>>(d_cov, np);
  cudaError_t ce = cudaGetLastError();
  if (ce != cudaSuccess) return cuda_fail(h, ce, "covariance launch");
  return DIA_OK;
}

extern "C" int dia_difference_image(dia_handle* h, int n_epochs, const float* d_I, const unsigned char* d_mask,
                                    const float* d_var, const float* d_theta, float* d_D, double* d_metrics) {
  int rc = check_eval_args(h, n_epochs, d_I, d_var, d_theta);
  if (rc != DIA_OK) return rc;
  if (!d_D || !d_metrics) return fail(h, DIA_ERR_INVALID_ARG, "null output");
  const size_t npix = (size_t)h->cfg.n_rows * h->cfg.n_cols;
  cudaError_t ce = cudaMemsetAsync(d_D, 0, sizeof(float) * npix * n_epochs, h->stream);   // pixels outside V read 0
  if (ce != cudaSuccess) return cuda_fail(h, ce, "memset");
  dia::EvalParams p;
  dia::TensorMaps tm;
  fill_params(h, n_epochs, d_I, d_mask, d_var, d_theta, nullptr, &p, &tm);
  p.part_rows = 3;
  p.diff = d_D;
  if (p.small_rpt > 0) { p.small_rpt = 0;  p.epoch_per_cta = dia::eval_by_epoch(h, n_epochs) ? 1 : 0; }   // generic kernel
  ce = dia::launch_eval(h, p, tm, true);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "difference-image launch");
  dia::diff_metrics_kernel<<<n_epochs, 32, 0, h->stream>>>(h->d_partials, dia::eval_part_cols(h, n_epochs), d_metrics);
  ce = cudaGetLastError();
  if (ce != cudaSuccess) return cuda_fail(h, ce, "metrics launch");
  return DIA_OK;
}

extern "C" int dia_fit(dia_handle* h, const dia_fit_opts* opts, int n_epochs, const float* d_I,
                       const unsigned char* d_mask, const float* d_var, float* d_theta,
                       dia_fit_result* d_result) {
  int rc = check_eval_args(h, n_epochs, d_I, d_var, d_theta);
  if (rc != DIA_OK) return rc;
  if (!opts || !d_result) return fail(h, DIA_ERR_INVALID_ARG, "null opts or result");
  if (opts->lbfgs_history < 1 || opts->lbfgs_history > dia::kMaxHistory)
    return fail(h, DIA_ERR_INVALID_ARG, "lbfgs_history out of range");
  dia::EvalParams p;
  dia::TensorMaps tm;
  fill_params(h, n_epochs, d_I, d_mask, d_var, h->fit.d_theta32, h->fit.d_done, &p, &tm);
  // Small image pairs, plain objective: the whole fit inside one kernel, one cluster of `tiles` CTAs per epoch
  // (dia_fit_cluster.cuh).  Chosen when every cluster is resident at once, or for free-running fits of larger
  // batches: there each cluster leaves when its own fit has stopped and the next pair starts (measured, 296 stamps
  // of 142^2, m = 19: 2.7 s against 4.0 s for the graph loop, which iterates until the slowest pair is done), while
  // in lock-step -- every pair takes the same number of steps -- the graph loop's batched evaluations are faster
  // (19 ms against 29 ms for 121 iterations).  A single 128^2 pair: 8.5 us per Adam iteration against 12.1 us.
  // Otherwise the graph loop below.
  const bool lockstep = opts->force_adam_iters >= 0 || opts->force_lbfgs_iters >= 0;
  if (h->cluster_fit != 0 && h->tiles <= dia::kMaxClusterTiles && !dia::eval_is_aux(p) && h->cfg.bg_degree == 0 &&
      (!lockstep || (long long)n_epochs * h->tiles <= (long long)h->sms * 2)) {
    const void* kf = cluster_kernel_for(h->cfg.m);
    const size_t smem = cluster_smem_for(h->cfg.m);
    if (h->cluster_fit < 0) {
      int o = 0;
      cudaError_t ce = cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (ce == cudaSuccess) ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kf, dia::kThreads, smem);
      h->cluster_fit = (ce == cudaSuccess && o >= 1) ? 1 : 0;
      if (ce != cudaSuccess) cudaGetLastError();
    }
    if (h->cluster_fit == 1) {
      dia::fit_init_kernel<<<n_epochs, 256, 0, h->stream>>>(h->fit.b, d_theta, h->np, n_epochs);
      dia::StepArgs sa;
      sa.b = h->fit.b;  sa.partials = h->d_partials;  sa.n_blocks = h->tiles;  sa.np = h->np;  sa.hist_cap = h->fit.hist_cap;
      sa.o = *opts;  sa.theta_out = d_theta;  sa.result = d_result;  sa.cond = 0;  sa.m = h->cfg.m;  sa.lamN = lambda_n(h);
      sa.use_graph = 0;
      p.epoch_per_cta = 0;  p.small_rpt = 0;
      cudaLaunchConfig_t lc = {};
      lc.gridDim = dim3((unsigned)(n_epochs * h->tiles));  lc.blockDim = dim3(dia::kThreads);
      lc.dynamicSmemBytes = smem;  lc.stream = h->stream;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = (unsigned)h->tiles;  at[0].val.clusterDim.y = 1;  at[0].val.clusterDim.z = 1;
      lc.attrs = at;  lc.numAttrs = 1;
      void* args[] = {(void*)&p, (void*)&tm, (void*)&sa};
      cudaError_t ce = cudaLaunchKernelExC(&lc, kf, args);
      if (ce != cudaSuccess) return cuda_fail(h, ce, "cluster fit launch");
      return DIA_OK;
    }
  }
  std::string err;
  const int unroll = 4;        // (eval ; step) pairs per WHILE iteration: 8 % faster on 128^2 images than 1
  rc = dia::fit_run(&h->fit, h, p, tm, *opts, n_epochs, d_theta, d_result, dia::eval_grid_p(h, p),
                    dia::eval_part_cols_p(h, p), unroll, h->cfg.m, lambda_n(h), h->stream, &err);
  if (rc != DIA_OK) return fail(h, rc, err);
  return DIA_OK;
}

extern "C" int dia_measure_fp32_peak(void* stream, double* fma_per_second) {
  if (!fma_per_second) return DIA_ERR_INVALID_ARG;
  const double v = dia::measure_fp32_peak((cudaStream_t)stream, 5);
  if (v <= 0.0) { cudaGetLastError(); return fail(nullptr, DIA_ERR_CUDA, "FP32 peak probe failed (no CUDA device?)"); }
  *fma_per_second = v;
  return DIA_OK;
}

extern "C" int dia_measure_fp32_pattern(void* stream, int pattern, double* fma_per_second) {
  if (!fma_per_second || pattern < 0 || pattern >= dia::kProbePatterns) return DIA_ERR_INVALID_ARG;
  const double v = dia::measure_fp32_pattern((cudaStream_t)stream, pattern, 5);
  if (v <= 0.0) { cudaGetLastError(); return fail(nullptr, DIA_ERR_CUDA, "FP32 probe failed (no CUDA device?)"); }
  *fma_per_second = v;
  return DIA_OK;
}

// ---------------------------------------------------------------------------------------------
// host-buffer entry points (include/dia.h): copies on a second stream, the device calls above in between
// ---------------------------------------------------------------------------------------------
static int host_path_prepare(dia_handle* h, bool want_mask) {
  dia_handle::HostPath& hp = h->host;
  const size_t E = (size_t)h->cfg.max_epochs, npix = (size_t)h->cfg.n_rows * h->cfg.n_cols, np = (size_t)h->np;
  cudaError_t ce = cudaSuccess;
  if (!hp.dI) {
    ce = cudaMalloc(&hp.dI, sizeof(float) * E * npix);
    if (ce == cudaSuccess) ce = cudaMalloc(&hp.dth, sizeof(float) * E * np);
    if (ce == cudaSuccess) ce = cudaMalloc(&hp.dres, sizeof(dia_fit_result) * E);
    if (ce == cudaSuccess) ce = cudaMalloc(&hp.dloss, sizeof(double) * E);
    if (ce == cudaSuccess) ce = cudaMalloc(&hp.dgrad, sizeof(double) * E * np);
    if (ce == cudaSuccess) ce = cudaStreamCreateWithFlags(&hp.copy_stream, cudaStreamNonBlocking);
    for (cudaEvent_t& e : hp.ready) if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
    if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&hp.free_ev, cudaEventDisableTiming);
  }
  if (ce == cudaSuccess && want_mask && !hp.dmask) ce = cudaMalloc(&hp.dmask, E * npix);
  if (ce != cudaSuccess) {
    cudaGetLastError();
    host_path_destroy(h);
    return fail(h, DIA_ERR_ALLOC, std::string("host-path staging buffers: ") + cudaGetErrorString(ce));
  }
  return DIA_OK;
}

extern "C" int dia_eval_loss_grad_host(dia_handle* h, int n_epochs, const float* h_I, const float* h_theta, double* h_loss,
                                       double* h_grad) {
  if (!h) return DIA_ERR_INVALID_ARG;
  if (n_epochs < 1 || n_epochs > h->cfg.max_epochs) return fail(h, DIA_ERR_INVALID_ARG, "n_epochs out of range");
  if (!h_I || !h_theta || !h_loss || !h_grad) return fail(h, DIA_ERR_INVALID_ARG, "null host buffer");
  if (h->cfg.noise == DIA_NOISE_FIXED) return fail(h, DIA_ERR_UNSUPPORTED, "the host-buffer calls take no variance map");
  int rc = host_path_prepare(h, false);
  if (rc != DIA_OK) return rc;
  dia_handle::HostPath& hp = h->host;
  const size_t npix = (size_t)h->cfg.n_rows * h->cfg.n_cols, np = (size_t)h->np, E = (size_t)n_epochs;
  cudaError_t ce = cudaMemcpyAsync(hp.dI, h_I, sizeof(float) * E * npix, cudaMemcpyHostToDevice, h->stream);
  if (ce == cudaSuccess) ce = cudaMemcpyAsync(hp.dth, h_theta, sizeof(float) * E * np, cudaMemcpyHostToDevice, h->stream);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "host to device copy");
  rc = dia_eval_loss_grad(h, n_epochs, hp.dI, nullptr, nullptr, hp.dth, hp.dloss, hp.dgrad);
  if (rc != DIA_OK) return rc;
  ce = cudaMemcpyAsync(h_loss, hp.dloss, sizeof(double) * E, cudaMemcpyDeviceToHost, h->stream);
  if (ce == cudaSuccess) ce = cudaMemcpyAsync(h_grad, hp.dgrad, sizeof(double) * E * np, cudaMemcpyDeviceToHost, h->stream);
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(h->stream);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "device to host copy");
  return DIA_OK;
}

extern "C" int dia_fit_host(dia_handle* h, const dia_fit_opts* opts, int n_epochs, const float* h_I,
                            const unsigned char* h_mask, float* h_theta, dia_fit_result* h_result, int chunks) {
  if (!h) return DIA_ERR_INVALID_ARG;
  if (n_epochs < 1 || n_epochs > h->cfg.max_epochs) return fail(h, DIA_ERR_INVALID_ARG, "n_epochs out of range");
  if (!opts || !h_I || !h_theta || !h_result) return fail(h, DIA_ERR_INVALID_ARG, "null opts or host buffer");
  if (h->cfg.noise == DIA_NOISE_FIXED) return fail(h, DIA_ERR_UNSUPPORTED, "the host-buffer calls take no variance map");
  int rc = host_path_prepare(h, h_mask != nullptr);
  if (rc != DIA_OK) return rc;
  dia_handle::HostPath& hp = h->host;
  const size_t npix = (size_t)h->cfg.n_rows * h->cfg.n_cols, np = (size_t)h->np;
  const int max_chunks = (int)(sizeof(hp.ready) / sizeof(hp.ready[0]));
  if (chunks <= 0) chunks = n_epochs >= 8 ? 4 : 1;
  if (chunks > n_epochs) chunks = n_epochs;
  if (chunks > max_chunks) chunks = max_chunks;
  // the copy stream starts when everything enqueued on the handle's stream so far (a previous user of the staging
  // buffers) is done
  cudaError_t ce = cudaEventRecord(hp.free_ev, h->stream);
  if (ce == cudaSuccess) ce = cudaStreamWaitEvent(hp.copy_stream, hp.free_ev, 0);
  for (int k = 0; k < chunks && ce == cudaSuccess; ++k) {
    const size_t a = (size_t)k * n_epochs / chunks, b = (size_t)(k + 1) * n_epochs / chunks;
    ce = cudaMemcpyAsync(hp.dI + a * npix, h_I + a * npix, sizeof(float) * (b - a) * npix, cudaMemcpyHostToDevice, hp.copy_stream);
    if (ce == cudaSuccess)
      ce = cudaMemcpyAsync(hp.dth + a * np, h_theta + a * np, sizeof(float) * (b - a) * np, cudaMemcpyHostToDevice, hp.copy_stream);
    if (ce == cudaSuccess && h_mask)
      ce = cudaMemcpyAsync(hp.dmask + a * npix, h_mask + a * npix, (b - a) * npix, cudaMemcpyHostToDevice, hp.copy_stream);
    if (ce == cudaSuccess) ce = cudaEventRecord(hp.ready[k], hp.copy_stream);
  }
  if (ce != cudaSuccess) { cudaStreamSynchronize(hp.copy_stream); return cuda_fail(h, ce, "host to device copy"); }
  for (int k = 0; k < chunks; ++k) {
    const size_t a = (size_t)k * n_epochs / chunks, b = (size_t)(k + 1) * n_epochs / chunks;
    ce = cudaStreamWaitEvent(h->stream, hp.ready[k], 0);
    if (ce != cudaSuccess) { cudaStreamSynchronize(hp.copy_stream); return cuda_fail(h, ce, "stream wait"); }
    rc = dia_fit(h, opts, (int)(b - a), hp.dI + a * npix, h_mask ? hp.dmask + a * npix : nullptr, nullptr, hp.dth + a * np,
                 hp.dres + a);
    if (rc != DIA_OK) { cudaStreamSynchronize(hp.copy_stream); cudaStreamSynchronize(h->stream); return rc; }
  }
  ce = cudaMemcpyAsync(h_theta, hp.dth, sizeof(float) * (size_t)n_epochs * np, cudaMemcpyDeviceToHost, h->stream);
  if (ce == cudaSuccess)
    ce = cudaMemcpyAsync(h_result, hp.dres, sizeof(dia_fit_result) * (size_t)n_epochs, cudaMemcpyDeviceToHost, h->stream);
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(h->stream);
  if (ce != cudaSuccess) return cuda_fail(h, ce, "device to host copy");
  return DIA_OK;
}

extern "C" int dia_hess_tc_plan(int m, int bg_degree, int* n_groups, int* n_types, unsigned char* types, int max_types,
                                short* perm, int max_slots) {
  if (m < 1 || m % 2 == 0 || m > DIA_MAX_KERNEL_SIZE || bg_degree < 0 || bg_degree > DIA_MAX_BG_DEGREE || !n_groups || !n_types ||
      !types || !perm)
    return fail(nullptr, DIA_ERR_INVALID_ARG, "dia_hess_tc_plan: bad argument");
  const int np = m * m + (bg_degree + 1) * (bg_degree + 2) / 2;
  const int G = (np + dia::kTcGroup - 1) / dia::kTcGroup;
  dia::HessTcTypes t;
  const int n = dia::hess_tc_make_types(np, &t);
  if (n == 0) return fail(nullptr, DIA_ERR_UNSUPPORTED, "type table exceeds the kernel's limit");
  if (n > max_types || G * dia::kTcGroup > max_slots) return fail(nullptr, DIA_ERR_INVALID_ARG, "dia_hess_tc_plan: outputs too small");
  int rpitch = 0, rh = 0;
  geometry_for(m, &rpitch, &rh);
  dia::hess_tc_make_perm(m, np, rpitch, perm);
  for (int i = 0; i < n; ++i) {
    types[5 * i] = t.g0[i];  types[5 * i + 1] = t.g1[i];  types[5 * i + 2] = t.a_sel[i];  types[5 * i + 3] = t.b_start[i];
    types[5 * i + 4] = t.n_groups[i];
  }
  *n_groups = G;  *n_types = n;
  return DIA_OK;
}

extern "C" int dia_tc_probe_gemm(void* stream, const float* d_A, const float* d_B, float* d_D, int K, int N, int mode) {
  if (!d_A || !d_B || !d_D) return fail(nullptr, DIA_ERR_INVALID_ARG, "null argument");
  if (K < dia::kTcProbeKC || K % dia::kTcProbeKC != 0 || N < 32 || N > 256 || N % 32 != 0 || mode < 0 || mode > 3)
    return fail(nullptr, DIA_ERR_INVALID_ARG, "dia_tc_probe_gemm: K must be a positive multiple of 64, N a multiple of 32 up to 256, mode 0..3");
  const cudaError_t ce = dia::tc_probe_launch((cudaStream_t)stream, d_A, d_B, d_D, K, N, mode);
  if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "tensor-core probe launch");
  return DIA_OK;
}

extern "C" int dia_get_info(const dia_handle* h, int* grid_blocks, int* threads_per_block, int* smem_bytes,
                            int* launches_per_eval) {
  if (!h) return DIA_ERR_INVALID_ARG;
  if (grid_blocks) *grid_blocks = h->grid;
  if (threads_per_block) *threads_per_block = dia::kThreads;
  if (smem_bytes) *smem_bytes = (int)h->smem;
  // kernels per stand-alone evaluation of the plain objective: (pack,) eval, reduce (, penalty); a dia_fit
  // iteration launches the same number (its step kernel takes the place of the reduce kernel)
  if (launches_per_eval) {
    dia::EvalParams p = {};               // a full batch of the plain objective
    p.n_epochs = h->cfg.max_epochs;  p.flat = h->cfg.d_flat;  p.noise_kind = h->cfg.noise;  p.hess_q0 = -1;
    if (h->small_grid > 0) p.small_rpt = small_plan(h, p.n_epochs).rpt;     // such handles run eval_small_kernel: no bank
    const bool kc = dia::eval_uses_const(h, p, false);
    *launches_per_eval = 2 + (kc ? 1 : 0) + (h->cfg.lambda_reg > 0.f ? 1 : 0);
  }
  return DIA_OK;
}

// ---------------------------------------------------------------------------------------------
// dia_eval_loss_grad_static: the evaluation for callers that cannot allocate (include/dia.h).
// The block partials live in a file-scope device array.  In host code `g_static_partials` is only the host-side
// shadow of the symbol, not a device address: the address is looked up once per device with cudaGetSymbolAddress,
// with that device current, and passed to the kernels in EvalParams::partials like any other workspace.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_static_partials[DIA_STATIC_SCRATCH_BYTES / sizeof(double)];

namespace {
constexpr int kStaticMaxDevices = 64;
struct StaticDevice {
  double* partials = nullptr;                               // device address of g_static_partials on this device
  int sms = 0;
  signed char occ[DIA_MAX_KERNEL_SIZE + 1] = {};            // resident CTAs per SM of eval_kernel<m> (0: not set up yet)
};
std::mutex g_static_mutex;
StaticDevice g_static_dev[kStaticMaxDevices];
}  // namespace

// once per device (address, SM count) and once per (device, m) (shared-memory attribute, occupancy); no allocation
static int static_setup(int dev, int m, size_t smem, StaticDevice* out) {
  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticDevice& d = g_static_dev[dev];
  if (!d.partials) {
    double* ptr = nullptr;
    cudaError_t ce = cudaGetSymbolAddress((void**)&ptr, g_static_partials);
    if (ce != cudaSuccess || !ptr) return cuda_fail(nullptr, ce, "cudaGetSymbolAddress(static scratch)");
    int sms = 0;
    ce = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaDeviceGetAttribute");
    d.sms = sms;
    d.partials = ptr;
  }
  if (d.occ[m] == 0) {
    int occ = 0;
    for (int aux = 0; aux < 2; ++aux) {                     // plain and generic (mask / flat / variance map) variants
      const void* k = kernel_for(m, aux == 1);
      cudaError_t ce = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaFuncSetAttribute(smem)");
      int o = 0;
      ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, k, dia::kThreads, smem);
      if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "occupancy query");
      if (o < 1) return fail(nullptr, DIA_ERR_UNSUPPORTED, "the evaluation kernel of this kernel size does not fit on an SM of this device");
      occ = (aux == 0 || o < occ) ? o : occ;
    }
    d.occ[m] = (signed char)(occ > 127 ? 127 : occ);
  }
  *out = d;
  return DIA_OK;
}

extern "C" int dia_eval_loss_grad_static(const dia_config* cfg, const float* d_R, int n_epochs, const float* d_I,
                                         const unsigned char* d_mask, const float* d_var, const float* d_theta,
                                         double* d_loss, double* d_grad) {
  if (!cfg || !d_R || !d_I || !d_theta || !d_loss || !d_grad) return fail(nullptr, DIA_ERR_INVALID_ARG, "null argument");
  if (cfg->m < 1 || cfg->m % 2 == 0) return fail(nullptr, DIA_ERR_INVALID_ARG, "m must be odd and >= 1");
  if (cfg->m > DIA_MAX_KERNEL_SIZE) return fail(nullptr, DIA_ERR_UNSUPPORTED, "m exceeds DIA_MAX_KERNEL_SIZE");
  if (cfg->n_rows < cfg->m || cfg->n_cols < cfg->m) return fail(nullptr, DIA_ERR_INVALID_ARG, "image smaller than kernel");
  if (n_epochs < 1) return fail(nullptr, DIA_ERR_INVALID_ARG, "n_epochs must be >= 1");
  if (!(cfg->lambda_reg >= 0.f)) return fail(nullptr, DIA_ERR_INVALID_ARG, "lambda_reg must be >= 0");
  if (cfg->bg_degree < 0) return fail(nullptr, DIA_ERR_INVALID_ARG, "bg_degree must be >= 0");
  if (cfg->bg_degree > DIA_MAX_BG_DEGREE) return fail(nullptr, DIA_ERR_UNSUPPORTED, "bg_degree exceeds DIA_MAX_BG_DEGREE");
  if (cfg->n_refs > 1 && cfg->n_refs != n_epochs) return fail(nullptr, DIA_ERR_INVALID_ARG, "n_refs must be 0, 1 or n_epochs");
  if (cfg->loss != DIA_LOSS_GAUSSIAN && cfg->loss != DIA_LOSS_HUBER) return fail(nullptr, DIA_ERR_INVALID_ARG, "bad loss");
  if (cfg->noise != DIA_NOISE_MODEL && cfg->noise != DIA_NOISE_FIXED) return fail(nullptr, DIA_ERR_INVALID_ARG, "bad noise mode");
  if (cfg->loss == DIA_LOSS_HUBER && !(cfg->huber_c > 0.f)) return fail(nullptr, DIA_ERR_INVALID_ARG, "huber_c must be > 0");
  if (cfg->noise == DIA_NOISE_MODEL && !(cfg->gain > 0.f && cfg->sigma0 >= 0.f))
    return fail(nullptr, DIA_ERR_INVALID_ARG, "need gain > 0 and sigma0 >= 0");
  if (cfg->noise == DIA_NOISE_FIXED && !d_var) return fail(nullptr, DIA_ERR_INVALID_ARG, "DIA_NOISE_FIXED needs d_var");
  if (cfg->noise == DIA_NOISE_MODEL && d_var) return fail(nullptr, DIA_ERR_INVALID_ARG, "d_var must be NULL in DIA_NOISE_MODEL");

  int dev = 0;
  cudaError_t ce = cudaGetDevice(&dev);
  if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "cudaGetDevice (no CUDA device: there is no CPU fallback)");
  if (dev < 0 || dev >= kStaticMaxDevices) return fail(nullptr, DIA_ERR_UNSUPPORTED, "device ordinal beyond the static set-up table");
  StaticDevice sd;
  int rc = static_setup(dev, cfg->m, smem_for(cfg->m), &sd);
  if (rc != DIA_OK) return rc;

  // a handle on the stack, laid out as dia_create would for max_epochs == n_epochs; generic kernel only (no
  // eval_small_kernel, no constant bank), its workspace pointer aimed at the static array
  dia_handle hs;
  hs.cfg = *cfg;  hs.cfg.max_epochs = n_epochs;
  hs.d_R = d_R;  hs.stream = (cudaStream_t)cfg->stream;  hs.sms = sd.sms;
  hs.n_refs = cfg->n_refs > 1 ? cfg->n_refs : 1;
  hs.np = cfg->m * cfg->m + (cfg->bg_degree + 1) * (cfg->bg_degree + 2) / 2;
  hs.smem = smem_for(cfg->m);
  hs.d_const_stage = nullptr;  hs.small_grid = 0;  hs.grid_limit = 0;  hs.cluster_fit = 0;
  hs.flush_tiles = dia::kFlushTiles;
  hs.tiles = ((cfg->n_cols - cfg->m + 1 + dia::kTW - 1) / dia::kTW) * ((cfg->n_rows - cfg->m + 1 + dia::kTH - 1) / dia::kTH);
  const long long items = (long long)hs.tiles * n_epochs, resident = (long long)sd.sms * sd.occ[cfg->m];
  hs.grid = (int)(items < resident ? items : resident);
  hs.use_tma = 0;
  if (cfg->n_cols % 4 == 0 && aligned16(d_R)) {             // descriptor encoding is host arithmetic, no allocation
    int rpitch = 0, rh = 0;
    geometry_for(cfg->m, &rpitch, &rh);
    hs.use_tma = make_tensor_map(&hs.tmR, d_R, cfg->n_cols, cfg->n_rows, hs.n_refs, rpitch, rh) ? 1 : 0;
  }
  hs.d_partials = sd.partials;
  std::memset(&hs.fit, 0, sizeof(hs.fit));                  // never touched on this path

  const int np1 = hs.np + 1;
  const unsigned long long need = 8ull * (unsigned long long)n_epochs * np1 * (unsigned long long)dia::eval_part_cols(&hs, n_epochs);
  if (need > DIA_STATIC_SCRATCH_BYTES)
    return fail(nullptr, DIA_ERR_UNSUPPORTED, "dia_eval_loss_grad_static: this batch needs " + std::to_string(need) +
                " bytes of block partials, the static scratch holds DIA_STATIC_SCRATCH_BYTES = " +
                std::to_string((unsigned long long)DIA_STATIC_SCRATCH_BYTES) + " (use a handle, or fewer epochs per call)");

  dia::EvalParams p;
  dia::TensorMaps tm;
  fill_params(&hs, n_epochs, d_I, d_mask, d_var, d_theta, nullptr, &p, &tm, -1);
  ce = dia::launch_eval(&hs, p, tm);
  if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "eval launch");
  dia::reduce_partials_kernel<<<dim3((np1 + 7) / 8, n_epochs), 256, 0, hs.stream>>>(
      hs.d_partials, dia::eval_part_cols_p(&hs, p), np1, nullptr, d_loss, d_grad);
  if (cfg->lambda_reg > 0.f)
    dia::penalty_kernel<<<n_epochs, dia::kFitThreads, 0, hs.stream>>>(d_theta, cfg->m, hs.np, lambda_n(&hs), d_loss, d_grad);
  ce = cudaGetLastError();
  if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "reduce launch");
  return DIA_OK;
}
