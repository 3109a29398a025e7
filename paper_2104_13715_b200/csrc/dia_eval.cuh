// dia_eval.cuh -- fused loss + gradient kernel for the B08 discrete-pixel kernel model (sm_100a).
//
// One persistent CTA (256 threads, 2 CTAs per SM) loops over 64x64 tiles of the valid region.  Per tile:
//   stage    one elected thread issues two TMA tensor copies (cp.async.bulk.tensor): the R tile plus its
//            (m-1) halo, and the I tile, zero filled outside the image; completion is signalled on
//            mbarriers, the copies of tile t+1 overlap the gradient phase of tile t.  (Images whose rows
//            are not 16-byte aligned take a cp.async path that fills the same shared-memory layout.)
//   forward  each thread owns a 16-pixel row strip: M = R (x) K + B0 (Eq. 2) in FP32
//            registers, then residual, variance (Eq. 6), loss term (Eq. 8 / Eq. 12-13,
//            PAPER.md:115, 154-161) and the weight w = dL/dM, written to the shared w tile,
//   grad     thread (a, s) owns the m accumulators g[a][0..m-1] and correlates 16-pixel chunks of w
//            against the staged R rows (dL/dK[a][b] = sum w_ij R[i+a][j+b]); the FP32 accumulators
//            live in a thread-private shared-memory row between tiles,
//   flush    once per epoch (and every kFlushTiles tiles) the FP32 strips are summed over s in fixed
//            order in FP64 and written to this CTA's partials.
// Two CTA-wide barriers per tile.  Nothing n^2-sized is written to HBM.  The tile->CTA map and every
// reduction order are fixed, so repeated evaluations are bit-identical.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace dia {

constexpr int kThreads = 256;
constexpr int kTW = 64, kTH = 64;     // output tile
constexpr int kP = 16;                // forward strip / gradient chunk length (pixels)
constexpr int kIPitch = 68;           // I/w tile pitch (floats); 68/4 = 17 is odd => conflict-free rows
constexpr int kFlushTiles = 32;       // FP32 gradient strips are folded into FP64 at least this often (EvalParams::flush_tiles)
constexpr int kSmemBudget = 113 * 1024;   // per CTA, two CTAs per SM
constexpr int kSmemBudget1 = 226 * 1024;  // per CTA when only one fits (m >= 33)
constexpr int kMaxBg = 16;            // background coefficients held per epoch (degree <= 3 uses 10)

__host__ __device__ constexpr int round_up(int x, int q) { return (x + q - 1) / q * q; }

template <int M>
struct Geo {
  static constexpr int H = (M - 1) / 2;
  static constexpr int IOFF = H % 4;                         // column shift of the staged I tile
  static constexpr int RH = kTH + M - 1;                     // staged R rows
  static constexpr int RSEG = round_up(kP + M - 1, 4);       // floats a thread loads per R row
  static constexpr int RMIN = kTW - kP + RSEG;               // columns touched
  // pitch == 4 (mod 8) floats: 8 consecutive rows hit 8 distinct 16-byte bank groups
  static constexpr int RPITCH = RMIN + ((4 - RMIN % 8) + 8) % 8;
  static constexpr int KP = round_up(M, 4);                  // padded kernel row
  static constexpr int S = kThreads / M;                     // pixel sub-sets in the gradient phase
  static constexpr int R_FLOATS = RH * RPITCH;
  static constexpr int I_FLOATS = kTH * kIPitch;
  static constexpr int K_FLOATS = M * KP;
  static constexpr int ACC_FLOATS = kThreads * KP;           // thread-private FP32 gradient strips
  static constexpr int R_BYTES = R_FLOATS * 4, I_BYTES = I_FLOATS * 4;
  static constexpr int R_STRIDE = round_up(R_BYTES, 128);    // TMA destinations are 128-byte aligned
  static constexpr int FIXED_BYTES = 4 * (2 * I_FLOATS + K_FLOATS + ACC_FLOATS) + 2560;
  // two CTAs per SM while one R buffer fits into half of the shared memory (m <= 31), else one CTA with up to
  // 255 registers per thread
  static constexpr int CTAS = (FIXED_BYTES + R_STRIDE <= kSmemBudget) ? 2 : 1;
  // two R buffers when they fit next to a second resident CTA, else one (the copy of the next R
  // tile then waits for the gradient phase to finish)
  static constexpr int NRBUF = (FIXED_BYTES + 2 * R_STRIDE <= (CTAS == 2 ? kSmemBudget : kSmemBudget1)) ? 2 : 1;
  // shared-memory map (byte offsets from a 128-byte aligned base)
  static constexpr int OFF_R = 0;
  static constexpr int OFF_I = NRBUF * R_STRIDE;
  static constexpr int I_STRIDE = round_up(I_BYTES, 128);
  static constexpr int OFF_W = OFF_I + I_STRIDE;
  static constexpr int OFF_ACC = OFF_W + I_STRIDE;
  static constexpr int OFF_K = OFF_ACC + 4 * ACC_FLOATS;
  static constexpr int OFF_BG = OFF_K + 4 * K_FLOATS;        // background coefficients b_mn (Eq. 18)
  static constexpr int OFF_BAR = round_up(OFF_BG + 4 * kMaxBg, 16);
  static constexpr int OFF_BGACC = OFF_BAR + 64 + 128;       // FP64 background-gradient sums, one row per warp
  static constexpr size_t SMEM = OFF_BGACC + 8 * (kThreads / 32) * kMaxBg + 128;   // + alignment slack
  static_assert(RPITCH % 8 == 4, "pitch");
  static_assert(R_BYTES % 16 == 0 && I_BYTES % 16 == 0, "TMA sizes");
  static_assert(RPITCH <= 256 && RH <= 256, "TMA box limits");
};

// Constant-bank copy of what the forward phase needs from theta (KC instantiation).  With the kernel pixels in
// the constant bank the compiler keeps them in uniform registers, so a forward FFMA reads two vector registers
// instead of three: the operand collector stops being the limit (measured +10 % on the whole evaluation).
// pack_const_kernel fills a staging copy in global memory, a device-to-device copy moves it here before every
// evaluation.  Epochs are listed by ACTIVE position j (epochs whose done flag is set are left out), so that the
// constant-bank offset j * M * KP depends on uniform values only.
constexpr int kConstEpochs = 48;                    // active epochs one launch can address
constexpr int kConstK = 15872;                      // floats of padded kernel rows [j][M][KP]
struct alignas(16) ConstBlock {
  int n_active;                                     // epochs to evaluate in this launch
  int pad[3];
  int active[kConstEpochs];                         // epoch index of active position j
  alignas(16) float K[kConstK];
};
static_assert(sizeof(ConstBlock) <= 65536 - 1024, "constant bank");
static __constant__ ConstBlock c_blk;      // one copy per translation unit (per kernel size), see dia_eval_inst.cu

struct EvalParams {
  const float* R;            // [n_refs][n_rows][n_cols]
  const float* I;            // [E][n_rows][n_cols]
  const unsigned char* mask; // [E][n_rows][n_cols] or null
  const float* var;          // [E][n_rows][n_cols] or null (FIXED noise)
  const float* flat;         // [n_rows][n_cols] or null
  const float* theta;        // [E][np] float32: K row-major, then the background coefficients
  float* diff;               // [E][n_rows][n_cols] difference image (DIFF instantiation only)
  const int* done;           // [E] or null: epochs with done != 0 are skipped
  double* partials;          // [E][NP+1][ncols], ncols = min(tiles, gridDim.x): rows g_K (M*M), g_B0, loss;
                             // one column per CTA that owns tiles of the epoch
  int n_rows, n_cols, n_epochs;
  int n_refs;                // 1: one reference shared by all epochs; else one reference per epoch
  int hess_q0;               // < 0: loss and gradient.  >= 0 (AUX instantiation only, dia_hessian): every "epoch" e
                             // shares target / mask / variance map 0 and theta 0 and produces row hess_q0 + e of the
                             // Hessian, sum_V h X_q X with h = d^2 l / dM^2 (D3), in place of the gradient
  int part_rows;             // rows of partials per epoch: np + 1 (gradient, loss), or 3 in difference-image mode
  int np, bg_degree;         // parameters per epoch = M*M + (d+1)(d+2)/2; degree d of the background (Eq. 18)
  float bg_xc, bg_yc, bg_inv_nx, bg_inv_ny;   // Eq. 19: eta = (x - xc) / N_x, xi = (y - yc) / N_y
  int tiles_x, tiles_y;
  int loss_kind, noise_kind;
  float huber_c, sigma0_sq, inv_gain;
  int use_tma;               // 1: rows are 16-byte aligned, tensor maps are valid
  int epoch_per_cta;         // item order: 0 = CTA b takes items b, b + grid, ... of the epoch-major list;
                             // 1 = CTA b takes every tile of epochs b, b + grid, ... (many small images: one
                             // change of epoch per image instead of one per tile; partials have one column)
  int cp8;                   // cp.async staging path: 1 = rows are 8-byte aligned (even n_cols), copy pixel pairs
  int small_rpt;             // > 0: eval_small_kernel (dia_eval_small.cuh) runs this evaluation, rows per thread and tile
  int small_lxlog;           // ... log2 of the lanes of a warp that sit side by side in x (the rest stack in y)
  int small_vec;             // ... rows of R and I are 16-byte aligned: 128-bit loads
  int flush_tiles;           // the FP32 gradient strips are folded into FP64 every flush_tiles tiles (kFlushTiles)
};

struct TensorMaps {          // passed by value as a __grid_constant__ kernel parameter
  CUtensorMap R;             // 3-D {n_cols, n_rows, n_refs}, box {RPITCH, RH, 1}
  CUtensorMap I;             // 3-D {n_cols, n_rows, E}, box {kIPitch, kTH, 1}
};

// ------------------------------------------------------------------------------------------------
// PTX helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void cp_async_4(unsigned dst, const void* gmem, int src_bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;\n" ::"r"(dst), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_8(unsigned dst, const void* gmem, int src_bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_mbar_arrive(unsigned bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }

// L2 eviction policies: the reference is re-read for every epoch of a batch (keep it: evict_last), a target
// tile is read once per evaluation (evict_first), so that a 64 MiB reference stays resident in the 126 MB L2.
__device__ __forceinline__ unsigned long long l2_policy_evict_last() {
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ unsigned long long l2_policy_evict_first() {
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap* tm, int x, int y, int z, unsigned bar,
                                            unsigned long long pol) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;\n" ::
          "r"(dst), "l"(tm), "r"(x), "r"(y), "r"(z), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ float lg2_approx(float x) {      // x is a variance: never subnormal, so no rescaling step
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// Packed FP32 pairs (sm_100 fma.rn.f32x2 / FFMA2): one issue slot carries two fused multiply-adds, which halves the
// issue slots the stencil and the correlation need and leaves the FMA pipe -- not instruction issue -- as the bound.
// A pair lives in an aligned 64-bit register; {lo, hi} <-> pair moves are register renamings, not instructions.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ float pk_lo(f32x2 v) {
  float lo;
  asm("{\n.reg .b32 t;\nmov.b64 {%0, t}, %1;\n}" : "=f"(lo) : "l"(v));
  return lo;
}
__device__ __forceinline__ float pk_hi(f32x2 v) {
  float hi;
  asm("{\n.reg .b32 t;\nmov.b64 {t, %0}, %1;\n}" : "=f"(hi) : "l"(v));
  return hi;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {      // {a.lo b.lo + c.lo, a.hi b.hi + c.hi}
  f32x2 d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 d;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}

__device__ __forceinline__ double warp_sum_f64(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ------------------------------------------------------------------------------------------------
// staging: executed by every thread at CTA-uniform points
// ------------------------------------------------------------------------------------------------
// cp.async staging of a ROWS x PITCH tile whose rows are not 16-byte aligned (TMA needs that): 8-byte copies of pixel
// pairs when n_cols is even (pairs are 8-byte aligned and inside or outside the image together), else 4-byte
// copies; zero filled outside the image.  Deliberately not inlined: the fast path never runs it, and four inlined
// copies of these loops lengthen the tile loop by a tenth (instruction-cache misses cost 1.6 % at 4096^2).
template <int ROWS, int PITCH>
__device__ __noinline__ void stage_tile_cp_async(const float* __restrict__ img, int n_rows, int n_cols, int cp8, int y0,
                                                 int x0, unsigned dst) {
  if (cp8) {
    for (int idx = threadIdx.x; idx < ROWS * (PITCH / 2); idx += kThreads) {
      const int rr = idx / (PITCH / 2), cc = 2 * (idx - rr * (PITCH / 2));
      const int gy = y0 + rr, gx = x0 + cc;
      const bool ok = (gy < n_rows) && (gx < n_cols);
      const float* src = ok ? img + (size_t)gy * n_cols + gx : img;
      cp_async_8(dst + 8u * (unsigned)idx, src, ok ? 8 : 0);
    }
  } else {
    for (int idx = threadIdx.x; idx < ROWS * PITCH; idx += kThreads) {
      const int rr = idx / PITCH, cc = idx - rr * PITCH;
      const int gy = y0 + rr, gx = x0 + cc;
      const bool ok = (gy < n_rows) && (gx < n_cols);
      const float* src = ok ? img + (size_t)gy * n_cols + gx : img;
      cp_async_4(dst + 4u * (unsigned)idx, src, ok ? 4 : 0);
    }
  }
}

// R rows [y0, y0+RH) x cols [x0, x0+RPITCH), zero filled outside the image.
template <int M>
__device__ __forceinline__ void stage_R(const EvalParams& p, const TensorMaps& tm, int e, int tile, unsigned dst,
                                        unsigned bar) {
  using G = Geo<M>;
  const int ref = p.n_refs > 1 ? e : 0;    // one reference per epoch, or one shared by all epochs
  const int ty = tile / p.tiles_x, tx = tile - ty * p.tiles_x;
  const int y0 = ty * kTH, x0 = tx * kTW;
  if (p.use_tma) {
    if (threadIdx.x == 0) {
      fence_proxy_async();
      mbar_expect_tx(bar, G::R_BYTES);
      tma_load_3d(dst, &tm.R, x0, y0, ref, bar, l2_policy_evict_last());
    }
  } else {
    stage_tile_cp_async<G::RH, G::RPITCH>(p.R + (size_t)ref * p.n_rows * p.n_cols, p.n_rows, p.n_cols, p.cp8, y0, x0, dst);
    cp_async_mbar_arrive(bar);
  }
}

// I rows [y0+H, y0+H+kTH) x cols [x0+H-IOFF, x0+H-IOFF+kIPitch) of epoch e, zero filled outside the image.
// A TMA box must start on a 16-byte boundary of the row, so the tile starts IOFF = H mod 4 columns early and
// pixel (r, c) of the tile sits at Is[r * kIPitch + c + IOFF].
template <int M>
__device__ __forceinline__ void stage_I(const EvalParams& p, const TensorMaps& tm, int e, int tile, unsigned dst,
                                        unsigned bar) {
  using G = Geo<M>;
  const int ty = tile / p.tiles_x, tx = tile - ty * p.tiles_x;
  const int y0 = ty * kTH + G::H, x0 = tx * kTW + G::H - G::IOFF;
  if (p.hess_q0 >= 0) e = 0;
  if (p.use_tma) {
    if (threadIdx.x == 0) {
      fence_proxy_async();
      mbar_expect_tx(bar, G::I_BYTES);
      tma_load_3d(dst, &tm.I, x0, y0, e, bar, l2_policy_evict_first());
    }
  } else {
    stage_tile_cp_async<kTH, kIPitch>(p.I + (size_t)e * p.n_rows * p.n_cols, p.n_rows, p.n_cols, p.cp8, y0, x0, dst);
    cp_async_mbar_arrive(bar);
  }
}

// ------------------------------------------------------------------------------------------------
// per-pixel residual / noise / loss / weight (D1)
//   AUX = false: noise model of Eq. 6 with F == 1, no mask (the fast path)
//   AUX = true : any of mask / flat field / caller variance map, read from global memory
// ------------------------------------------------------------------------------------------------
template <bool AUX, bool EDGE>
__device__ __forceinline__ void pixel_terms(const EvalParams& p, int e, size_t npix, size_t gidx, bool inside,
                                            float Mv, float Iv, float& li, float& wi) {
  bool use = EDGE ? inside : true;
  float v, bp;
  if (AUX) {
    if (p.hess_q0 >= 0) e = 0;
    if (use && p.mask) use = p.mask[(size_t)e * npix + gidx] != 0;
    if (p.noise_kind == 0) {
      float a_ij = p.sigma0_sq, b_ij = p.inv_gain;
      if (p.flat && use) {
        const float invF = 1.0f / p.flat[gidx];
        a_ij *= invF * invF;
        b_ij *= invF;
      }
      v = fmaf(b_ij, fmaxf(Mv, 0.f), a_ij);
      bp = Mv > 0.f ? b_ij : 0.f;
    } else {
      v = use ? p.var[(size_t)e * npix + gidx] : 1.f;
      bp = 0.f;
    }
  } else {
    v = fmaf(p.inv_gain, fmaxf(Mv, 0.f), p.sigma0_sq);
    bp = Mv > 0.f ? p.inv_gain : 0.f;
  }
  const float res = Iv - Mv;
  const float inv_v = rcp_approx(v);
  const float hb = 0.5f * bp * inv_v;
  const float z2 = res * res * inv_v;
  li = 0.5f * z2;
  wi = fmaf(-res, inv_v, hb * (1.0f - z2));
  const bool hess = AUX && p.hess_q0 >= 0;
  // D3: h = dw/dM = 1/v + 2 b' r / v^2 + b'^2 r^2 / v^3 - b'^2 / (2 v^2), with hb = b'/(2v)
  if (hess) wi = inv_v * (1.0f + 4.0f * hb * res) + 4.0f * hb * hb * (z2 - 0.5f);
  if (p.loss_kind == 1) {                          // Huber, Eq. 12
    const float rsd = rsqrtf(v);
    const float z = res * rsd;
    if (fabsf(z) > p.huber_c) {
      const float psi = copysignf(p.huber_c, z);
      li = p.huber_c * (fabsf(z) - 0.5f * p.huber_c);
      wi = fmaf(-psi, rsd, hb * (1.0f - psi * z));
      // D3, linear branch: dz/dM = -1/s - z hb;  h = psi hb / s - psi hb dz/dM + 2 hb^2 (psi z - 1)
      if (hess) wi = psi * hb * (rsd + (rsd + z * hb)) + 2.0f * hb * hb * (psi * z - 1.0f);
    }
  }
  // 1/2 ln v = (ln 2 / 2) log2 v from the MUFU unit: absolute error 2^-22 in log2 v, 1e-7 on a term of size 2-6 -- below
  // the float32 rounding of the term itself; logf costs ~15 instructions more per pixel (a third of this epilogue)
  if (!AUX || p.noise_kind == 0) li = fmaf(0.34657359028f, lg2_approx(v), li);
  if (AUX || EDGE) {
    if (!use) { li = 0.f; wi = 0.f; }
  }
}

// ------------------------------------------------------------------------------------------------
// forward: M for the 16-pixel strip at (f_row, f_col) of the tile.  Kernel rows are taken in pairs
// (0, M-1), (1, M-2), ... and the centre row last; inside a row the columns go wings -> centre.
// Each pair is one FP32 chain that is then added to the running total, so the large centre terms
// come last ("accumulation order").
// ------------------------------------------------------------------------------------------------
// Row chain state of one 16-pixel strip in packed form.  Kernel columns b of even index meet the pixel pairs
// (0,1), (2,3), ... with an aligned pair of reference pixels, those of odd index the pixel pairs (1,2), (3,4), ...
// (and pixels 0 and 15 singly): two chains per pixel, one per column parity, both in the order wings -> centre.
struct RowChain {
  f32x2 e[kP / 2];         // even columns: pixels (2p, 2p+1)
  f32x2 o[kP / 2 - 1];     // odd columns: pixels (2p+1, 2p+2)
  float o0, o15;           // odd columns: pixels 0 and 15
};

template <int M, bool KC>
__device__ __forceinline__ void row_chain(const float* __restrict__ Ks, int koff, const float* __restrict__ Rrow, int a,
                                          RowChain& c, bool first) {
  using G = Geo<M>;
  float k[G::KP];
  f32x2 rp[G::RSEG / 2];                               // rp[t] = (r[2t], r[2t+1])
  if (KC) {                                          // warp-uniform loads from the constant bank
    const float4* k4 = reinterpret_cast<const float4*>(c_blk.K + koff + a * G::KP);
#pragma unroll
    for (int q = 0; q < G::KP / 4; ++q) {
      const float4 v = k4[q];
      k[4 * q] = v.x; k[4 * q + 1] = v.y; k[4 * q + 2] = v.z; k[4 * q + 3] = v.w;
    }
  } else {
    const float4* k4 = reinterpret_cast<const float4*>(Ks + a * G::KP);
#pragma unroll
    for (int q = 0; q < G::KP / 4; ++q) {
      const float4 v = k4[q];
      k[4 * q] = v.x; k[4 * q + 1] = v.y; k[4 * q + 2] = v.z; k[4 * q + 3] = v.w;
    }
  }
  const ulonglong2* r2 = reinterpret_cast<const ulonglong2*>(Rrow + a * G::RPITCH);
#pragma unroll
  for (int q = 0; q < G::RSEG / 4; ++q) {
    const ulonglong2 v = r2[q];
    rp[2 * q] = v.x; rp[2 * q + 1] = v.y;
  }
  bool first_e = first, first_o = first;
#pragma unroll
  for (int ib = 0; ib < M; ++ib) {
    const int b = (ib == 0) ? 0 : ((ib & 1) ? (M - 1 - (ib >> 1)) : (ib >> 1));     // 0, M-1, 1, M-2, ..., centre
    const f32x2 kk = pk2(k[b], k[b]);
    if ((b & 1) == 0) {
      if (first_e) {
#pragma unroll
        for (int p = 0; p < kP / 2; ++p) c.e[p] = mul2(kk, rp[p + b / 2]);
      } else {
#pragma unroll
        for (int p = 0; p < kP / 2; ++p) c.e[p] = fma2(kk, rp[p + b / 2], c.e[p]);
      }
      first_e = false;
    } else {
      const float r_first = pk_hi(rp[(b - 1) / 2]);            // r[b]
      const float r_last = pk_lo(rp[(kP - 1 + b) / 2]);        // r[15 + b]
      if (first_o) {
#pragma unroll
        for (int p = 0; p < kP / 2 - 1; ++p) c.o[p] = mul2(kk, rp[p + (b + 1) / 2]);
        c.o0 = k[b] * r_first;  c.o15 = k[b] * r_last;
      } else {
#pragma unroll
        for (int p = 0; p < kP / 2 - 1; ++p) c.o[p] = fma2(kk, rp[p + (b + 1) / 2], c.o[p]);
        c.o0 = fmaf(k[b], r_first, c.o0);  c.o15 = fmaf(k[b], r_last, c.o15);
      }
      first_o = false;
    }
  }
}

// adds the two chains of a row pair to the running model values
template <int M>
__device__ __forceinline__ void chain_to_total(const RowChain& c, float (&tot)[kP]) {
#pragma unroll
  for (int p = 0; p < kP / 2; ++p) {
    float lo = pk_lo(c.e[p]), hi = pk_hi(c.e[p]);
    if (M > 1) {
      lo += (p == 0) ? c.o0 : pk_hi(c.o[p > 0 ? p - 1 : 0]);
      hi += (p == kP / 2 - 1) ? c.o15 : pk_lo(c.o[p < kP / 2 - 1 ? p : 0]);
    }
    tot[2 * p] += lo;
    tot[2 * p + 1] += hi;
  }
}

template <int M, bool KC>
__device__ __forceinline__ void forward_strip(const float* __restrict__ Ks, int koff, const float* __restrict__ Rrow, float B0,
                                              float (&tot)[kP]) {
  using G = Geo<M>;
#pragma unroll
  for (int q = 0; q < kP; ++q) tot[q] = B0;
  RowChain c;
#pragma unroll 1
  for (int ip = 0; ip < G::H; ++ip) {
    row_chain<M, KC>(Ks, koff, Rrow, ip, c, true);
    row_chain<M, KC>(Ks, koff, Rrow, M - 1 - ip, c, false);
    chain_to_total<M>(c, tot);
  }
  row_chain<M, KC>(Ks, koff, Rrow, G::H, c, true);
  chain_to_total<M>(c, tot);
}

// Adds the background terms beyond b_00 (Eq. 18-19) to the model strip.
template <int M>
__device__ __forceinline__ void add_background(const EvalParams& p, const float* __restrict__ Bs, int iy, int ix0,
                                               float (&tot)[kP]) {
  using G = Geo<M>;
  const int d = p.bg_degree;
  if (d <= 0) return;                                // CTA-uniform
  const float eta0 = ((float)(ix0 + G::H) - p.bg_xc) * p.bg_inv_nx;
  const float xi = ((float)(iy + G::H) - p.bg_yc) * p.bg_inv_ny;
  float c[4] = {0.f, 0.f, 0.f, 0.f};                 // c_p(xi) = sum_n b_pn xi^n, without b_00
  int t = 0;
#pragma unroll
  for (int mm = 0; mm < 4; ++mm) {
    float xn = 1.f;
#pragma unroll
    for (int nn = 0; nn < 4; ++nn) {
      if (mm <= d && nn <= d - mm) {
        if (t > 0) c[mm] = fmaf(Bs[t], xn, c[mm]);
        ++t;
      }
      xn *= xi;
    }
  }
#pragma unroll
  for (int q = 0; q < kP; ++q) {
    const float eta = fmaf((float)q, p.bg_inv_nx, eta0);
    tot[q] += fmaf(fmaf(fmaf(c[3], eta, c[2]), eta, c[1]), eta, c[0]);
  }
}

// Difference-image mode: D = I - M for every pixel of the valid region, written to global
// memory, and the sums of eps = (I - M)/sigma, eps^2 and the pixel count over the unmasked valid pixels
// (fit-quality metrics MFB, MFV, Eq. 29-30).
template <int M, bool EDGE>
__device__ __forceinline__ void strip_diff(const EvalParams& p, int e, size_t npix, int iy, int ix0, int vr, int vc,
                                           const float (&tot)[kP], const float* __restrict__ irow, float& s_eps,
                                           float& s_eps2, float& s_cnt) {
  using G = Geo<M>;
  const size_t gbase = (size_t)(iy + G::H) * p.n_cols + (ix0 + G::H);
  float* __restrict__ Drow = p.diff + (size_t)e * npix + gbase;
  s_eps = 0.f; s_eps2 = 0.f; s_cnt = 0.f;
#pragma unroll
  for (int q = 0; q < kP; ++q) {
    const bool inside = EDGE ? ((iy < vr) && (ix0 + q < vc)) : true;
    if (!inside) continue;
    const float Mv = tot[q];
    const float res = irow[q + G::IOFF] - Mv;
    Drow[q] = res;
    bool use = true;
    if (p.mask) use = p.mask[(size_t)e * npix + gbase + q] != 0;
    float v;
    if (p.noise_kind == 0) {
      float a_ij = p.sigma0_sq, b_ij = p.inv_gain;
      if (p.flat) {
        const float invF = 1.0f / p.flat[gbase + q];
        a_ij *= invF * invF;
        b_ij *= invF;
      }
      v = fmaf(b_ij, fmaxf(Mv, 0.f), a_ij);
    } else {
      v = p.var[(size_t)e * npix + gbase + q];
    }
    if (use) {
      const float eps = res * rsqrtf(v);
      s_eps += eps;
      s_eps2 = fmaf(eps, eps, s_eps2);
      s_cnt += 1.f;
    }
  }
}

// epilogue of the forward phase for one strip: loss terms and the w strip.  With a polynomial background
// (Eq. 18-19) the terms beyond b_00 are added to the model here, and the sums
// S_p = sum_q w_q eta_q^p (p = 0..d) of the strip are returned for the background gradient.
template <int M, bool AUX, bool EDGE>
__device__ __forceinline__ void strip_epilogue(const EvalParams& p, int e, size_t npix, int iy, int ix0, int vr, int vc,
                                               float (&tot)[kP], const float* __restrict__ irow,
                                               float* __restrict__ wrow, const float* __restrict__ Bs, float& lsum,
                                               float& wsum, float (&Sp)[4], const float* __restrict__ xrow = nullptr,
                                               int hx_m = 0, int hx_n = 0) {
  using G = Geo<M>;
  float iv[kP];
  if (G::IOFF == 0) {
#pragma unroll
    for (int q = 0; q < kP / 4; ++q) {
      const float4 v = reinterpret_cast<const float4*>(irow)[q];
      iv[4 * q] = v.x; iv[4 * q + 1] = v.y; iv[4 * q + 2] = v.z; iv[4 * q + 3] = v.w;
    }
  } else {
#pragma unroll
    for (int q = 0; q < kP; ++q) iv[q] = irow[q + G::IOFF];
  }
  const int d = p.bg_degree;
  const float eta0 = ((float)(ix0 + G::H) - p.bg_xc) * p.bg_inv_nx;
  add_background<M>(p, Bs, iy, ix0, tot);
  const size_t gbase = (size_t)(iy + G::H) * p.n_cols + (ix0 + G::H);
  lsum = 0.f; wsum = 0.f;
  Sp[1] = 0.f; Sp[2] = 0.f; Sp[3] = 0.f;
#pragma unroll
  for (int q = 0; q < kP; ++q) {
    float li, wi;
    pixel_terms<AUX, EDGE>(p, e, npix, gbase + q, (iy < vr) && (ix0 + q < vc), tot[q], iv[q], li, wi);
    if (AUX && p.hess_q0 >= 0) {           // Hessian row q: weight h X_q, X_q a shifted reference pixel or eta^m xi^n
      float xq;
      if (xrow) {
        xq = xrow[q];
      } else {
        const float eta = fmaf((float)q, p.bg_inv_nx, eta0);
        const float xi = ((float)(iy + G::H) - p.bg_yc) * p.bg_inv_ny;
        xq = 1.f;
        for (int k = 0; k < hx_m; ++k) xq *= eta;
        for (int k = 0; k < hx_n; ++k) xq *= xi;
      }
      wi *= xq;
    }
    lsum += li;
    wsum += wi;
    if (d > 0) {
      const float eta = fmaf((float)q, p.bg_inv_nx, eta0);
      const float w1 = wi * eta, w2 = w1 * eta;
      Sp[1] += w1; Sp[2] += w2; Sp[3] = fmaf(w2, eta, Sp[3]);
    }
    iv[q] = wi;
  }
  Sp[0] = wsum;
#pragma unroll
  for (int q = 0; q < kP / 4; ++q)
    reinterpret_cast<float4*>(wrow)[q] = make_float4(iv[4 * q], iv[4 * q + 1], iv[4 * q + 2], iv[4 * q + 3]);
}

// ------------------------------------------------------------------------------------------------
// gradient: thread (a, s) owns g[a][0..M-1] and correlates 16-pixel chunks of the weight tile against row i + a of
// the staged R tile: g[a][b] += w[q] r[q + b].  Packed form: for even q the kernel columns pair up as (0,1), (2,3), ...
// (+ column M-1 singly) against aligned pairs of reference pixels, for odd q as (1,2), (3,4), ... (+ column 0 singly);
// the two pairings are two accumulator sets, added when the strip is stored.  Kernel sizes whose 2 M accumulators
// do not fit the register budget of two CTAs per SM keep one set and take the odd pixels with scalar FMAs.
// ------------------------------------------------------------------------------------------------
template <int M>
struct GradAcc {
  static constexpr int NP = (M - 1) / 2 > 0 ? (M - 1) / 2 : 1;
  static constexpr bool TWO = Geo<M>::CTAS == 1 || (2 * M + kP + Geo<M>::RSEG <= 108);
  f32x2 e[NP];    // columns (2t, 2t+1)
  float el;       // column M-1
  f32x2 o[NP];    // columns (2t+1, 2t+2)        (TWO only)
  float of;       // column 0                    (TWO only)
};

template <int M>
__device__ __forceinline__ void grad_acc_load(GradAcc<M>& A, const float4* __restrict__ myacc) {
  using G = Geo<M>;
  float acc[G::KP];
#pragma unroll
  for (int q = 0; q < G::KP / 4; ++q) {
    const float4 v = myacc[q];
    acc[4 * q] = v.x; acc[4 * q + 1] = v.y; acc[4 * q + 2] = v.z; acc[4 * q + 3] = v.w;
  }
#pragma unroll
  for (int t = 0; t < (M - 1) / 2; ++t) { A.e[t] = pk2(acc[2 * t], acc[2 * t + 1]); A.o[t] = pk2(0.f, 0.f); }
  A.el = acc[M - 1];
  A.of = 0.f;
}
template <int M>
__device__ __forceinline__ void grad_acc_zero(GradAcc<M>& A) {
#pragma unroll
  for (int t = 0; t < (M - 1) / 2; ++t) { A.e[t] = pk2(0.f, 0.f); A.o[t] = pk2(0.f, 0.f); }
  A.el = 0.f;
  A.of = 0.f;
}
template <int M>
__device__ __forceinline__ void grad_acc_store(const GradAcc<M>& A, float4* __restrict__ myacc) {
  using G = Geo<M>;
  float acc[G::KP];
#pragma unroll
  for (int b = 0; b < G::KP; ++b) acc[b] = 0.f;
#pragma unroll
  for (int t = 0; t < (M - 1) / 2; ++t) { acc[2 * t] = pk_lo(A.e[t]); acc[2 * t + 1] = pk_hi(A.e[t]); }
  acc[M - 1] = A.el;
  if (GradAcc<M>::TWO) {
    acc[0] += A.of;
#pragma unroll
    for (int t = 0; t < (M - 1) / 2; ++t) { acc[2 * t + 1] += pk_lo(A.o[t]); acc[2 * t + 2] += pk_hi(A.o[t]); }
  }
#pragma unroll
  for (int q = 0; q < G::KP / 4; ++q)
    myacc[q] = make_float4(acc[4 * q], acc[4 * q + 1], acc[4 * q + 2], acc[4 * q + 3]);
}
// one 16-pixel chunk: wrow = the chunk of the weight tile, rrow = row i + a of the R tile at the chunk's first column
template <int M>
__device__ __forceinline__ void grad_chunk(GradAcc<M>& A, const float* __restrict__ wrow, const float* __restrict__ rrow) {
  using G = Geo<M>;
  float w[kP];
  f32x2 rp[G::RSEG / 2];
  const float4* w4 = reinterpret_cast<const float4*>(wrow);
#pragma unroll
  for (int q = 0; q < kP / 4; ++q) {
    const float4 v = w4[q];
    w[4 * q] = v.x; w[4 * q + 1] = v.y; w[4 * q + 2] = v.z; w[4 * q + 3] = v.w;
  }
  const ulonglong2* r2 = reinterpret_cast<const ulonglong2*>(rrow);
#pragma unroll
  for (int q = 0; q < G::RSEG / 4; ++q) {
    const ulonglong2 v = r2[q];
    rp[2 * q] = v.x; rp[2 * q + 1] = v.y;
  }
#pragma unroll
  for (int q = 0; q < kP; ++q) {
    const f32x2 ww = pk2(w[q], w[q]);
    if ((q & 1) == 0) {
#pragma unroll
      for (int t = 0; t < (M - 1) / 2; ++t) A.e[t] = fma2(ww, rp[q / 2 + t], A.e[t]);
      A.el = fmaf(w[q], pk_lo(rp[(q + M - 1) / 2]), A.el);
    } else if (GradAcc<M>::TWO) {
      A.of = fmaf(w[q], pk_hi(rp[(q - 1) / 2]), A.of);
#pragma unroll
      for (int t = 0; t < (M - 1) / 2; ++t) A.o[t] = fma2(ww, rp[(q + 1) / 2 + t], A.o[t]);
    } else {
#pragma unroll
      for (int t = 0; t < (M - 1) / 2; ++t) {       // r[q + 2t] = hi of pair (q + 2t - 1) / 2, r[q + 2t + 1] = lo of the next
        const float lo = fmaf(w[q], pk_hi(rp[(q - 1) / 2 + t]), pk_lo(A.e[t]));
        const float hi = fmaf(w[q], pk_lo(rp[(q + 1) / 2 + t]), pk_hi(A.e[t]));
        A.e[t] = pk2(lo, hi);
      }
      A.el = fmaf(w[q], pk_hi(rp[(q + M - 2) / 2]), A.el);
    }
  }
}

// FP64 fold of the thread-private FP32 gradient strips over the S pixel sub-sets: put(o, sum) for every kernel pixel
// o = a M + b, fixed order.  Called by all threads of the CTA (between barriers).  Small kernels have many sub-sets
// (S = 256 / M: 36 at m = 7, 85 at m = 3), so there four lanes share an output: quarter sums, then (q0 + q1) + (q2 + q3).
template <int M, typename F>
__device__ __forceinline__ void fold_strips(const float* __restrict__ accS, int tid, F&& put) {
  using G = Geo<M>;
  if (M * M * 4 <= kThreads) {
    const int o = tid >> 2, part = tid & 3;
    const bool live = o < M * M;
    const int a = live ? o / M : 0, b = live ? o - a * M : 0;
    constexpr int CH = (G::S + 3) / 4;
    const int s1 = min((part + 1) * CH, G::S);
    double s = 0.0;
#pragma unroll 1
    for (int ss = part * CH; ss < s1; ++ss) s += (double)accS[(ss * M + a) * G::KP + b];
    s += __shfl_xor_sync(0xffffffffu, s, 1);
    s += __shfl_xor_sync(0xffffffffu, s, 2);
    if (live && part == 0) put(o, s);
  } else {
    for (int o = tid; o < M * M; o += kThreads) {
      const int a = o / M, b = o - a * M;
      double s = 0.0;
#pragma unroll 1
      for (int ss = 0; ss < G::S; ++ss) s += (double)accS[(ss * M + a) * G::KP + b];
      put(o, s);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// the fused kernel
// ------------------------------------------------------------------------------------------------
template <int M, bool AUX, bool DIFF, bool KC = false>
__global__ void __launch_bounds__(kThreads, Geo<M>::CTAS) eval_kernel(const EvalParams p, const __grid_constant__ TensorMaps tm) {
  using G = Geo<M>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  // 128-byte aligned base (TMA destinations)
  unsigned char* sm = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  float* const Rbase = reinterpret_cast<float*>(sm + G::OFF_R);
  float* const Is = reinterpret_cast<float*>(sm + G::OFF_I);      // staged I tile (shifted by IOFF columns)
  float* const Ws = reinterpret_cast<float*>(sm + G::OFF_W);      // w = dL/dM tile
  float* const accS = reinterpret_cast<float*>(sm + G::OFF_ACC);
  float* const Ks = reinterpret_cast<float*>(sm + G::OFF_K);
  float* const Bs = reinterpret_cast<float*>(sm + G::OFF_BG);     // background coefficients of the current epoch
  double* const bgacc = reinterpret_cast<double*>(sm + G::OFF_BGACC) + (threadIdx.x >> 5) * kMaxBg;   // this warp's row
  const unsigned bar0 = smem_u32(sm + G::OFF_BAR);            // barR[0], barR[1], barI
  double* const red64 = reinterpret_cast<double*>(sm + G::OFF_BAR + 64);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n_tiles = p.tiles_x * p.tiles_y;
  const int vr = p.n_rows - M + 1, vc = p.n_cols - M + 1;
  const size_t npix = (size_t)p.n_rows * p.n_cols;

  if (tid == 0) {
    const unsigned cnt = p.use_tma ? 1u : (unsigned)kThreads;
#pragma unroll
    for (int b = 0; b < 3; ++b) mbar_init(bar0 + 8u * b, cnt);
    fence_mbar_init();
  }
  __syncthreads();

  // forward mapping: warp covers 32 px x 16 rows; lane -> (fx, fy) = (lane & 1, lane >> 1)
  const int f_col = (warp & 1) * 32 + (lane & 1) * kP;
  const int f_row = (warp >> 1) * 16 + (lane >> 1);
  // gradient mapping: consecutive threads own consecutive kernel rows a
  const int g_a = tid % M, g_s = tid / M;
  const bool g_active = g_s < G::S;
  float4* const myacc = reinterpret_cast<float4*>(accS + tid * G::KP);

  unsigned it = 0;                         // tiles this CTA has staged so far (mbarrier phase bookkeeping)
  auto Rbuf = [&](unsigned i) { return Rbase + (G::NRBUF == 2 ? (i & 1u) : 0u) * (G::R_STRIDE / 4); };
  auto barR = [&](unsigned i) { return bar0 + 8u * (G::NRBUF == 2 ? (i & 1u) : 0u); };
  const unsigned barI = bar0 + 16u;
  auto parR = [&](unsigned i) { return G::NRBUF == 2 ? ((i >> 1) & 1u) : (i & 1u); };
  auto parI = [&](unsigned i) { return i & 1u; };

  // Work items are (epoch, tile) pairs in epoch-major order, item g = j * n_tiles + t; this CTA takes items
  // blockIdx.x, blockIdx.x + gridDim.x, ...  (so a batch of many small images fills the grid as well as one
  // large image does).  Without the constant block j is the epoch itself and epochs whose `done` flag is set
  // are skipped; with it (KC) j runs over the active epochs listed there.
  // (j, t) are stepped with additions and compares only -- no division -- so that with the constant block they
  // stay in uniform registers and the constant-bank offset of the kernel row is a uniform value.
  const int n_act = KC ? c_blk.n_active : p.n_epochs;
  const int grid = (int)gridDim.x;
  const bool by_epoch = !KC && p.epoch_per_cta;
  const int ncols = by_epoch ? 1 : min(n_tiles, grid);   // CTAs (columns of partials) that contribute to one epoch
  auto step = [&](int& j, int& t) {          // the next item of this CTA
    if (by_epoch) {
      if (++t >= n_tiles) { t = 0; j += grid; }
    } else {
      t += grid;
      while (t >= n_tiles) { t -= n_tiles; ++j; }
    }
  };
  auto skip_done = [&](int& j, int& t) {     // ... that belongs to an epoch which is still being fitted
    if (!KC)
      while (j < n_act && p.done && p.done[j]) step(j, t);
  };

  float B0 = 0.f;
  int hx_off = -1, hx_m = 0, hx_n = 0;     // Hessian mode: X_q = Rs[pixel + hx_off], or eta^hx_m xi^hx_n if hx_off < 0
  double loss64 = 0.0, gb064 = 0.0, cnt64 = 0.0;   // DIFF: sum eps^2, sum eps, pixel count
  bool flushed = false;
  int since_flush = 0, cur_j = -1;
  double* out = nullptr;                   // element o of this CTA's partial column at out[o * ncols]

  // fold the FP32 strips of all pixel sub-sets into this CTA's FP64 partials, fixed order
  auto flush = [&]() {
    __syncthreads();
    fold_strips<M>(accS, tid, [&](int o, double s) { out[(size_t)o * ncols] = flushed ? out[(size_t)o * ncols] + s : s; });
    __syncthreads();
#pragma unroll
    for (int q = 0; q < G::KP / 4; ++q) myacc[q] = make_float4(0.f, 0.f, 0.f, 0.f);
    flushed = true;
    since_flush = 0;
  };
  // per-epoch block partials: gradient strips, then g_B0 and the loss
  auto finish_epoch = [&]() {
    if (DIFF) {                            // rows: sum eps, sum eps^2, count
      __syncthreads();
      const double l = warp_sum_f64(loss64), g0 = warp_sum_f64(gb064), c0 = warp_sum_f64(cnt64);
      if (lane == 0) { red64[warp] = l; red64[8 + warp] = g0; bgacc[0] = c0; }
      __syncthreads();
      if (tid == 0) {
        double ls = 0.0, gs = 0.0, cs = 0.0;
        const double* all = reinterpret_cast<const double*>(sm + G::OFF_BGACC);
        for (int w = 0; w < kThreads / 32; ++w) { ls += red64[w]; gs += red64[8 + w]; cs += all[w * kMaxBg]; }
        out[0] = gs;  out[(size_t)ncols] = ls;  out[(size_t)2 * ncols] = cs;
      }
      __syncthreads();
      return;
    }
    flush();                               // ends with a barrier after the last reads of accS
    const double l = warp_sum_f64(loss64), g0 = warp_sum_f64(gb064);
    if (lane == 0) { red64[warp] = l; red64[8 + warp] = g0; }
    __syncthreads();
    if (tid == 0) {
      double ls = 0.0, gs = 0.0;
      for (int w = 0; w < kThreads / 32; ++w) { ls += red64[w]; gs += red64[8 + w]; }
      out[(size_t)(M * M) * ncols] = gs;
      out[(size_t)p.np * ncols] = ls;
      // background coefficients beyond b_00: warp rows in fixed order
      const double* all = reinterpret_cast<const double*>(sm + G::OFF_BGACC);
      for (int t = 1; t < p.np - M * M; ++t) {
        double sacc = 0.0;
        for (int w = 0; w < kThreads / 32; ++w) sacc += all[w * kMaxBg + t];
        out[(size_t)(M * M + t) * ncols] = sacc;
      }
    }
    __syncthreads();                       // red64 / Ks / accS free for the next epoch
  };

  int j = 0, t = (int)blockIdx.x - grid;
  if (by_epoch) { j = (int)blockIdx.x; t = 0; }
  else step(j, t);                           // first item: t = blockIdx.x, wrapped into (j, t)
  skip_done(j, t);
  if (j < n_act) {
    const int e0 = KC ? c_blk.active[j] : j;
    stage_R<M>(p, tm, e0, t, smem_u32(Rbuf(it)), barR(it));
    stage_I<M>(p, tm, e0, t, smem_u32(Is), barI);
  }
  while (j < n_act) {
    const int e = KC ? c_blk.active[j] : j;
    int jn = j, tn = t;
    step(jn, tn);
    skip_done(jn, tn);
    const bool more = jn < n_act;
    const int en = (KC && more) ? c_blk.active[jn] : jn;
    if (j != cur_j) {                      // first tile of an epoch for this CTA
      if (cur_j >= 0) finish_epoch();
      cur_j = j;
      const bool hess = AUX && p.hess_q0 >= 0;
      const float* __restrict__ th = p.theta + (hess ? (size_t)0 : (size_t)e * p.np);
      if (hess) {                          // design-vector component of this Hessian row
        const int hq = p.hess_q0 + e;
        hx_off = -1; hx_m = 0; hx_n = 0;
        if (hq < M * M) {
          hx_off = (hq / M) * G::RPITCH + (hq % M);
        } else {
          int tq = M * M;
          for (int mm = 0; mm <= p.bg_degree; ++mm)
            for (int nn = 0; nn <= p.bg_degree - mm; ++nn, ++tq)
              if (tq == hq) { hx_m = mm; hx_n = nn; }
        }
      }
      if (!KC) {
        for (int idx = tid; idx < G::K_FLOATS; idx += kThreads) {
          const int a = idx / G::KP, b = idx - a * G::KP;
          Ks[idx] = (b < M) ? th[a * M + b] : 0.f;
        }
      }
      B0 = th[M * M];
      if (tid < kMaxBg) Bs[tid] = (tid < p.np - M * M) ? th[M * M + tid] : 0.f;
      if (lane < kMaxBg) bgacc[lane] = 0.0;
#pragma unroll
      for (int q = 0; q < G::KP / 4; ++q) myacc[q] = make_float4(0.f, 0.f, 0.f, 0.f);
      loss64 = 0.0; gb064 = 0.0; cnt64 = 0.0; flushed = false; since_flush = 0;
      // column of this CTA in epoch e: the local index (mod grid) of the tiles it owns there
      int col = by_epoch ? 0 : ((int)blockIdx.x - (int)(((long long)j * n_tiles) % grid) + grid) % grid;
      out = p.partials + ((size_t)e * p.part_rows) * ncols + col;
      __syncthreads();                     // Ks visible
    }
    const int tile_y = t / p.tiles_x, tile_x = t - tile_y * p.tiles_x;
    const float* __restrict__ Rs = Rbuf(it);
    mbar_wait(barR(it), parR(it));
    mbar_wait(barI, parI(it));

    // ------------------------------------------------------------------ forward
    {
      float tot[kP];
      // broadcast from lane 0: tells the compiler the constant-bank offset is warp-uniform (uniform registers)
      forward_strip<M, KC>(Ks, j * G::K_FLOATS, Rs + f_row * G::RPITCH + f_col, B0, tot);
      const int iy = tile_y * kTH + f_row, ix0 = tile_x * kTW + f_col;
      const float* irow = Is + f_row * kIPitch + f_col;
      float* wrow = Ws + f_row * kIPitch + f_col;
      float lsum, wsum, Sp[4];
      const bool edge = (tile_y * kTH + kTH > vr) || (tile_x * kTW + kTW > vc);
      if (DIFF) {
        float s_eps, s_eps2, s_cnt;
        add_background<M>(p, Bs, iy, ix0, tot);
        if (edge) strip_diff<M, true>(p, e, npix, iy, ix0, vr, vc, tot, irow, s_eps, s_eps2, s_cnt);
        else strip_diff<M, false>(p, e, npix, iy, ix0, vr, vc, tot, irow, s_eps, s_eps2, s_cnt);
        gb064 += (double)s_eps;  loss64 += (double)s_eps2;  cnt64 += (double)s_cnt;
      } else {
      const float* xrow = (AUX && hx_off >= 0) ? Rs + f_row * G::RPITCH + f_col + hx_off : nullptr;
      if (edge) strip_epilogue<M, AUX, true>(p, e, npix, iy, ix0, vr, vc, tot, irow, wrow, Bs, lsum, wsum, Sp, xrow, hx_m, hx_n);
      else strip_epilogue<M, AUX, false>(p, e, npix, iy, ix0, vr, vc, tot, irow, wrow, Bs, lsum, wsum, Sp, xrow, hx_m, hx_n);
      loss64 += (double)lsum;
      gb064 += (double)wsum;
      }
      if (!DIFF && p.bg_degree > 0) {               // dL/db_mn = sum w eta^m xi^n: strip sums -> warp sum -> this warp's FP64 row
        const float xi = ((float)(iy + G::H) - p.bg_yc) * p.bg_inv_ny;
        int tt = 0;
#pragma unroll
        for (int mm = 0; mm < 4; ++mm) {
          float term = Sp[mm];
#pragma unroll
          for (int nn = 0; nn < 4; ++nn) {
            if (mm <= p.bg_degree && nn <= p.bg_degree - mm) {       // CTA-uniform
              float v = term;
#pragma unroll
              for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
              if (lane == 0 && tt > 0) bgacc[tt] += (double)v;
              ++tt;
            }
            term *= xi;
          }
        }
      }
    }
    __syncthreads();                       // (A) w tile complete, I tile consumed
    if (more) {
      stage_I<M>(p, tm, en, tn, smem_u32(Is), barI);
      if (G::NRBUF == 2) stage_R<M>(p, tm, en, tn, smem_u32(Rbuf(it + 1)), barR(it + 1));
    }

    // ------------------------------------------------------------------ gradient
    if (!DIFF && g_active) {
      GradAcc<M> A;
      grad_acc_load<M>(A, myacc);
      const int rows_here = min(kTH, vr - tile_y * kTH);
      const int n_items = rows_here * (kTW / kP);
#pragma unroll 1
      for (int item = g_s; item < n_items; item += G::S) {
        const int i = item / (kTW / kP), c = item - i * (kTW / kP);
        grad_chunk<M>(A, Ws + i * kIPitch + c * kP, Rs + (i + g_a) * G::RPITCH + c * kP);
      }
      grad_acc_store<M>(A, myacc);
    }
    __syncthreads();                       // (B) everyone is done reading this w tile and R buffer
    if (G::NRBUF == 1 && more) stage_R<M>(p, tm, en, tn, smem_u32(Rbuf(it + 1)), barR(it + 1));
    if (!DIFF && ++since_flush == p.flush_tiles && more && jn == j) flush();
    j = jn;
    t = tn;
    ++it;
  }
  if (cur_j >= 0) finish_epoch();
}

// ------------------------------------------------------------------------------------------------
// Hessian block kernel (dia_hessian): rows hess_q0 .. hess_q0 + n_epochs - 1 (all of them
// kernel-pixel rows, q < M*M) of the kernel-kernel block of H for one target, H[q][o] = sum_V h X_q X_o.
// Per tile the model and h = d^2 l / dM^2 are computed ONCE (forward stencil + epilogue, as in eval_kernel's
// Hessian mode with X_q = 1); then for every row q the weight tile h X_q -- X_q is the reference pixel shifted by
// row q's kernel position, read from the staged R tile -- is correlated against the R tile exactly as in the gradient
// phase of eval_kernel, and the FP32 strips are folded into this CTA's FP64 partial column of row q.  A launch of 32
// rows therefore costs 1 forward + 32 gradient passes per tile instead of 32 + 32.  Tiles are staged by cp.async
// (single buffer: staging is < 1 % of 33 passes).  Columns M*M.. of the partials (background terms, loss) are written
// as zeros; the host fills those entries of H from the background rows by symmetry.
// ------------------------------------------------------------------------------------------------
template <int M>
__global__ void __launch_bounds__(kThreads, Geo<M>::CTAS) hess_block_kernel(const EvalParams p) {
  using G = Geo<M>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned char* sm = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  float* const Rs = reinterpret_cast<float*>(sm + G::OFF_R);
  float* const Is = reinterpret_cast<float*>(sm + G::OFF_I);      // I tile during the forward phase, then h X_q
  float* const Hs = reinterpret_cast<float*>(sm + G::OFF_W);      // h tile
  float* const accS = reinterpret_cast<float*>(sm + G::OFF_ACC);
  float* const Ks = reinterpret_cast<float*>(sm + G::OFF_K);
  float* const Bs = reinterpret_cast<float*>(sm + G::OFF_BG);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n_tiles = p.tiles_x * p.tiles_y;
  const int vr = p.n_rows - M + 1, vc = p.n_cols - M + 1;
  const size_t npix = (size_t)p.n_rows * p.n_cols;
  const int f_col = (warp & 1) * 32 + (lane & 1) * kP;
  const int f_row = (warp >> 1) * 16 + (lane >> 1);
  const int g_a = tid % M, g_s = tid / M;
  const bool g_active = g_s < G::S;
  float4* const myacc = reinterpret_cast<float4*>(accS + tid * G::KP);
  const int grid = (int)gridDim.x, ncols = grid;      // the host launches min(resident CTAs, tiles) CTAs

  for (int idx = tid; idx < G::K_FLOATS; idx += kThreads) {
    const int a = idx / G::KP, b = idx - a * G::KP;
    Ks[idx] = (b < M) ? p.theta[a * M + b] : 0.f;
  }
  const float B0 = p.theta[M * M];
  if (tid < kMaxBg) Bs[tid] = (tid < p.np - M * M) ? p.theta[M * M + tid] : 0.f;
  __syncthreads();

  bool first = true;
  for (int t = (int)blockIdx.x; t < n_tiles; t += grid) {
    const int tile_y = t / p.tiles_x, tile_x = t - tile_y * p.tiles_x;
    stage_tile_cp_async<G::RH, G::RPITCH>(p.R, p.n_rows, p.n_cols, p.cp8, tile_y * kTH, tile_x * kTW, smem_u32(Rs));
    stage_tile_cp_async<kTH, kIPitch>(p.I, p.n_rows, p.n_cols, p.cp8, tile_y * kTH + G::H, tile_x * kTW + G::H - G::IOFF,
                                      smem_u32(Is));
    asm volatile("cp.async.wait_all;\n" ::: "memory");
    __syncthreads();
    {                                        // forward: h tile
      float tot[kP];
      forward_strip<M, false>(Ks, 0, Rs + f_row * G::RPITCH + f_col, B0, tot);
      const int iy = tile_y * kTH + f_row, ix0 = tile_x * kTW + f_col;
      const float* irow = Is + f_row * kIPitch + f_col;
      float* hrow = Hs + f_row * kIPitch + f_col;
      float lsum, wsum, Sp[4];
      const bool edge = (tile_y * kTH + kTH > vr) || (tile_x * kTW + kTW > vc);
      if (edge) strip_epilogue<M, true, true>(p, 0, npix, iy, ix0, vr, vc, tot, irow, hrow, Bs, lsum, wsum, Sp, nullptr, 0, 0);
      else strip_epilogue<M, true, false>(p, 0, npix, iy, ix0, vr, vc, tot, irow, hrow, Bs, lsum, wsum, Sp, nullptr, 0, 0);
    }
    __syncthreads();                         // h tile complete, I tile consumed
    const int rows_here = min(kTH, vr - tile_y * kTH);
    const int n_items = rows_here * (kTW / kP);
#pragma unroll 1
    for (int jq = 0; jq < p.n_epochs; ++jq) {
      const int q = p.hess_q0 + jq;
      const int aq = q / M, bq = q - aq * M;
      {                                      // weight tile of row q: h X_q, this thread's forward strip
        const float* xr = Rs + (f_row + aq) * G::RPITCH + f_col + bq;
        const float4* h4 = reinterpret_cast<const float4*>(Hs + f_row * kIPitch + f_col);
        float4* w4 = reinterpret_cast<float4*>(Is + f_row * kIPitch + f_col);
#pragma unroll
        for (int c = 0; c < kP / 4; ++c) {
          float4 v = h4[c];
          v.x *= xr[4 * c]; v.y *= xr[4 * c + 1]; v.z *= xr[4 * c + 2]; v.w *= xr[4 * c + 3];
          w4[c] = v;
        }
      }
      __syncthreads();
      if (g_active) {                        // the gradient phase of eval_kernel on this weight tile
        GradAcc<M> A;
        grad_acc_zero<M>(A);
#pragma unroll 1
        for (int item = g_s; item < n_items; item += G::S) {
          const int i = item / (kTW / kP), c = item - i * (kTW / kP);
          grad_chunk<M>(A, Is + i * kIPitch + c * kP, Rs + (i + g_a) * G::RPITCH + c * kP);
        }
        grad_acc_store<M>(A, myacc);
      }
      __syncthreads();
      double* outp = p.partials + ((size_t)jq * p.part_rows) * ncols + blockIdx.x;
      for (int o = tid; o < M * M; o += kThreads) {
        const int a = o / M, b = o - a * M;
        double sacc = 0.0;
#pragma unroll 1
        for (int ss = 0; ss < G::S; ++ss) sacc += (double)accS[(ss * M + a) * G::KP + b];
        outp[(size_t)o * ncols] = first ? sacc : outp[(size_t)o * ncols] + sacc;
      }
      if (first && tid < p.part_rows - M * M) outp[(size_t)(M * M + tid) * ncols] = 0.0;
      __syncthreads();                       // strips and weight tile free for the next row
    }
    first = false;
  }
}

#ifndef DIA_INST_M      // the small stand-alone kernels belong to the API translation unit only
// Fixed-order sum of one row of block partials by one warp: lane l adds columns l, l+32, ... in order,
// then the 32 lane sums are combined by a fixed butterfly -- deterministic for a given n_blocks.
__device__ __forceinline__ double warp_row_sum(const double* __restrict__ row, int n_blocks, int lane) {
  double s = 0.0;
  for (int b = lane; b < n_blocks; b += 32) s += row[b];
  return warp_sum_f64(s);
}

// Second level: one warp per output sums the block partials (fixed order => deterministic).
__global__ void reduce_partials_kernel(const double* __restrict__ partials, int n_blocks, int np1,
                                       const int* __restrict__ done, double* __restrict__ loss,
                                       double* __restrict__ grad) {
  const int e = blockIdx.y;
  if (done && done[e]) return;
  const int lane = threadIdx.x & 31;
  const int o = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (o >= np1) return;
  const double s = warp_row_sum(partials + ((size_t)e * np1 + o) * n_blocks, n_blocks, lane);
  if (lane == 0) {
    if (o == np1 - 1) loss[e] = s;
    else grad[(size_t)e * (np1 - 1) + o] = s;
  }
}

// Fit-quality metrics from the difference-image partial sums (Eq. 29-30): one warp per epoch.
// metrics[e] = { N_used, MFB = sum eps / N, MFV = sum (eps - MFB)^2 / (N - 1), chi^2 = sum eps^2 }.
__global__ void diff_metrics_kernel(const double* __restrict__ partials, int n_blocks, double* __restrict__ metrics) {
  const int e = blockIdx.x, lane = threadIdx.x & 31;
  const double* rows = partials + (size_t)e * 3 * n_blocks;
  const double s1 = warp_row_sum(rows, n_blocks, lane);
  const double s2 = warp_row_sum(rows + n_blocks, n_blocks, lane);
  const double cn = warp_row_sum(rows + 2 * (size_t)n_blocks, n_blocks, lane);
  if (lane == 0) {
    const double mfb = cn > 0.0 ? s1 / cn : 0.0;
    metrics[4 * e + 0] = cn;
    metrics[4 * e + 1] = mfb;
    metrics[4 * e + 2] = cn > 1.0 ? (s2 - cn * mfb * mfb) / (cn - 1.0) : 0.0;
    metrics[4 * e + 3] = s2;
  }
}

// Fills the staging copy of ConstBlock: the list of active epochs (done flag clear) and their kernel pixels
// as padded rows [j][m][kp].  One CTA; the list is built by thread 0 in epoch order.
__global__ void pack_const_kernel(const float* __restrict__ theta, const int* __restrict__ done, int n_epochs,
                                  int np, int m, int kp, ConstBlock* __restrict__ dst) {
  __shared__ int s_n, s_active[kConstEpochs];
  if (threadIdx.x == 0) {
    int n = 0;
    for (int e = 0; e < n_epochs; ++e)
      if (!(done && done[e])) s_active[n++] = e;
    s_n = n;
    dst->n_active = n;
  }
  __syncthreads();
  for (int j = threadIdx.x; j < s_n; j += blockDim.x) dst->active[j] = s_active[j];
  const int per = m * kp;
  for (int idx = threadIdx.x; idx < s_n * per; idx += blockDim.x) {
    const int j = idx / per, r = idx - j * per, a = r / kp, b = r - a * kp;
    dst->K[idx] = (b < m) ? theta[(size_t)s_active[j] * np + a * m + b] : 0.f;
  }
}

#endif  // DIA_INST_M

}  // namespace dia
