// dia_hess_tc.cuh -- the kernel-kernel block of the Hessian on the tensor cores (dia_hessian).
//
// H[p][q] = sum_V h X_p X_q (Eq. 15; closed form D3 of DESIGN.md section 3) is a dense contraction
// over the pixels: with the im2col matrix X [pixels][m^2] (X_p of pixel (i, j) is the reference pixel shifted by
// kernel position p) it is X' diag(h) X, the one GEMM-shaped step of the path.  Here
//   * h = s_+^2 - s_-^2 with s_+- = sqrt(max(+-h, 0)), so that H = B_+' B_+ - B_-' B_- with B = diag(s) X: ONE operand
//     matrix serves both sides of the product (rows of negative h -- Huber's linear branch, gross outliers -- take a
//     second pass with the A operand negated; it runs only for tile rows that have such a pixel);
//   * every float32 element of B is split into two float16 numbers, hi with 8 significant bits and lo = x - hi with 11
//     (|x - hi - lo| <= 2^-20 |x|; a bfloat16 pair's 2^-17 was measured to leave e_H at 1 - 2e-6 on small images), and
//     the product is the four tcgen05.mma terms lo lo + lo hi + hi lo + hi hi, accumulated in float32 in TMEM.  The
//     widths follow from the accumulator's arithmetic (next item): hi hi products are 16 bits wide and stay exact
//     under a 64-pixel sum, the small terms go first while the accumulator is small.  Measured mean bias of the sums
//     against hi width: 11 bits (three terms) -2.1e-7, 10 bits -1.3e-7, 9 bits -7.5e-8, 8 bits -5.0e-8, 7 bits -4.4e-8
//     (narrower hi parts raise the random error of small images instead; profiles/r02_tc_hessian.md).  float16 has a narrow
//     exponent range, so B is scaled per tile by a power of two c with max s * max |R| * c < 2^15 (no overflow; elements
//     below 2^-39 of the largest lose precision, which no sum can see) and the tile's sums are multiplied by c^-2
//     when they are folded to FP64;
//   * the tensor core adds every product to the accumulator after aligning it to the larger exponent and TRUNCATING
//     below 2^-25 of it (measured, profiles/r02_tc_hessian.md): a chain of n pixels loses ~5e-9 n of the sum,
//     systematically.  So a chain is ONE TILE ROW (64 pixels, four k-steps, bias 3e-7); after it the accumulator
//     block is read back (tcgen05.ld) and added, round-to-nearest, to float32 registers that cover one 64 x 64 tile,
//     and those are folded into this CTA's FP64 partial block per tile -- the FP64 order is fixed, the result is
//     deterministic.
// The background rows (X = eta^m xi^n of Eq. 18-19, X = 1 for B0) are rows m^2 .. np - 1 of the same operand matrix, so
// the whole of H comes from this one contraction and every entry carries the same (tiny) accumulator bias.
// Operand row (slot) t of group g holds parameter perm[128 g + t] (hess_tc_make_perm): the slots are dealt so that the
// 32 rows of a warp read 32 different shared-memory banks of the staged R tile when they build their operand rows
// (in parameter order lanes 0 / 1 and 30 / 31 of most warps collide: 39 % of the wavefronts, ncu).
// The 128-slot groups g = 0 .. ceil(np / 128) - 1 give blocks (gi, gj) of H; by symmetry only
// gi <= gj are computed.  A CTA has one TYPE for its whole life (HessTcTypes): an operand tile of two row groups
// [g0 | g1], an A operand (one of the two: 128 rows of D in TMEM lanes) and a B operand of one or two groups
// (N = 128 or 256 columns of D), i.e. a diagonal block paired with an off-diagonal block that shares its rows, or a
// single block.  CTAs of one type share the tiles of the image round robin.
// Per tile: stage R (+ halo) and I, forward stencil and the per-pixel h exactly as hess_block_kernel (same device
// functions), the split into s_+ and s_-; then per tile row a software pipeline of
//   build   thread t owns operand row t (kernel position (a, b)): 64 products s[j] R[i+a][j+b], hi / lo split, into
//           the K-major no-swizzle core-matrix layout (8 rows x 16 bytes) of shared-memory buffer st % 2,
//   issue   one thread: 4 terms x 4 k-steps of tcgen05.mma (M = 128, N = 128 | 256, K = 16) into TMEM buffer
//           row % 2, tcgen05.commit to the buffer's mbarrier,
//   flush   of the PREVIOUS row's accumulators into the registers while these MMAs run.
#pragma once
#include <cuda_fp16.h>

#include "dia_eval.cuh"

namespace dia {

constexpr int kTcMaxTypes = 160;
constexpr int kTcRows = 256;                 // rows of an operand tile (two groups of 128 kernel positions)
constexpr int kTcGroup = 128;
struct HessTcTypes {
  int n_types, ctas_per_type;
  unsigned char g0[kTcMaxTypes], g1[kTcMaxTypes];   // row groups held by the operand tile (g1 = 255: none)
  unsigned char a_sel[kTcMaxTypes];                 // which of the two is the A operand (rows of D)
  unsigned char b_start[kTcMaxTypes];               // first group of the B operand
  unsigned char n_groups[kTcMaxTypes];              // groups of the B operand: 1 (N = 128) or 2 (N = 256)
};

template <int M>
struct TcGeo {
  using G = Geo<M>;
  static constexpr int OFF_R = 0;
  static constexpr int OFF_I = G::R_STRIDE;                       // I tile, then s_- = sqrt(max(-h, 0))
  static constexpr int OFF_W = OFF_I + G::I_STRIDE;               // h tile, then s_+ = sqrt(max(h, 0))
  static constexpr int OFF_K = OFF_W + G::I_STRIDE;
  static constexpr int OFF_BG = OFF_K + 4 * G::K_FLOATS;
  static constexpr int OFF_FLAG = round_up(OFF_BG + 4 * kMaxBg, 16);     // per tile row: has a pixel of negative h
  static constexpr int OFF_BAR = OFF_FLAG + 4 * kTH;              // two mbarriers, the TMEM base address
  static constexpr int OFF_RED = OFF_BAR + 32;                    // per-warp maxima of s and |R| (scale of the tile)
  static constexpr int OFF_POW = OFF_RED + 4 * 2 * (kThreads / 32);   // eta^k per tile column, xi^k per tile row, k = 0..3
  static constexpr int OFF_OP = round_up(OFF_POW + 4 * 2 * 4 * kTW, 128);
  static constexpr int OP_TILE = kTcRows * kTW * 2;               // hi or lo: 256 rows x 64 pixels of float16
  static constexpr int OP_BUF = 2 * OP_TILE;                      // hi, lo
  static constexpr int LBO = kTcRows / 8 * 128;                   // bytes between core matrices adjacent in K
  static constexpr int SBO = 128;                                 // ... adjacent in the row direction
  static constexpr size_t SMEM = OFF_OP + 2 * OP_BUF + 128;
  static constexpr bool FITS = SMEM <= 227 * 1024;
};

__device__ __forceinline__ unsigned long long tc_smem_desc(unsigned saddr, unsigned lbo, unsigned sbo) {
  // matrix descriptor: start address [0,14), leading byte offset [16,30), stride byte offset [32,46) (all >> 4),
  // version 1 at [46,48), no swizzle
  return (unsigned long long)((saddr >> 4) & 0x3FFFu) | ((unsigned long long)((lbo >> 4) & 0x3FFFu) << 16) |
         ((unsigned long long)((sbo >> 4) & 0x3FFFu) << 32) | (1ull << 46);
}
__device__ __forceinline__ void tc_mma_f16(unsigned tmem_d, unsigned long long ad, unsigned long long bd, unsigned idesc,
                                            unsigned accumulate) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}\n" ::"r"(tmem_d),
      "l"(ad), "l"(bd), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tc_commit(unsigned bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); }

// adds 32 accumulator columns (this warp's 32 lanes) to acc[0..31]
__device__ __forceinline__ void tc_flush32(unsigned taddr, float* acc) {
  unsigned v[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, "
      "%18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
        "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
        "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
#pragma unroll
  for (int j = 0; j < 32; ++j) acc[j] += __uint_as_float(v[j]);
}

// one operand row of one tile row: 64 products s[j] r[j], split into float16 hi + lo, 8 pixels (16 bytes) per store
template <bool SCALED>
__device__ __forceinline__ void tc_build_row(unsigned char* __restrict__ op_hi, unsigned char* __restrict__ op_lo, int lbo,
                                             const float* __restrict__ r, const float* __restrict__ s, float f = 1.f) {
#pragma unroll
  for (int kg = 0; kg < kTW / 8; ++kg) {
    const float4 s0 = reinterpret_cast<const float4*>(s)[2 * kg], s1 = reinterpret_cast<const float4*>(s)[2 * kg + 1];
    const float sv[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
    unsigned hi[4], lo[4];
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      float p0 = r[8 * kg + 2 * t] * sv[2 * t], p1 = r[8 * kg + 2 * t + 1] * sv[2 * t + 1];
      if (SCALED) { p0 *= f;  p1 *= f; }
      __half2 h = __floats2half2_rn(p0, p1);                                         // .x (low half) = p0
#ifndef DIA_TC_HI_DROP
#define DIA_TC_HI_DROP 3
#endif
      constexpr unsigned kHalf = (1u << (DIA_TC_HI_DROP - 1)) * 0x00010001u, kMask = ~(((1u << DIA_TC_HI_DROP) - 1u) * 0x00010001u);
      const unsigned hb = (*reinterpret_cast<const unsigned*>(&h) + kHalf) & kMask;                // 11 -> 8 significant bits, round to nearest
      h = *reinterpret_cast<const __half2*>(&hb);
      const __half2 l = __floats2half2_rn(p0 - __low2float(h), p1 - __high2float(h));
      hi[t] = *reinterpret_cast<const unsigned*>(&h);
      lo[t] = *reinterpret_cast<const unsigned*>(&l);
    }
    *reinterpret_cast<uint4*>(op_hi + kg * lbo) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4*>(op_lo + kg * lbo) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
  }
}

#ifdef DIA_TC_PROFILE
__device__ long long g_tc_prof[16];
#define TC_T(k) do { if (blockIdx.x == 0 && threadIdx.x == 32) { const long long t_ = clock64(); g_tc_prof[k] += t_ - tc_t0; tc_t0 = t_; } } while (0)
#else
#define TC_T(k) do { } while (0)
#endif

template <int M>
__global__ void __launch_bounds__(kThreads, 1) hess_tc_kernel(const EvalParams p, double* __restrict__ partials,
                                                              const short* __restrict__ perm,
                                                              const __grid_constant__ HessTcTypes ty) {
  using G = Geo<M>;
  using T = TcGeo<M>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned char* sm = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  float* const Rs = reinterpret_cast<float*>(sm + T::OFF_R);
  float* const Is = reinterpret_cast<float*>(sm + T::OFF_I);
  float* const Hs = reinterpret_cast<float*>(sm + T::OFF_W);
  float* const Ks = reinterpret_cast<float*>(sm + T::OFF_K);
  float* const Bs = reinterpret_cast<float*>(sm + T::OFF_BG);
  int* const rowneg = reinterpret_cast<int*>(sm + T::OFF_FLAG);
  float* const red = reinterpret_cast<float*>(sm + T::OFF_RED);
  float* const etapow = reinterpret_cast<float*>(sm + T::OFF_POW);          // [4][kTW]
  float* const xipow = etapow + 4 * kTW;                                    // [4][kTH]
  const unsigned bar0 = smem_u32(sm + T::OFF_BAR);
  unsigned* const tmem_slot = reinterpret_cast<unsigned*>(sm + T::OFF_BAR + 16);
  unsigned char* const ops = sm + T::OFF_OP;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n_tiles = p.tiles_x * p.tiles_y;
  const int vr = p.n_rows - M + 1, vc = p.n_cols - M + 1;
  const size_t npix = (size_t)p.n_rows * p.n_cols;
  const int f_col = (warp & 1) * 32 + (lane & 1) * kP;
  const int f_row = (warp >> 1) * 16 + (lane >> 1);

  // this CTA's type, this thread's operand row
  const int type = (int)blockIdx.x % ty.n_types, cidx = (int)blockIdx.x / ty.n_types;
  const int g0 = ty.g0[type], g1 = ty.g1[type];
  const int a_sel = ty.a_sel[type], b_start = ty.b_start[type], n_groups = ty.n_groups[type];
  const int my_g = (tid >> 7) ? g1 : g0;
  const int my_q = my_g != 255 ? (int)perm[my_g * kTcGroup + (tid & (kTcGroup - 1))] : -1;
  const bool my_valid = my_q >= 0;
  const bool my_bg = my_valid && my_q >= M * M;                 // a background row: X = eta^bg_m xi^bg_n
  const int my_a = (my_valid && !my_bg) ? my_q / M : 0, my_b = (my_valid && !my_bg) ? my_q - (my_q / M) * M : 0;
  int bg_m = 0, bg_n = 0;
  if (my_bg) {
    int tq = M * M;
    for (int mm = 0; mm <= p.bg_degree; ++mm)
      for (int nn = 0; nn <= p.bg_degree - mm; ++nn, ++tq)
        if (tq == my_q) { bg_m = mm; bg_n = nn; }
  }
  const unsigned my_off = (unsigned)((tid >> 3) * 128 + (tid & 7) * 16);    // row tid of a core-matrix column

  for (int idx = tid; idx < G::K_FLOATS; idx += kThreads) {
    const int a = idx / G::KP, b = idx - a * G::KP;
    Ks[idx] = (b < M) ? p.theta[a * M + b] : 0.f;
  }
  const float B0 = p.theta[M * M];
  if (tid < kMaxBg) Bs[tid] = (tid < p.np - M * M) ? p.theta[M * M + tid] : 0.f;
  for (int idx = tid; idx < 2 * T::OP_BUF / 16; idx += kThreads)          // rows beyond m^2 stay zero
    reinterpret_cast<uint4*>(ops)[idx] = make_uint4(0u, 0u, 0u, 0u);
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(tmem_slot)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
  }
  if (tid == 0) {
    mbar_init(bar0, 1u);
    mbar_init(bar0 + 8u, 1u);
    fence_mbar_init();
  }
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const unsigned tmem = *tmem_slot;

  // instruction descriptor: D float32, A and B float16 (format 0), both K-major, M = 128, N = 128 n_groups
  const unsigned idesc = (1u << 4) | ((unsigned)(kTcGroup * n_groups >> 3) << 17) | ((128u >> 4) << 24);
  const int ncol = kTcGroup * n_groups / 2;                     // accumulator columns per thread (two warps per lane quarter)
  const unsigned my_taddr = tmem + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)((warp >> 2) * ncol);

  float acc[kTcGroup];
#pragma unroll
  for (int c = 0; c < kTcGroup; ++c) acc[c] = 0.f;
  unsigned gst = 0, grow = 0;                                   // stages and tile rows so far (mbarrier / TMEM buffer bookkeeping)
  bool first_tile = true;
  double* const outp = partials + (size_t)blockIdx.x * (kTcRows * kTcGroup);

#ifdef DIA_TC_PROFILE
  long long tc_t0 = clock64();
#endif
  for (int t = cidx; t < n_tiles; t += ty.ctas_per_type) {
    const int tile_y = t / p.tiles_x, tile_x = t - tile_y * p.tiles_x;
    stage_tile_cp_async<G::RH, G::RPITCH>(p.R, p.n_rows, p.n_cols, p.cp8, tile_y * kTH, tile_x * kTW, smem_u32(Rs));
    stage_tile_cp_async<kTH, kIPitch>(p.I, p.n_rows, p.n_cols, p.cp8, tile_y * kTH + G::H, tile_x * kTW + G::H - G::IOFF,
                                      smem_u32(Is));
    if (tid < kTH) rowneg[tid] = 0;
    if (tid < 2 * kTW) {                     // powers of the background coordinates (as strip_epilogue forms them)
      const int j = tid & (kTW - 1);
      const float v = tid < kTW ? fmaf((float)j, p.bg_inv_nx, ((float)(tile_x * kTW + G::H) - p.bg_xc) * p.bg_inv_nx)
                                : ((float)(tile_y * kTH + j + G::H) - p.bg_yc) * p.bg_inv_ny;
      float* dst = (tid < kTW ? etapow : xipow) + j;
      float pw = 1.f;
#pragma unroll
      for (int k = 0; k < 4; ++k) { dst[k * kTW] = pw;  pw *= v; }
    }
    asm volatile("cp.async.wait_all;\n" ::: "memory");
    __syncthreads();
    {                                        // forward: h tile (hess_block_kernel's forward phase)
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
    double inv_c2;                           // c^-2 of this tile's power-of-two scale
    {                                        // h -> c s_+ (in place), c s_- (over the I tile), row flags
      const int r = tid >> 2, c0 = (tid & 3) * 16;
      float4* hp = reinterpret_cast<float4*>(Hs + r * kIPitch + c0);
      float4* np_ = reinterpret_cast<float4*>(Is + r * kIPitch + c0);
      float sp[16], sn[16];
      float smax = 0.f, rmax = 0.f;
      bool neg = false;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const float4 h = hp[c];
        const float hv[4] = {h.x, h.y, h.z, h.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          neg = neg || hv[k] < 0.f;
          sp[4 * c + k] = sqrtf(fmaxf(hv[k], 0.f));
          sn[4 * c + k] = sqrtf(fmaxf(-hv[k], 0.f));
          smax = fmaxf(smax, fmaxf(sp[4 * c + k], sn[4 * c + k]));
        }
      }
      if (neg) rowneg[r] = 1;
      rmax = 1.f;                            // the background rows: |eta^m xi^n| <= 1
      for (int idx = tid; idx < G::R_FLOATS; idx += kThreads) rmax = fmaxf(rmax, fabsf(Rs[idx]));
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        smax = fmaxf(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        rmax = fmaxf(rmax, __shfl_xor_sync(0xffffffffu, rmax, o));
      }
      if (lane == 0) { red[warp] = smax;  red[kThreads / 32 + warp] = rmax; }
      __syncthreads();
      smax = 0.f;  rmax = 0.f;
#pragma unroll
      for (int w = 0; w < kThreads / 32; ++w) { smax = fmaxf(smax, red[w]);  rmax = fmaxf(rmax, red[kThreads / 32 + w]); }
      int ex = 15;                           // s r < 2^ex  =>  c = 2^(15 - ex)
      const float prod = smax * rmax;
      if (prod > 0.f && prod < 3.0e38f) frexpf(prod, &ex);
      ex = max(-60, min(60, 15 - ex));
      const float cs = ldexpf(1.f, ex);
      inv_c2 = ldexp(1.0, -2 * ex);
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        hp[c] = make_float4(cs * sp[4 * c], cs * sp[4 * c + 1], cs * sp[4 * c + 2], cs * sp[4 * c + 3]);
        np_[c] = make_float4(cs * sn[4 * c], cs * sn[4 * c + 1], cs * sn[4 * c + 2], cs * sn[4 * c + 3]);
      }
    }
    __syncthreads();

    const int rows_here = min(kTH, vr - tile_y * kTH);
    TC_T(0);
#ifndef DIA_TC_FOLD_ROWS
#define DIA_TC_FOLD_ROWS 64
#endif
    int rows_in_acc = 0;
    // fold the float32 row sums into this CTA's FP64 block [column][row]
    auto fold = [&]() {
      double* o = outp + (size_t)((warp >> 2) * ncol) * kTcGroup + (warp & 3) * 32 + lane;
      if (n_groups == 2) {
#pragma unroll
        for (int c = 0; c < kTcGroup; ++c) {
          o[(size_t)c * kTcGroup] = first_tile ? inv_c2 * (double)acc[c] : o[(size_t)c * kTcGroup] + inv_c2 * (double)acc[c];
          acc[c] = 0.f;
        }
      } else {
#pragma unroll
        for (int c = 0; c < kTcGroup / 2; ++c) {
          o[(size_t)c * kTcGroup] = first_tile ? inv_c2 * (double)acc[c] : o[(size_t)c * kTcGroup] + inv_c2 * (double)acc[c];
          acc[c] = 0.f;
        }
      }
      first_tile = false;
      rows_in_acc = 0;
    };
    bool pend = false;                       // a finished row is waiting for its flush
    unsigned pend_bar = 0, pend_par = 0, pend_tb = 0;
    auto flush_pending = [&]() {
      mbar_wait(pend_bar, pend_par);
      tc_fence_after();
      const unsigned ta = my_taddr + pend_tb * (unsigned)kTcRows;
      if (n_groups == 2) {
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) tc_flush32(ta + 32u * cc, acc + 32 * cc);
      } else {
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) tc_flush32(ta + 32u * cc, acc + 32 * cc);
      }
      pend = false;
      if (++rows_in_acc == DIA_TC_FOLD_ROWS) fold();
    };
#pragma unroll 1
    for (int i = 0; i < rows_here; ++i) {
      const int n_pass = rowneg[i] ? 2 : 1;
#pragma unroll 1
      for (int pass = 0; pass < n_pass; ++pass) {
        const unsigned sb = gst & 1u;
        if (gst >= 2) mbar_wait(bar0 + 8u * sb, ((gst >> 1) - 1u) & 1u);      // the MMAs of stage gst - 2 have read this buffer
        TC_T(1);
        unsigned char* const op_hi = ops + sb * T::OP_BUF;
        if (my_bg)
          tc_build_row<true>(op_hi + my_off, op_hi + T::OP_TILE + my_off, T::LBO, etapow + bg_m * kTW, (pass ? Is : Hs) + i * kIPitch,
                             xipow[bg_n * kTH + i]);
        else if (my_valid)
          tc_build_row<false>(op_hi + my_off, op_hi + T::OP_TILE + my_off, T::LBO, Rs + (i + my_a) * G::RPITCH + my_b,
                              (pass ? Is : Hs) + i * kIPitch);
        TC_T(2);
        fence_proxy_async();
        tc_fence_before();
        __syncthreads();
        TC_T(3);
        if (tid == 0) {
          tc_fence_after();
          const unsigned base = smem_u32(op_hi);
          const unsigned d_addr = tmem + (grow & 1u) * (unsigned)kTcRows;
          const unsigned id = idesc | (pass ? (1u << 13) : 0u);                 // second pass: A negated
#pragma unroll
          for (int term = 0; term < 4; ++term) {             // lo lo, lo hi, hi lo, hi hi: small terms first (truncation, see above)
            const unsigned ta = base + (term < 2 ? T::OP_TILE : 0) + a_sel * (kTcGroup / 8 * 128);
            const unsigned tb = base + ((term & 1) ? 0 : T::OP_TILE) + b_start * (kTcGroup / 8 * 128);
#pragma unroll
            for (int s = 0; s < kTW / 16; ++s)
              tc_mma_f16(d_addr, tc_smem_desc(ta + s * 2 * T::LBO, T::LBO, T::SBO), tc_smem_desc(tb + s * 2 * T::LBO, T::LBO, T::SBO),
                          id, (pass > 0 || term > 0 || s > 0) ? 1u : 0u);
          }
          tc_commit(bar0 + 8u * sb);
        }
        TC_T(4);
        if (pend) flush_pending();           // the previous row, while this stage's MMAs run
        TC_T(5);
        if (pass == n_pass - 1) {
          pend = true;  pend_bar = bar0 + 8u * sb;  pend_par = (gst >> 1) & 1u;  pend_tb = grow & 1u;
          ++grow;
        }
        ++gst;
      }
    }
    if (pend) flush_pending();
    TC_T(6);
    if (rows_in_acc > 0) fold();
    TC_T(7);
    tc_fence_before();
    __syncthreads();                         // tiles and flags free for the next tile
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem), "r"(512u) : "memory");
}

#ifndef DIA_INST_M
// Sums the FP64 blocks of the CTAs of each type in CTA order and writes the entries of H (both
// triangles for an off-diagonal block; a diagonal block delivers both of its triangles itself).
__global__ void hess_tc_reduce_kernel(const double* __restrict__ partials, const short* __restrict__ perm,
                                      const __grid_constant__ HessTcTypes ty, int np, double* __restrict__ H) {
  const int type = blockIdx.y;
  const int n_cols = kTcGroup * ty.n_groups[type];
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n_cols * kTcGroup) return;
  const int n = idx / kTcGroup, r = idx - n * kTcGroup;
  const int gA = ty.a_sel[type] ? ty.g1[type] : ty.g0[type];
  const int gB = (ty.b_start[type] + n / kTcGroup) ? ty.g1[type] : ty.g0[type];
  const int pr = perm[gA * kTcGroup + r], qc = perm[gB * kTcGroup + (n % kTcGroup)];
  if (pr < 0 || qc < 0) return;
  double s = 0.0;
  for (int c = 0; c < ty.ctas_per_type; ++c)
    s += partials[(size_t)(c * ty.n_types + type) * (kTcRows * kTcGroup) + idx];
  H[(size_t)pr * np + qc] = s;
  if (gA != gB) H[(size_t)qc * np + pr] = s;
}

// perm[slot] for the 128 G slots (G = ceil(np / 128)), -1 for an empty slot: kernel pixel (a, b) reads the staged R tile
// at a * r_pitch + b + const, so its bank class is (a * r_pitch + b) mod 32; each row goes to the first warp (32 slots)
// that has no row of its class yet, background rows (no R reads) and leftovers fill the gaps.
inline void hess_tc_make_perm(int m, int np, int r_pitch, short* perm) {
  const int G = (np + kTcGroup - 1) / kTcGroup, n_warps = 4 * G;
  for (int s = 0; s < G * kTcGroup; ++s) perm[s] = -1;
  unsigned used[64 * 4] = {};                  // per warp: bank classes taken (G <= 64)
  int fill[64 * 4] = {};
  short late[kTcGroup * 64];
  int n_late = 0;
  for (int q = 0; q < np; ++q) {
    int w = -1;
    if (q < m * m) {
      const unsigned bit = 1u << (((q / m) * r_pitch + q % m) & 31);
      for (int c = 0; c < n_warps && w < 0; ++c)
        if (fill[c] < 32 && !(used[c] & bit)) { w = c;  used[c] |= bit; }
    }
    if (w < 0) { late[n_late++] = (short)q;  continue; }
    perm[32 * w + fill[w]++] = (short)q;
  }
  for (int k = 0, w = 0; k < n_late; ++k) {
    while (fill[w] >= 32) ++w;
    perm[32 * w + fill[w]++] = late[k];
  }
}

// The types for np parameters: every diagonal block (i, i) paired with an off-diagonal block of its row or column
// while one is free, the remaining blocks alone.  Returns the number of types (0: too many).
inline int hess_tc_make_types(int np, HessTcTypes* ty) {
  const int G = (np + kTcGroup - 1) / kTcGroup;
  bool used[32][32] = {};
  int n = 0;
  auto add = [&](int g0, int g1, int a_sel, int b_start, int n_groups) {
    if (n < kTcMaxTypes) {
      ty->g0[n] = (unsigned char)g0;  ty->g1[n] = (unsigned char)g1;  ty->a_sel[n] = (unsigned char)a_sel;
      ty->b_start[n] = (unsigned char)b_start;  ty->n_groups[n] = (unsigned char)n_groups;
    }
    ++n;
  };
  if (G > 32) return 0;
  for (int i = 0; i < G; ++i) {
    int j = -1;
    for (int c = i + 1; c < G && j < 0; ++c) if (!used[i][c]) j = c;
    if (j >= 0) { used[i][j] = true; add(i, j, 0, 0, 2); continue; }            // D = [ (i,i) | (i,j) ]
    for (int c = 0; c < i && j < 0; ++c) if (!used[c][i]) j = c;
    if (j >= 0) { used[j][i] = true; add(j, i, 1, 0, 2); continue; }            // D = [ (i,j) | (i,i) ]
    add(i, 255, 0, 0, 1);
  }
  for (int i = 0; i < G; ++i)
    for (int j = i + 1; j < G; ++j)
      if (!used[i][j]) add(i, j, 0, 1, 1);                                      // D = (i,j)
  ty->n_types = n;
  return n <= kTcMaxTypes ? n : 0;
}
#endif  // DIA_INST_M

}  // namespace dia
