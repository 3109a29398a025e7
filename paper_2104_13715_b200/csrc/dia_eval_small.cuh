// dia_eval_small.cuh -- fused loss + gradient kernel for SMALL kernels (m = 1, 3, 5), plain objective only
// (Eq. 2, 6, 8 / 12-13; no mask, flat field, variance map, background polynomial).
//
// For m <= 5 the evaluation has 4 m^2 <= 100 FLOP per 8 bytes of image: the algorithmic roofline is HBM bandwidth, and
// the generic kernel's shared-memory tiles (w tile, gradient strips, two barriers per tile) cost more instructions per
// pixel than the arithmetic itself (87 per pixel at m = 3, ncu reading in profiles/r01_sweeps.md).  What this kernel
// runs out of in practice is the FMA pipe at the ~50 % that 8 - 16 warps per SM can keep busy (the per-pixel terms'
// FP32 operations count as much as the stencil's; profiles/r02_small3.md).  Here everything stays in registers:
//   * a thread owns an 8-pixel row strip and walks down `rpt` rows with a sliding window of the m reference rows it
//     needs (one new row of 8 + m - 1 reference pixels and 8 target pixels per step, 128-bit loads straight from
//     global memory, the rows two steps ahead requested by prefetch.global.L1 -- neighbouring threads' halo re-reads
//     hit L1); lanes of a warp sit side by side (coalesced 1 KB rows);
//   * M, residual, variance, loss term and w = dL/dM per pixel: the generic kernel's formulas (rearranged for the
//     Gaussian loss: small_gauss_terms), ln v from lg2.approx;
//   * the m^2 gradient sums g[a][b] += w_q R[a][q + b] reuse the window registers: no w tile, no second pass;
//   * per tile the m^2 FP32 sums are reduced across the warp by a transposing butterfly (lane k ends up with sum k)
//     and added to a lane-held FP64 total; loss and g_B0 go to thread-private FP64 every row.
// Work items, partial-column layout and the `done` flags are those of the generic kernel, so the second level
// (reduce_partials_kernel / fit_step_kernel) is shared.  Fixed orders everywhere: bit-reproducible.
#pragma once
#include <type_traits>

#include "dia_eval.cuh"

namespace dia {

constexpr int kSmallPx = 8;        // pixels per thread and row
constexpr int kSmallAhead = 2;     // rows between the prefetch of a row and its use

__device__ __forceinline__ float4 ldg_hint_f4(const float* ptr, unsigned long long pol) {
  float4 v;
  asm volatile("ld.global.nc.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4], %5;\n"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(ptr), "l"(pol));
  return v;
}

// SEG floats of image row `row` starting at column x (x % 4 == 0); pixels outside the image read 0.
// vec: rows are 16-byte aligned (n_cols % 4 == 0 and an aligned base), so every float4 is inside or outside.
template <int SEG>
__device__ __forceinline__ void load_seg(const float* __restrict__ img, int n_rows, int n_cols, int row, int x, bool vec,
                                         unsigned long long pol, float (&r)[SEG]) {
  const bool row_ok = row < n_rows;
  const float* src = img + (size_t)row * n_cols + x;
  if (vec) {
#pragma unroll
    for (int q = 0; q < SEG / 4; ++q) {
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (row_ok && x + 4 * q + 4 <= n_cols) v = ldg_hint_f4(src + 4 * q, pol);
      r[4 * q] = v.x; r[4 * q + 1] = v.y; r[4 * q + 2] = v.z; r[4 * q + 3] = v.w;
    }
  } else {
#pragma unroll
    for (int q = 0; q < SEG; ++q) r[q] = (row_ok && x + q < n_cols) ? __ldg(src + q) : 0.f;
  }
}

// The same for a strip that lies inside the image with 16-byte aligned rows: no predicates, no zero fill.
template <int SEG>
__device__ __forceinline__ void load_fast(const float* __restrict__ src, unsigned long long pol, float (&r)[SEG]) {
#pragma unroll
  for (int q = 0; q < SEG / 4; ++q) {
    const float4 v = ldg_hint_f4(src + 4 * q, pol);
    r[4 * q] = v.x; r[4 * q + 1] = v.y; r[4 * q + 2] = v.z; r[4 * q + 3] = v.w;
  }
}

// Asks for the line that holds `ptr` (a row this thread reads kSmallAhead steps from now) to be brought to L1: the
// later load then waits for a cache hit instead of DRAM (measured at m = 1: 21.6 us per 4096^2 epoch without, 19.2 us
// with an L2 prefetch four rows ahead, 17.4 us with this L1 prefetch two rows ahead).  (Copying ahead into shared memory with per-thread cp.async was tried and was
// 25 % slower: 16-byte copies with a 32-byte lane stride use the LSU poorly.)
__device__ __forceinline__ void prefetch_row(const float* ptr) { asm volatile("prefetch.global.L1 [%0];\n" ::"l"(ptr)); }

// Transposing warp reduction of P = 1, 16 or 32 per-thread values: on return v[0] of lane l holds the sum over the
// warp of value index l (P = 32), l >> 1 (P = 16), 0 (P = 1).  Fixed order.
template <int C, int O, int P>
struct TransposeSum {
  static __device__ __forceinline__ void run(float (&v)[P], int lane) {
    if constexpr (C > 1) {
      constexpr int hc = C / 2;
      const bool up = (lane & O) != 0;
#pragma unroll
      for (int i = 0; i < hc; ++i) {
        const float send = up ? v[i] : v[i + hc];
        const float keep = up ? v[i + hc] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, O);
      }
      TransposeSum<hc, O / 2, P>::run(v, lane);
    } else {
      v[0] += __shfl_xor_sync(0xffffffffu, v[0], O);
      TransposeSum<1, O / 2, P>::run(v, lane);
    }
  }
};
template <int C, int P>
struct TransposeSum<C, 0, P> {
  static __device__ __forceinline__ void run(float (&)[P], int) {}
};
template <int P>
__device__ __forceinline__ void warp_transpose_sum(float (&v)[P], int lane) { TransposeSum<P, 16, P>::run(v, lane); }

template <int M>
struct SmallGeo {
  static constexpr int H = (M - 1) / 2;
  static constexpr int SEG = round_up(kSmallPx + M - 1, 4);     // 8 (m = 1) or 12 floats per window row
  static constexpr int P = M == 1 ? 1 : (M == 3 ? 16 : 32);     // padded number of kernel-gradient sums
  // m = 1: 3 CTAs of 8 warps at 80 registers; m = 3: 2 CTAs at 128 registers (3 CTAs of 7 warps at 96 registers, or
  // of 8 warps at 80, spill and were measured 19 % and 13 % slower); m = 5: one CTA at ~240 registers (three CTAs of
  // four warps at 168 spill and were measured 9 % slower)
  static constexpr int THREADS = 256;
  static constexpr int MAXREG = M == 1 ? 80 : (M == 3 ? 128 : 255);
};

// Per-pixel terms of the plain objective (D1; the formulas of pixel_terms<false, .> in
// dia_eval.cuh) with the loss a template parameter and ln v from the MUFU unit (lg2.approx, absolute error 2^-22 in
// log2 v: 1e-7 on a term of size 2-6).  hg = inv_gain / 2.
template <bool HUBER>
__device__ __forceinline__ void small_pixel_terms(float Mv, float Iv, float sigma0_sq, float inv_gain, float hg,
                                                  float huber_c, float& li, float& wi) {
  const float v = fmaf(inv_gain, fmaxf(Mv, 0.f), sigma0_sq);
  const float hbp = Mv > 0.f ? hg : 0.f;
  const float res = Iv - Mv;
  const float inv_v = rcp_approx(v);
  const float hb = hbp * inv_v;                    // b' / (2 v)
  const float rv = res * inv_v;
  const float z2 = res * rv;
  const float hlv = 0.34657359028f * lg2_approx(v);   // ln(v) / 2
  li = fmaf(0.5f, z2, hlv);
  wi = fmaf(hb, 1.0f - z2, -rv);
  if (HUBER) {                                     // Eq. 12
    const float rsd = rsqrtf(v);
    const float z = res * rsd;
    if (fabsf(z) > huber_c) {
      const float psi = copysignf(huber_c, z);
      li = fmaf(huber_c, fabsf(z) - 0.5f * huber_c, hlv);
      wi = fmaf(-psi, rsd, hb * (1.0f - psi * z));
    }
  }
}

// The Gaussian terms in the form the row loop uses: the FMA pipe, not instruction issue, is what this kernel runs out
// of (every variant that was tried -- fewer instructions, no memory stalls -- ends at the same ~31 pipe cycles per pixel,
// profiles/r02_small3.md), so the terms are arranged for the fewest FP32 operations: with t = r / v,
//   a = 1 - z^2 = fma(-t, r, 1),   w = (b' / 2 * a - r) / v,   l = z^2 / 2 + ln v / 2 = (1 - a) / 2 + ln 2 / 2 * log2 v,
// and the caller sums a and log2 v over the strip's row and forms the loss once per row: 9 FP32 operations per pixel
// (v, r, t, a, b, w and three running sums) instead of 11.
__device__ __forceinline__ void small_gauss_terms(float Mv, float Iv, float sigma0_sq, float inv_gain, float hg, float& a,
                                                  float& lg, float& wi) {
  const float v = fmaf(inv_gain, fmaxf(Mv, 0.f), sigma0_sq);
  const float hbp = Mv > 0.f ? hg : 0.f;
  const float res = Iv - Mv;
  const float inv_v = rcp_approx(v);
  const float t = res * inv_v;
  a = fmaf(-t, res, 1.0f);
  lg = lg2_approx(v);
  wi = fmaf(hbp, a, -res) * inv_v;
}

// One row of a strip: model, per-pixel terms, gradient sums.  EDGE: the strip crosses the right edge of the valid
// region, pixels beyond it contribute nothing (selects, not multiplications: zero-filled pixels may give NaN).
template <int M, int U, bool HUBER, bool EDGE>
__device__ __forceinline__ void small_row(const float (&win)[M][SmallGeo<M>::SEG], const float (&iv)[SmallGeo<M>::SEG],
                                          const float* __restrict__ K, float B0, const EvalParams& p, float hg, int n_in,
                                          float (&acc)[SmallGeo<M>::P], double& loss64, double& gb064) {
  constexpr int H = SmallGeo<M>::H;
  // window row a lives in win[(U + a) % M].  One FP32 chain per pixel, wings first, the centre pixel last (the
  // largest terms of a peaked kernel come last; with m^2 <= 25 terms the order matters little)
  float lsum = 0.f, wsum = 0.f, asum = 0.f;
#pragma unroll
  for (int q = 0; q < kSmallPx; ++q) {
    float tot = B0;
#pragma unroll
    for (int ia = 0; ia < M; ++ia) {
      const int a = (ia & 1) ? (M - 1 - (ia >> 1)) : (ia >> 1);       // 0, M-1, 1, M-2, ..., centre
#pragma unroll
      for (int ib = 0; ib < M; ++ib) {
        const int b = (ib & 1) ? (M - 1 - (ib >> 1)) : (ib >> 1);
        tot = fmaf(K[a * M + b], win[(U + a) % M][q + b], tot);
      }
    }
    float li, wi;
    if constexpr (HUBER) {
      small_pixel_terms<true>(tot, iv[q + H], p.sigma0_sq, p.inv_gain, hg, p.huber_c, li, wi);
      if (EDGE) {
        if (q >= n_in) { li = 0.f; wi = 0.f; }
      }
      lsum += li;
    } else {
      float a1;
      small_gauss_terms(tot, iv[q + H], p.sigma0_sq, p.inv_gain, hg, a1, li, wi);      // li: log2 v
      if (EDGE) {
        if (q >= n_in) { a1 = 1.f; li = 0.f; wi = 0.f; }
      }
      asum += a1;
      lsum += li;
    }
    wsum += wi;
#pragma unroll
    for (int a = 0; a < M; ++a)
#pragma unroll
      for (int b = 0; b < M; ++b) acc[a * M + b] = fmaf(wi, win[(U + a) % M][q + b], acc[a * M + b]);
  }
  if constexpr (!HUBER) lsum = fmaf(0.34657359028f, lsum, 0.5f * ((float)kSmallPx - asum));
  loss64 += (double)lsum;
  gb064 += (double)wsum;
}

// All rows of one thread's strip in one tile.  FAST: the strip's segments lie inside the image and rows are 16-byte
// aligned (every strip but the last of an image row): unpredicated 128-bit loads through running pointers; for
// m = 1, where nothing but the loads stands between the kernel and the HBM roofline, the next row is loaded into a
// second register set before the current one is used.
template <int M, bool HUBER, bool FAST>
__device__ __forceinline__ void small_strip(const EvalParams& p, const float* __restrict__ Rimg, const float* __restrict__ Iimg,
                                            int y0, int x0, int nrows, int n_in, bool vec, bool warp_full,
                                            unsigned long long pol_keep,
                                            unsigned long long pol_stream, const float* __restrict__ K, float B0, float hg,
                                            float (&acc)[SmallGeo<M>::P], double& loss64, double& gb064) {
  using G = SmallGeo<M>;
  constexpr int SEG = G::SEG, H = G::H;
  const size_t pitch = (size_t)p.n_cols;
  const float* __restrict__ Rp = Rimg + (size_t)(y0 + M - 1) * pitch + x0;   // new window row of the current step
  const float* __restrict__ Ip = Iimg + (size_t)(y0 + H) * pitch + x0;      // target row of the current step
  if constexpr (M == 1 && FAST) {
    float rA[1][SEG], iA[SEG], rB[1][SEG], iB[SEG];
    load_fast<SEG>(Rp, pol_keep, rA[0]);
    load_fast<SEG>(Ip, pol_stream, iA);
#pragma unroll 1
    for (int r = 0; r < nrows; r += 2) {
      if (r + kSmallAhead < nrows) { prefetch_row(Rp + kSmallAhead * pitch); prefetch_row(Ip + kSmallAhead * pitch); }
      if (r + 1 < nrows) { load_fast<SEG>(Rp + pitch, pol_keep, rB[0]); load_fast<SEG>(Ip + pitch, pol_stream, iB); }
      small_row<M, 0, HUBER, false>(rA, iA, K, B0, p, hg, n_in, acc, loss64, gb064);
      if (r + 1 < nrows) {
        if (r + 2 < nrows) { load_fast<SEG>(Rp + 2 * pitch, pol_keep, rA[0]); load_fast<SEG>(Ip + 2 * pitch, pol_stream, iA); }
        small_row<M, 0, HUBER, false>(rB, iB, K, B0, p, hg, n_in, acc, loss64, gb064);
      }
      Rp += 2 * pitch;
      Ip += 2 * pitch;
    }
  } else {
    float win[M][SEG];
#pragma unroll
    for (int a = 0; a < M - 1; ++a) {
      if constexpr (FAST) load_fast<SEG>(Rimg + (size_t)(y0 + a) * pitch + x0, pol_keep, win[a]);
      else load_seg<SEG>(Rimg, p.n_rows, p.n_cols, y0 + a, x0, vec, pol_keep, win[a]);
    }
#pragma unroll 1
    for (int r0 = 0; r0 < nrows; r0 += M) {
      // M steps with compile-time window rotation: the new bottom row of step u goes to win[(u + M - 1) % M]
      auto body = [&](auto uc) {
        constexpr int U = decltype(uc)::value;
        const int r = r0 + U;
        if (r < nrows) {
          if (r + kSmallAhead < nrows) { prefetch_row(Rp + kSmallAhead * pitch); prefetch_row(Ip + kSmallAhead * pitch); }
          float iv[SEG];
          if constexpr (FAST) {
            load_fast<SEG>(Rp, pol_keep, win[(U + M - 1) % M]);
            load_fast<SEG>(Ip, pol_stream, iv);
            small_row<M, U, HUBER, false>(win, iv, K, B0, p, hg, n_in, acc, loss64, gb064);
          } else {
            load_seg<SEG>(Rimg, p.n_rows, p.n_cols, y0 + r + M - 1, x0, vec, pol_keep, win[(U + M - 1) % M]);
            load_seg<SEG>(Iimg, p.n_rows, p.n_cols, y0 + r + H, x0, vec, pol_stream, iv);
            if (warp_full) small_row<M, U, HUBER, false>(win, iv, K, B0, p, hg, n_in, acc, loss64, gb064);
            else small_row<M, U, HUBER, true>(win, iv, K, B0, p, hg, n_in, acc, loss64, gb064);
          }
          Rp += pitch;
          Ip += pitch;
        }
      };
      body(std::integral_constant<int, 0>());
      if constexpr (M >= 3) { body(std::integral_constant<int, 1>()); body(std::integral_constant<int, 2>()); }
      if constexpr (M >= 5) { body(std::integral_constant<int, 3>()); body(std::integral_constant<int, 4>()); }
    }
  }
}

template <int M, bool HUBER>
__global__ void __maxnreg__(SmallGeo<M>::MAXREG) eval_small_kernel(const EvalParams p) {
  using G = SmallGeo<M>;
  constexpr int SEG = G::SEG, P = G::P, H = G::H;
  __shared__ double red[(G::THREADS / 32)][32];
  __shared__ double red2[2][(G::THREADS / 32)];
  __shared__ float K[M * M];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int lxlog = p.small_lxlog, rpt = p.small_rpt;
  const int lx = lane & ((1 << lxlog) - 1), ly = lane >> lxlog;
  const int rows_per_warp = (32 >> lxlog) * rpt;
  const int tile_w = kSmallPx << lxlog, tile_h = ((G::THREADS / 32)) * rows_per_warp;
  const int vr = p.n_rows - M + 1, vc = p.n_cols - M + 1;
  const int tiles_x = (vc + tile_w - 1) / tile_w, tiles_y = (vr + tile_h - 1) / tile_h;
  const int n_tiles = tiles_x * tiles_y;
  const size_t npix = (size_t)p.n_rows * p.n_cols;
  const bool vec = p.small_vec != 0;
  const float hg = 0.5f * p.inv_gain;
  const unsigned long long pol_keep = l2_policy_evict_last(), pol_stream = l2_policy_evict_first();

  const int grid = (int)gridDim.x;
  const int ncols = min(n_tiles, grid);
  auto step = [&](int& j, int& t) {
    t += grid;
    while (t >= n_tiles) { t -= n_tiles; ++j; }
  };
  auto skip_done = [&](int& j, int& t) {
    while (j < p.n_epochs && p.done && p.done[j]) step(j, t);
  };

  float B0 = 0.f;
  double loss64 = 0.0, gb064 = 0.0, g64 = 0.0;   // g64: lane-held total of kernel-gradient sum (lane, or lane >> 1)
  int cur_j = -1;
  double* out = nullptr;

  auto finish_epoch = [&]() {
    const double l = warp_sum_f64(loss64), g0 = warp_sum_f64(gb064);
    red[warp][lane] = g64;
    if (lane == 0) { red2[0][warp] = l; red2[1][warp] = g0; }
    __syncthreads();
    if (tid < M * M) {
      const int src = P == 32 ? tid : (P == 16 ? 2 * tid : 0);
      double s = 0.0;
#pragma unroll
      for (int w = 0; w < (G::THREADS / 32); ++w) s += red[w][src];
      out[(size_t)tid * ncols] = s;
    }
    if (tid == 32) {
      double ls = 0.0, gs = 0.0;
#pragma unroll
      for (int w = 0; w < (G::THREADS / 32); ++w) { ls += red2[0][w]; gs += red2[1][w]; }
      out[(size_t)(M * M) * ncols] = gs;
      out[(size_t)p.np * ncols] = ls;
    }
    __syncthreads();
  };

  int j = 0, t = (int)blockIdx.x - grid;
  step(j, t);
  skip_done(j, t);
  while (j < p.n_epochs) {
    const int e = j;
    if (j != cur_j) {
      if (cur_j >= 0) finish_epoch();
      cur_j = j;
      const float* __restrict__ th = p.theta + (size_t)e * p.np;
      if (tid < M * M) K[tid] = __ldg(th + tid);
      B0 = __ldg(th + M * M);
      loss64 = 0.0; gb064 = 0.0; g64 = 0.0;
      const int col = ((int)blockIdx.x - (int)(((long long)j * n_tiles) % grid) + grid) % grid;
      out = p.partials + ((size_t)e * p.part_rows) * ncols + col;
      __syncthreads();                     // K visible (finish_epoch ended with a barrier after its last reads)
    }
    // item t -> tile (tile_y, tile_x), the columns rotated by the row: a CTA's items are `grid` apart, and with
    // gcd(grid, tiles_x) > 1 (296 and 16 at 4096^2) an unrotated map hands the same few tile columns -- for some CTAs
    // the ragged right-edge column every other item -- to a CTA for its whole life
    const int tile_y = t / tiles_x;
    int tile_x = t - tile_y * tiles_x + tile_y % tiles_x;
    if (tile_x >= tiles_x) tile_x -= tiles_x;
    const int x0 = tile_x * tile_w + kSmallPx * lx;                       // first pixel of the strip (valid coords)
    const int y0 = tile_y * tile_h + (warp * (32 >> lxlog) + ly) * rpt;   // first row of this thread
    const int nrows = min(rpt, vr - y0);                                  // <= 0: nothing to do
    const int n_in = vc - x0;                                             // pixels of the strip inside the valid region
    const float* __restrict__ Rimg = p.R + (p.n_refs > 1 ? (size_t)e * npix : (size_t)0);
    const float* __restrict__ Iimg = p.I + (size_t)e * npix;

    float acc[P];
#pragma unroll
    for (int i = 0; i < P; ++i) acc[i] = 0.f;
    // One path per WARP: a warp whose last lane's strip crosses the edge would otherwise run the fast path for 31
    // lanes and then the predicated one for the last (measured: the edge tile column cost 2.1 x an inner one, 6.5 % of
    // all warp instructions ran with one lane, and the CTAs that owned that column held the grid up: SMs 76 % active)
    const bool live = n_in > 0 && nrows > 0;
    const bool fast = vec && n_in >= kSmallPx && x0 + SEG <= p.n_cols;
    const bool warp_fast = __all_sync(0xffffffffu, fast || !live);
    const bool warp_full = __all_sync(0xffffffffu, n_in >= kSmallPx || !live);
    if (live) {
      if (warp_fast)
        small_strip<M, HUBER, true>(p, Rimg, Iimg, y0, x0, nrows, n_in, vec, warp_full, pol_keep, pol_stream, K, B0, hg, acc, loss64, gb064);
      else
        small_strip<M, HUBER, false>(p, Rimg, Iimg, y0, x0, nrows, n_in, vec, warp_full, pol_keep, pol_stream, K, B0, hg, acc, loss64, gb064);
    }
    warp_transpose_sum<P>(acc, lane);
    g64 += (double)acc[0];
    step(j, t);
    skip_done(j, t);
  }
  if (cur_j >= 0) finish_epoch();
}

}  // namespace dia
