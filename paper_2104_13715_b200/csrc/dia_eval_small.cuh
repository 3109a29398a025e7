// dia_eval_small.cuh -- fused loss + gradient kernel for SMALL kernels (m = 1, 3, 5), plain objective only
// (Eq. 2, 6, 8 / 12-13; no mask, flat field, variance map, background polynomial).
//
// For m <= 5 the evaluation has 4 m^2 <= 100 FLOP per 8 bytes of image: the roofline is HBM bandwidth (m <= 3) or
// instruction issue, not the FMA pipe, and the generic kernel's shared-memory tiles (w tile, gradient strips, two
// barriers per tile) cost more instructions per pixel than the arithmetic itself (87 per pixel at m = 3, ncu reading
// in profiles/r01_sweeps.md).  Here everything stays in registers:
//   * a thread owns an 8-pixel row strip and walks down `rpt` rows with a sliding window of the m reference rows it
//     needs (one new row of 8 + m - 1 pixels per step, 128-bit loads straight from global memory -- neighbouring
//     threads' halo re-reads hit L1), lanes of a warp sit side by side (coalesced 1 KB rows);
//   * M, residual, variance, loss term and w = dL/dM per pixel as in the generic kernel (same pixel_terms);
//   * the m^2 gradient sums g[a][b] += w_q R[a][q + b] reuse the window registers: no w tile, no second pass;
//   * per tile the m^2 FP32 sums are reduced across the warp by a transposing butterfly (lane k ends up with sum k)
//     and added to a lane-held FP64 total; loss and g_B0 go to thread-private FP64 every row.
// Work items, partial-column layout and the `done` flags are those of the generic kernel, so the second level
// (reduce_partials_kernel / fit_step_kernel) is shared.  Fixed orders everywhere: bit-reproducible.
#pragma once
#include "dia_eval.cuh"

namespace dia {

constexpr int kSmallPx = 8;        // pixels per thread and row

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
};

template <int M>
__global__ void __launch_bounds__(kThreads, 2) eval_small_kernel(const EvalParams p) {
  using G = SmallGeo<M>;
  constexpr int SEG = G::SEG, P = G::P, H = G::H;
  __shared__ double red[kThreads / 32][32];
  __shared__ double red2[2][kThreads / 32];
  __shared__ float K[M * M];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int lxlog = p.small_lxlog, rpt = p.small_rpt;
  const int lx = lane & ((1 << lxlog) - 1), ly = lane >> lxlog;
  const int rows_per_warp = (32 >> lxlog) * rpt;
  const int tile_w = kSmallPx << lxlog, tile_h = (kThreads / 32) * rows_per_warp;
  const int vr = p.n_rows - M + 1, vc = p.n_cols - M + 1;
  const int tiles_x = (vc + tile_w - 1) / tile_w, tiles_y = (vr + tile_h - 1) / tile_h;
  const int n_tiles = tiles_x * tiles_y;
  const size_t npix = (size_t)p.n_rows * p.n_cols;
  const bool vec = p.small_vec != 0;
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
      for (int w = 0; w < kThreads / 32; ++w) s += red[w][src];
      out[(size_t)tid * ncols] = s;
    }
    if (tid == 32) {
      double ls = 0.0, gs = 0.0;
#pragma unroll
      for (int w = 0; w < kThreads / 32; ++w) { ls += red2[0][w]; gs += red2[1][w]; }
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
    const int tile_y = t / tiles_x, tile_x = t - tile_y * tiles_x;
    const int x0 = tile_x * tile_w + kSmallPx * lx;                       // first pixel of the strip (valid coords)
    const int y0 = tile_y * tile_h + (warp * (32 >> lxlog) + ly) * rpt;   // first row of this thread
    const int nrows = min(rpt, vr - y0);                                  // <= 0: nothing to do
    const float* __restrict__ Rimg = p.R + (p.n_refs > 1 ? (size_t)e * npix : (size_t)0);
    const float* __restrict__ Iimg = p.I + (size_t)e * npix;

    float acc[P];
#pragma unroll
    for (int i = 0; i < P; ++i) acc[i] = 0.f;
    if (x0 < vc && nrows > 0) {
      float win[M][SEG];
#pragma unroll
      for (int a = 0; a < M - 1; ++a) load_seg<SEG>(Rimg, p.n_rows, p.n_cols, y0 + a, x0, vec, pol_keep, win[a]);
#pragma unroll 1
      for (int r0 = 0; r0 < nrows; r0 += M) {
#pragma unroll
        for (int u = 0; u < M; ++u) {
          const int r = r0 + u;
          if (r < nrows) {
            // window row a of this step lives in win[(u + a) % M]; the new bottom row goes to win[(u + M - 1) % M]
            load_seg<SEG>(Rimg, p.n_rows, p.n_cols, y0 + r + M - 1, x0, vec, pol_keep, win[(u + M - 1) % M]);
            float iv[SEG];
            load_seg<SEG>(Iimg, p.n_rows, p.n_cols, y0 + r + H, x0, vec, pol_stream, iv);
            // model: kernel rows in pairs (0, M-1), (1, M-2), ..., centre last; columns wings -> centre
            float tot[kSmallPx];
#pragma unroll
            for (int q = 0; q < kSmallPx; ++q) tot[q] = B0;
#pragma unroll
            for (int ia = 0; ia < M; ++ia) {
              const int a = (ia & 1) ? (M - 1 - (ia >> 1)) : (ia >> 1);
              float rs[kSmallPx];
#pragma unroll
              for (int ib = 0; ib < M; ++ib) {
                const int b = (ib & 1) ? (M - 1 - (ib >> 1)) : (ib >> 1);
#pragma unroll
                for (int q = 0; q < kSmallPx; ++q) {
                  const float rv = win[(u + a) % M][q + b];
                  rs[q] = ib == 0 ? K[a * M + b] * rv : fmaf(K[a * M + b], rv, rs[q]);
                }
              }
#pragma unroll
              for (int q = 0; q < kSmallPx; ++q) tot[q] += rs[q];
            }
            float lsum = 0.f, wsum = 0.f;
#pragma unroll
            for (int q = 0; q < kSmallPx; ++q) {
              float li, wi;
              pixel_terms<false, true>(p, e, npix, 0, x0 + q < vc, tot[q], iv[q + H], li, wi);
              lsum += li;
              wsum += wi;
#pragma unroll
              for (int a = 0; a < M; ++a)
#pragma unroll
                for (int b = 0; b < M; ++b) acc[a * M + b] = fmaf(wi, win[(u + a) % M][q + b], acc[a * M + b]);
            }
            loss64 += (double)lsum;
            gb064 += (double)wsum;
          }
        }
      }
    }
    warp_transpose_sum<P>(acc, lane);
    g64 += (double)acc[0];
    step(j, t);
    skip_done(j, t);
  }
  if (cur_j >= 0) finish_epoch();
}

}  // namespace dia
