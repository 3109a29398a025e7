// dia_eval.cuh -- fused loss + gradient kernel for the B08 discrete-pixel kernel model (sm_100a).
//
// One persistent CTA loops over 64x64 tiles of the valid region.  Per tile:
//   stage   R tile + (m-1) halo and the I tile into shared memory with cp.async (double buffered),
//   forward each thread owns a 16-pixel row strip: M = R (x) K + B0 (Eq. 2) in FP32
//           registers, then residual, variance (Eq. 6), loss term (Eq. 8 / Eq. 12-13,
//           PAPER.md:115, 154-161) and the weight w = dL/dM, written back over the I tile,
//   grad    thread (a, s) owns the m accumulators g[a][0..m-1] and correlates 16-pixel chunks of w
//           against the staged R rows (dL/dK[a][b] = sum w_ij R[i+a][j+b]),
//   flush   per-tile FP32 strips are summed over s in fixed order and added to FP64 accumulators.
// Nothing n^2-sized is written to HBM.  The tile->CTA map and every reduction order are fixed, so
// repeated evaluations are bit-identical.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dia {

constexpr int kThreads = 256;
constexpr int kTW = 64, kTH = 64;     // output tile
constexpr int kP = 16;                // forward strip / gradient chunk length (pixels)
constexpr int kIPitch = 68;           // I/w tile pitch (floats); 68/4 = 17 is odd => conflict-free rows

__host__ __device__ constexpr int round_up(int x, int q) { return (x + q - 1) / q * q; }

template <int M>
struct Geo {
  static constexpr int H = (M - 1) / 2;
  static constexpr int NP = M * M + 1;                       // parameters per epoch
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
  static constexpr int RED_FLOATS = S * M * M;               // aliases the current R buffer
  static constexpr int NOUT = (M * M + kThreads - 1) / kThreads;   // FP64 accumulators per thread
  static constexpr size_t SMEM = sizeof(float) * (2 * R_FLOATS + 2 * I_FLOATS + K_FLOATS) + 64;
  static_assert(RED_FLOATS <= R_FLOATS, "reduction scratch must fit in one R buffer");
  static_assert(RPITCH % 8 == 4, "pitch");
};

struct EvalParams {
  const float* R;            // [n_rows][n_cols]
  const float* I;            // [E][n_rows][n_cols]
  const unsigned char* mask; // [E][n_rows][n_cols] or null
  const float* var;          // [E][n_rows][n_cols] or null (FIXED noise)
  const float* flat;         // [n_rows][n_cols] or null
  const float* theta;        // [E][NP] float32
  const int* done;           // [E] or null: epochs with done != 0 are skipped
  double* partials;          // [E][gridDim.x][NP+1]: g_K (M*M), g_B0, loss
  int n_rows, n_cols, n_epochs;
  int tiles_x, tiles_y;
  int loss_kind, noise_kind;
  float huber_c, sigma0_sq, inv_gain;
  int r_vec4;                // 1: R rows are 16-byte aligned (n_cols % 4 == 0 and base aligned)
};

__device__ __forceinline__ void cp_async_16(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_4(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// Stage one tile: R rows [y0, y0+RH) x cols [x0, x0+RPITCH) and the I tile, zero filled outside.
template <int M>
__device__ __forceinline__ void stage_tile(const EvalParams& p, const float* __restrict__ Iep,
                                           float* Rs, float* Is, int ty, int tx) {
  using G = Geo<M>;
  const int y0 = ty * kTH, x0 = tx * kTW;
  if (p.r_vec4) {
    constexpr int C4 = G::RPITCH / 4;
    for (int idx = threadIdx.x; idx < G::RH * C4; idx += kThreads) {
      const int rr = idx / C4, c4 = idx - rr * C4;
      const int gy = y0 + rr, gx = x0 + 4 * c4;
      const bool ok = (gy < p.n_rows) && (gx < p.n_cols);
      const float* src = ok ? p.R + (size_t)gy * p.n_cols + gx : p.R;
      cp_async_16(Rs + rr * G::RPITCH + 4 * c4, src, ok ? 16 : 0);
    }
  } else {
    for (int idx = threadIdx.x; idx < G::RH * G::RPITCH; idx += kThreads) {
      const int rr = idx / G::RPITCH, cc = idx - rr * G::RPITCH;
      const int gy = y0 + rr, gx = x0 + cc;
      const bool ok = (gy < p.n_rows) && (gx < p.n_cols);
      const float* src = ok ? p.R + (size_t)gy * p.n_cols + gx : p.R;
      cp_async_4(Rs + rr * G::RPITCH + cc, src, ok ? 4 : 0);
    }
  }
  const int vr = p.n_rows - M + 1, vc = p.n_cols - M + 1;
  for (int idx = threadIdx.x; idx < kTH * kTW; idx += kThreads) {
    const int rr = idx / kTW, cc = idx - rr * kTW;
    const int iy = y0 + rr, ix = x0 + cc;
    const bool ok = (iy < vr) && (ix < vc);
    const float* src = ok ? Iep + (size_t)(iy + G::H) * p.n_cols + (ix + G::H) : Iep;
    cp_async_4(Is + rr * kIPitch + cc, src, ok ? 4 : 0);
  }
}

__device__ __forceinline__ double warp_sum_f64(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <int M>
__global__ void __launch_bounds__(kThreads, 2) eval_kernel(const EvalParams p) {
  using G = Geo<M>;
  extern __shared__ __align__(16) float smem[];
  float* Rbuf[2] = {smem, smem + G::R_FLOATS};
  float* Ibuf[2] = {smem + 2 * G::R_FLOATS, smem + 2 * G::R_FLOATS + G::I_FLOATS};
  float* Ks = smem + 2 * G::R_FLOATS + 2 * G::I_FLOATS;
  __shared__ double red64[2][kThreads / 32];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n_tiles = p.tiles_x * p.tiles_y;
  const int vr = p.n_rows - M + 1, vc = p.n_cols - M + 1;
  const size_t npix = (size_t)p.n_rows * p.n_cols;

  // forward mapping: warp covers 32 px x 16 rows; lane -> (fx, fy) = (lane & 1, lane >> 1)
  const int f_col = (warp & 1) * 32 + (lane & 1) * kP;
  const int f_row = (warp >> 1) * 16 + (lane >> 1);
  // gradient mapping: consecutive threads own consecutive kernel rows a
  const int g_a = tid % M, g_s = tid / M;
  const bool g_active = g_s < G::S;

  for (int e = 0; e < p.n_epochs; ++e) {
    if (p.done && p.done[e]) continue;
    const float* __restrict__ Iep = p.I + (size_t)e * npix;
    const float* __restrict__ th = p.theta + (size_t)e * G::NP;
    __syncthreads();                       // previous epoch finished with Ks / buffers
    for (int idx = tid; idx < G::K_FLOATS; idx += kThreads) {
      const int a = idx / G::KP, b = idx - a * G::KP;
      Ks[idx] = (b < M) ? th[a * M + b] : 0.f;
    }
    const float B0 = th[M * M];

    double loss64 = 0.0, gb064 = 0.0;
    double gacc64[G::NOUT];
#pragma unroll
    for (int q = 0; q < G::NOUT; ++q) gacc64[q] = 0.0;

    int t = blockIdx.x;
    int buf = 0;
    if (t < n_tiles) stage_tile<M>(p, Iep, Rbuf[0], Ibuf[0], t / p.tiles_x, t % p.tiles_x);
    cp_async_commit();

    for (; t < n_tiles; t += gridDim.x, buf ^= 1) {
      const int tile_y = t / p.tiles_x, tile_x = t - tile_y * p.tiles_x;
      cp_async_wait<0>();
      __syncthreads();                     // tile t landed; everyone is done with the other buffers
      {
        const int tn = t + gridDim.x;
        if (tn < n_tiles) stage_tile<M>(p, Iep, Rbuf[buf ^ 1], Ibuf[buf ^ 1], tn / p.tiles_x, tn % p.tiles_x);
        cp_async_commit();
      }
      const float* __restrict__ Rs = Rbuf[buf];
      float* __restrict__ Ws = Ibuf[buf];

      // ------------------------------------------------------------------ forward
      {
        float tot[kP];
#pragma unroll
        for (int q = 0; q < kP; ++q) tot[q] = B0;
        // kernel rows outer -> inner, each row chain wings -> centre, rows combined in FP32:
        // keeps the large centre terms last ("accumulation order")
#pragma unroll 1
        for (int ia = 0; ia < M; ++ia) {
          const int a = (ia & 1) ? (M - 1 - (ia >> 1)) : (ia >> 1);
          float k[G::KP], r[G::RSEG];
          const float4* k4 = reinterpret_cast<const float4*>(Ks + a * G::KP);
#pragma unroll
          for (int q = 0; q < G::KP / 4; ++q) {
            const float4 v = k4[q];
            k[4 * q] = v.x; k[4 * q + 1] = v.y; k[4 * q + 2] = v.z; k[4 * q + 3] = v.w;
          }
          const float4* r4 = reinterpret_cast<const float4*>(Rs + (f_row + a) * G::RPITCH + f_col);
#pragma unroll
          for (int q = 0; q < G::RSEG / 4; ++q) {
            const float4 v = r4[q];
            r[4 * q] = v.x; r[4 * q + 1] = v.y; r[4 * q + 2] = v.z; r[4 * q + 3] = v.w;
          }
          float rs[kP];
#pragma unroll
          for (int q = 0; q < kP; ++q) rs[q] = k[0] * r[q];
#pragma unroll
          for (int ib = 1; ib < M; ++ib) {
            const int b = (ib & 1) ? (M - 1 - (ib >> 1)) : (ib >> 1);
#pragma unroll
            for (int q = 0; q < kP; ++q) rs[q] = fmaf(k[b], r[q + b], rs[q]);
          }
#pragma unroll
          for (int q = 0; q < kP; ++q) tot[q] += rs[q];
        }
        // ---------------------------------------------------------------- residual, noise, loss, weight
        const int iy = tile_y * kTH + f_row, ix0 = tile_x * kTW + f_col;
        float* wrow = Ws + f_row * kIPitch + f_col;
        float iv4[kP];
#pragma unroll
        for (int q = 0; q < kP / 4; ++q) {
          const float4 v = reinterpret_cast<const float4*>(wrow)[q];
          iv4[4 * q] = v.x; iv4[4 * q + 1] = v.y; iv4[4 * q + 2] = v.z; iv4[4 * q + 3] = v.w;
        }
        float lsum = 0.f, wsum = 0.f;
        const size_t gbase = (size_t)(iy + G::H) * p.n_cols + (ix0 + G::H);
#pragma unroll
        for (int q = 0; q < kP; ++q) {
          bool use = (iy < vr) && (ix0 + q < vc);
          if (use && p.mask) use = p.mask[(size_t)e * npix + gbase + q] != 0;
          const float Mv = tot[q];
          float v, bp;
          if (p.noise_kind == 0) {
            float a_ij = p.sigma0_sq, b_ij = p.inv_gain;
            if (p.flat && use) {
              const float invF = 1.0f / p.flat[gbase + q];
              a_ij *= invF * invF;
              b_ij *= invF;
            }
            v = fmaf(b_ij, fmaxf(Mv, 0.f), a_ij);
            bp = Mv > 0.f ? b_ij : 0.f;
          } else {
            v = use ? p.var[(size_t)e * npix + gbase + q] : 1.f;
            bp = 0.f;
          }
          const float res = iv4[q] - Mv;
          const float inv_v = 1.0f / v;
          const float hb = 0.5f * bp * inv_v;
          float li, wi;
          const float z2 = res * res * inv_v;
          bool lin = false;
          float rsd = 0.f, z = 0.f;
          if (p.loss_kind == 1) {
            rsd = rsqrtf(v);
            z = res * rsd;
            lin = fabsf(z) > p.huber_c;
          }
          if (!lin) {
            li = 0.5f * z2;
            wi = fmaf(-res, inv_v, hb * (1.0f - z2));
          } else {
            const float psi = copysignf(p.huber_c, z);
            li = p.huber_c * (fabsf(z) - 0.5f * p.huber_c);
            wi = fmaf(-psi, rsd, hb * (1.0f - psi * z));
          }
          if (p.noise_kind == 0) li = fmaf(0.5f, logf(v), li);
          if (!use) { li = 0.f; wi = 0.f; }
          lsum += li;
          wsum += wi;
          iv4[q] = wi;
        }
#pragma unroll
        for (int q = 0; q < kP / 4; ++q)
          reinterpret_cast<float4*>(wrow)[q] = make_float4(iv4[4 * q], iv4[4 * q + 1], iv4[4 * q + 2], iv4[4 * q + 3]);
        loss64 += (double)lsum;
        gb064 += (double)wsum;
      }
      __syncthreads();                     // w tile complete

      // ------------------------------------------------------------------ gradient
      float acc[M];
#pragma unroll
      for (int b = 0; b < M; ++b) acc[b] = 0.f;
      if (g_active) {
        const int rows_here = min(kTH, vr - tile_y * kTH);
        const int n_items = rows_here * (kTW / kP);
#pragma unroll 1
        for (int it = g_s; it < n_items; it += G::S) {
          const int i = it / (kTW / kP), c = it - i * (kTW / kP);
          float w[kP], r[G::RSEG];
          const float4* w4 = reinterpret_cast<const float4*>(Ws + i * kIPitch + c * kP);
#pragma unroll
          for (int q = 0; q < kP / 4; ++q) {
            const float4 v = w4[q];
            w[4 * q] = v.x; w[4 * q + 1] = v.y; w[4 * q + 2] = v.z; w[4 * q + 3] = v.w;
          }
          const float4* r4 = reinterpret_cast<const float4*>(Rs + (i + g_a) * G::RPITCH + c * kP);
#pragma unroll
          for (int q = 0; q < G::RSEG / 4; ++q) {
            const float4 v = r4[q];
            r[4 * q] = v.x; r[4 * q + 1] = v.y; r[4 * q + 2] = v.z; r[4 * q + 3] = v.w;
          }
#pragma unroll
          for (int q = 0; q < kP; ++q)
#pragma unroll
            for (int b = 0; b < M; ++b) acc[b] = fmaf(w[q], r[q + b], acc[b]);
        }
      }
      __syncthreads();                     // all reads of Rs / Ws done; Rs becomes the scratch
      float* red = Rbuf[buf];
      if (g_active) {
#pragma unroll
        for (int b = 0; b < M; ++b) red[g_s * (M * M) + g_a * M + b] = acc[b];
      }
      __syncthreads();
#pragma unroll
      for (int q = 0; q < G::NOUT; ++q) {
        const int o = tid + q * kThreads;
        if (o < M * M) {
          double s = 0.0;
#pragma unroll 1
          for (int ss = 0; ss < G::S; ++ss) s += (double)red[ss * (M * M) + o];
          gacc64[q] += s;
        }
      }
      // the next iteration's first __syncthreads orders these reads before the buffer is re-staged
    }
    cp_async_wait<0>();

    // ---------------------------------------------------------------- per-epoch block partials
    double* out = p.partials + ((size_t)e * gridDim.x + blockIdx.x) * (G::NP + 1);
#pragma unroll
    for (int q = 0; q < G::NOUT; ++q) {
      const int o = tid + q * kThreads;
      if (o < M * M) out[o] = gacc64[q];
    }
    const double l = warp_sum_f64(loss64), g0 = warp_sum_f64(gb064);
    __syncthreads();
    if (lane == 0) { red64[0][warp] = l; red64[1][warp] = g0; }
    __syncthreads();
    if (tid == 0) {
      double ls = 0.0, gs = 0.0;
      for (int w = 0; w < kThreads / 32; ++w) { ls += red64[0][w]; gs += red64[1][w]; }
      out[M * M] = gs;
      out[M * M + 1] = ls;
    }
  }
}

// Second level: sum the block partials in block order (fixed order => deterministic).
__global__ void reduce_partials_kernel(const double* __restrict__ partials, int n_blocks, int np1,
                                       const int* __restrict__ done, double* __restrict__ loss,
                                       double* __restrict__ grad) {
  const int e = blockIdx.y;
  if (done && done[e]) return;
  const int o = blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= np1) return;
  const double* src = partials + (size_t)e * n_blocks * np1 + o;
  double s = 0.0;
  for (int b = 0; b < n_blocks; ++b) s += src[(size_t)b * np1];
  if (o == np1 - 1) loss[e] = s;
  else grad[(size_t)e * (np1 - 1) + o] = s;
}

}  // namespace dia
