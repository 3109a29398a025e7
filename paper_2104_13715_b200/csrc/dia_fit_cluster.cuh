// dia_fit_cluster.cuh -- the whole fit of a SMALL image pair inside one kernel: one thread-block cluster per epoch.
//
// For images of a few tiles (128^2 - 142^2 stamps: 4 tiles; SURVEY.md section 7 hard part 4) an evaluation is ~1 us of
// arithmetic, and the graph loop of dia_fit.cuh spends ~13 us per iteration on two kernel launches, tile staging and
// reduction latency.  Here a cluster of T = tiles CTAs (T <= 8) owns one epoch for the whole fit:
//   once       every CTA stages ITS tile of R (+ halo) and of I into shared memory (TMA or cp.async) and keeps them;
//   iteration  K and B0 from theta32 -> forward stencil, residual, noise model, loss, weights -> gradient correlation
//              (the device functions of eval_kernel, same arithmetic, same orders) -> this CTA's FP64 partial column
//              -> cluster barrier -> rank 0 runs the optimiser transition (fit_step_body: second-level reduction, Adam
//              or L-BFGS step, stop tests) -> cluster barrier -> next iteration, until the epoch's done flag is set.
// No host round trip, no launch, no re-staging per iteration.  Epochs are independent clusters, so a batch of hundreds
// of stamps is one launch; clusters that finish make room for the next.  Plain objective only (no mask / flat /
// variance map / background polynomial): dia_fit falls back to the graph loop otherwise.  For an image whose tiles
// all sit on different CTAs in the graph loop (single image pairs) the results are bit-identical to it (tested).
#pragma once
#include "dia_fit.cuh"

namespace dia {

constexpr int kMaxClusterTiles = 8;      // portable cluster size

__device__ __forceinline__ unsigned cluster_ctarank() {
  unsigned r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}

template <int M>
struct ClusterGeo {
  using G = Geo<M>;
  static constexpr int PER = (M * M + 1 <= kFitThreads * kPerThreadSmall) ? kPerThreadSmall : kPerThreadLarge;
  static constexpr size_t SCRATCH = step_scratch_bytes<PER>();
  // the optimiser's scratch takes the second R buffer when there is one and it is large enough, else it is appended
  static constexpr bool IN_RBUF = G::NRBUF == 2 && (size_t)G::R_STRIDE >= SCRATCH;
  static constexpr size_t OFF_SCRATCH = IN_RBUF ? (size_t)G::R_STRIDE : ((G::SMEM + 15) / 16 * 16);
  static constexpr size_t SMEM = IN_RBUF ? G::SMEM : OFF_SCRATCH + SCRATCH + 16;
};

template <int M>
__global__ void __launch_bounds__(kThreads, Geo<M>::CTAS) fit_cluster_kernel(const EvalParams p, const __grid_constant__ TensorMaps tm,
                                                                 const StepArgs a) {
  using G = Geo<M>;
  using CG = ClusterGeo<M>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned char* sm = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  float* const Rs = reinterpret_cast<float*>(sm + G::OFF_R);
  float* const Is = reinterpret_cast<float*>(sm + G::OFF_I);
  float* const Ws = reinterpret_cast<float*>(sm + G::OFF_W);
  float* const accS = reinterpret_cast<float*>(sm + G::OFF_ACC);
  float* const Ks = reinterpret_cast<float*>(sm + G::OFF_K);
  float* const Bs = reinterpret_cast<float*>(sm + G::OFF_BG);
  const unsigned bar0 = smem_u32(sm + G::OFF_BAR);
  double* const red64 = reinterpret_cast<double*>(sm + G::OFF_BAR + 64);
  double* const scr = reinterpret_cast<double*>(sm + CG::OFF_SCRATCH);
  StepScratch sc;
  sc.sh_rows = reinterpret_cast<double (*)[kFitThreads / 32]>(scr);
  sc.s_alpha = scr + 2 * (kFitThreads / 32);
  sc.gsum = sc.s_alpha + kMaxHistory;
  sc.xs = sc.gsum + kFitThreads * CG::PER;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n_tiles = p.tiles_x * p.tiles_y;               // == cluster size
  const int rank = (int)cluster_ctarank();
  const int e = (int)blockIdx.x / n_tiles, tile = rank;
  const int vr = p.n_rows - M + 1, vc = p.n_cols - M + 1;
  const size_t npix = (size_t)p.n_rows * p.n_cols;
  const int tile_y = tile / p.tiles_x, tile_x = tile - tile_y * p.tiles_x;

  if (tid == 0) {
    const unsigned cnt = p.use_tma ? 1u : (unsigned)kThreads;
#pragma unroll
    for (int b = 0; b < 3; ++b) mbar_init(bar0 + 8u * b, cnt);
    fence_mbar_init();
  }
  __syncthreads();
  stage_R<M>(p, tm, e, tile, smem_u32(Rs), bar0);          // once: the tiles stay resident for the whole fit
  stage_I<M>(p, tm, e, tile, smem_u32(Is), bar0 + 16u);
  mbar_wait(bar0, 0u);
  mbar_wait(bar0 + 16u, 0u);

  const int f_col = (warp & 1) * 32 + (lane & 1) * kP;
  const int f_row = (warp >> 1) * 16 + (lane >> 1);
  const int g_a = tid % M, g_s = tid / M;
  const bool g_active = g_s < G::S;
  float4* const myacc = reinterpret_cast<float4*>(accS + tid * G::KP);
  const int ncols = n_tiles;
  double* const out = p.partials + ((size_t)e * p.part_rows) * ncols + rank;
  const float* __restrict__ th = p.theta + (size_t)e * p.np;
  const bool edge = (tile_y * kTH + kTH > vr) || (tile_x * kTW + kTW > vc);
  const int rows_here = min(kTH, vr - tile_y * kTH);
  const int n_items = rows_here * (kTW / kP);
  if (tid < kMaxBg) Bs[tid] = 0.f;

  while (true) {
    if (__ldcg(a.b.done + e)) break;                       // set by rank 0 before the barrier that ended the last pass
    for (int idx = tid; idx < G::K_FLOATS; idx += kThreads) {
      const int ka = idx / G::KP, kb = idx - ka * G::KP;
      Ks[idx] = (kb < M) ? __ldcg(th + ka * M + kb) : 0.f;
    }
    const float B0 = __ldcg(th + M * M);
#pragma unroll
    for (int q = 0; q < G::KP / 4; ++q) myacc[q] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();
    double loss64, gb064;
    {                                                      // forward, exactly as eval_kernel
      float tot[kP];
      forward_strip<M, false>(Ks, 0, Rs + f_row * G::RPITCH + f_col, B0, tot);
      const int iy = tile_y * kTH + f_row, ix0 = tile_x * kTW + f_col;
      const float* irow = Is + f_row * kIPitch + f_col;
      float* wrow = Ws + f_row * kIPitch + f_col;
      float lsum, wsum, Sp[4];
      if (edge) strip_epilogue<M, false, true>(p, e, npix, iy, ix0, vr, vc, tot, irow, wrow, Bs, lsum, wsum, Sp);
      else strip_epilogue<M, false, false>(p, e, npix, iy, ix0, vr, vc, tot, irow, wrow, Bs, lsum, wsum, Sp);
      loss64 = (double)lsum;
      gb064 = (double)wsum;
    }
    __syncthreads();
    if (g_active) {                                        // gradient
      GradAcc<M> A;
      grad_acc_load<M>(A, myacc);
#pragma unroll 1
      for (int item = g_s; item < n_items; item += G::S) {
        const int i = item / (kTW / kP), c = item - i * (kTW / kP);
        grad_chunk<M>(A, Ws + i * kIPitch + c * kP, Rs + (i + g_a) * G::RPITCH + c * kP);
      }
      grad_acc_store<M>(A, myacc);
    }
    __syncthreads();
    for (int o = tid; o < M * M; o += kThreads) {          // FP64 fold of the strips, the order of eval_kernel's flush
      const int oa = o / M, ob = o - oa * M;
      double s = 0.0;
#pragma unroll 1
      for (int ss = 0; ss < G::S; ++ss) s += (double)accS[(ss * M + oa) * G::KP + ob];
      out[(size_t)o * ncols] = s;
    }
    {
      const double l = warp_sum_f64(loss64), g0 = warp_sum_f64(gb064);
      if (lane == 0) { red64[warp] = l; red64[8 + warp] = g0; }
    }
    __syncthreads();
    if (tid == 0) {
      double ls = 0.0, gs = 0.0;
      for (int w = 0; w < kThreads / 32; ++w) { ls += red64[w]; gs += red64[8 + w]; }
      out[(size_t)(M * M) * ncols] = gs;
      out[(size_t)p.np * ncols] = ls;
    }
    __threadfence();
    cluster_sync_all();                                    // every partial column of this epoch is in global memory
    if (rank == 0) fit_step_body<CG::PER>(a, e, sc);
    __threadfence();
    cluster_sync_all();                                    // theta32 / done of the next pass are visible
  }
}

}  // namespace dia
