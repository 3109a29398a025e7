// dia_fit_cluster.cuh -- the whole fit of a SMALL image pair inside one kernel: one thread-block cluster per epoch.
//
// For images of a few tiles (128^2 - 142^2 stamps: 4 tiles; SURVEY.md section 7 hard part 4) an evaluation is ~1 us of
// arithmetic, and the graph loop of dia_fit.cuh spends ~13 us per iteration on two kernel launches, tile staging and
// reduction latency.  Here a cluster of T = tiles CTAs (T <= 8) owns one epoch for the whole fit:
//   once       every CTA stages ITS tile of R (+ halo) and of I into shared memory (TMA or cp.async) and keeps them;
//   iteration  K and B0 from this CTA's shared-memory copy of theta -> forward stencil, residual, noise model, loss,
//              weights -> gradient correlation (the device functions of eval_kernel, same arithmetic, same orders) ->
//              this CTA's FP64 partial column, in ITS shared memory -> cluster barrier -> rank 0 runs the optimiser
//              transition (fit_step_body: second-level reduction reading the columns of all CTAs through distributed
//              shared memory, Adam or L-BFGS step, stop tests) and stores the next evaluation point and the done
//              flag into every CTA's shared memory -> cluster barrier -> next iteration, until done.
// No host round trip, no launch, no re-staging and no global-memory hand-over per iteration (the optimiser state --
// FP64 theta, moments, L-BFGS history -- stays in global memory and is touched by rank 0 only).  Epochs are independent clusters, so a batch of hundreds
// of stamps is one launch; clusters that finish make room for the next.  Plain objective only (no mask / flat /
// variance map / background polynomial): dia_fit falls back to the graph loop otherwise.  For an image whose tiles
// all sit on different CTAs in the graph loop (single image pairs) the results are bit-identical to it (tested).
#pragma once
#include <cooperative_groups.h>

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
  static constexpr int NP = M * M + 1;
  // the optimiser's scratch, then the exchange area: this CTA's partial column [np + 1] doubles, theta [np] floats, the
  // table of peer columns, the done flag
  static constexpr size_t SCRATCH = (step_scratch_bytes<PER>() + 15) / 16 * 16;
  static constexpr size_t X_PCOL = SCRATCH;
  static constexpr size_t X_TH = X_PCOL + 8 * (NP + 1);
  static constexpr size_t X_PEERS = (X_TH + 4 * NP + 15) / 16 * 16;
  static constexpr size_t X_DONE = X_PEERS + 8 * 16;
  static constexpr size_t EXTRA = X_DONE + 16;
  // both take the second R buffer when there is one and it is large enough (m = 19: two CTAs per SM as in eval_kernel),
  // else they are appended
  static constexpr bool IN_RBUF = G::NRBUF == 2 && (size_t)G::R_STRIDE >= EXTRA;
  static constexpr size_t OFF_SCRATCH = IN_RBUF ? (size_t)G::R_STRIDE : ((G::SMEM + 15) / 16 * 16);
  static constexpr size_t OFF_PCOL = OFF_SCRATCH + X_PCOL, OFF_TH = OFF_SCRATCH + X_TH, OFF_PEERS = OFF_SCRATCH + X_PEERS,
                          OFF_DONE = OFF_SCRATCH + X_DONE;
  static constexpr size_t SMEM = IN_RBUF ? G::SMEM : OFF_SCRATCH + EXTRA + 128;
};

#ifdef DIA_CLUSTER_PROFILE
__device__ long long g_cl_prof[16];
#define CL_T(k) do { if (blockIdx.x == 0 && threadIdx.x == 0) { const long long t_ = clock64(); g_cl_prof[k] += t_ - cl_t0; cl_t0 = t_; } } while (0)
#else
#define CL_T(k) do { } while (0)
#endif

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
  double* const pcol = reinterpret_cast<double*>(sm + CG::OFF_PCOL);          // this CTA's partial column
  float* const thl = reinterpret_cast<float*>(sm + CG::OFF_TH);              // theta of the next evaluation
  const double** const peers = reinterpret_cast<const double**>(sm + CG::OFF_PEERS);
  int* const done_l = reinterpret_cast<int*>(sm + CG::OFF_DONE);
  StepScratch sc;
  sc.sh_rows = reinterpret_cast<double (*)[kFitThreads / 32]>(scr);
  sc.s_alpha = scr + 2 * (kFitThreads / 32);
  sc.gsum = sc.s_alpha + kMaxHistory;
  sc.xs = sc.gsum + kFitThreads * CG::PER;
  sc.peer_cols = peers;  sc.th_local = thl;  sc.done_local = done_l;

  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n_tiles = p.tiles_x * p.tiles_y;               // == cluster size
  const int rank = (int)cluster.block_rank();
  const int e = (int)blockIdx.x / n_tiles, tile = rank;
  const int vr = p.n_rows - M + 1, vc = p.n_cols - M + 1;
  const size_t npix = (size_t)p.n_rows * p.n_cols;
  const int tile_y = tile / p.tiles_x, tile_x = tile - tile_y * p.tiles_x;
  const int np = p.np;                                     // == M * M + 1 (no background polynomial here)

  if (tid == 0) {
    const unsigned cnt = p.use_tma ? 1u : (unsigned)kThreads;
#pragma unroll
    for (int b = 0; b < 3; ++b) mbar_init(bar0 + 8u * b, cnt);
    fence_mbar_init();
    *done_l = 0;
  }
  if (rank == 0 && tid < n_tiles) peers[tid] = cluster.map_shared_rank(pcol, tid);
  for (int k = tid; k < np; k += kThreads) thl[k] = p.theta[(size_t)e * np + k];     // fit_init_kernel's theta32
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
  const bool edge = (tile_y * kTH + kTH > vr) || (tile_x * kTW + kTW > vc);
  const int rows_here = min(kTH, vr - tile_y * kTH);
  const int n_items = rows_here * (kTW / kP);
  if (tid < kMaxBg) Bs[tid] = 0.f;
  cluster.sync();                                          // every CTA of the cluster has started (its shared memory exists)

#ifdef DIA_CLUSTER_PROFILE
  long long cl_t0 = clock64();
#endif
  while (true) {
    if (*done_l) break;                                    // stored by rank 0 before the barrier that ended the last pass
    for (int idx = tid; idx < G::K_FLOATS; idx += kThreads) {
      const int ka = idx / G::KP, kb = idx - ka * G::KP;
      Ks[idx] = (kb < M) ? thl[ka * M + kb] : 0.f;
    }
    const float B0 = thl[M * M];
#pragma unroll
    for (int q = 0; q < G::KP / 4; ++q) myacc[q] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();
    CL_T(0);
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
    CL_T(1);
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
    CL_T(2);
    fold_strips<M>(accS, tid, [&](int o, double s) { pcol[o] = s; });      // the order of eval_kernel's flush
    {
      const double l = warp_sum_f64(loss64), g0 = warp_sum_f64(gb064);
      if (lane == 0) { red64[warp] = l; red64[8 + warp] = g0; }
    }
    __syncthreads();
    if (tid == 0) {
      double ls = 0.0, gs = 0.0;
      for (int w = 0; w < kThreads / 32; ++w) { ls += red64[w]; gs += red64[8 + w]; }
      pcol[M * M] = gs;
      pcol[np] = ls;
    }
    CL_T(3);
    cluster.sync();                                        // every partial column of this epoch is complete
    CL_T(4);
    if (rank == 0) {
      fit_step_body<CG::PER>(a, e, sc);                    // leaves the next theta in thl, the done flag in done_l
      __syncthreads();
      CL_T(5);
      for (int r = 1; r < n_tiles; ++r) {                  // hand both to the other CTAs of the cluster
        float* rth = cluster.map_shared_rank(thl, r);
        for (int k = tid; k < np; k += kThreads) rth[k] = thl[k];
        if (tid == 0) *cluster.map_shared_rank(done_l, r) = *done_l;
      }
    }
    CL_T(6);
    cluster.sync();                                        // theta / done of the next pass are in place; pcol is free
    CL_T(7);
  }
}

}  // namespace dia
