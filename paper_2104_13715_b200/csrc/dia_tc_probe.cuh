// dia_tc_probe.cuh -- one-CTA tcgen05 GEMM probe (measurement only): D[128][N] = sum_k A[r][k] B[n][k] with the operands
// built in shared memory from float32 arrays, in the layout and with the descriptors hess_tc_kernel uses (K-major, no
// swizzle, core matrices of 8 rows x 16 bytes) and ONE accumulation chain over all of K in TMEM.  It answers, on the
// hardware, the questions the design of dia_hess_tc.cuh rests on (profiles/r02_tc_hessian.md, tests/test_gpu_tc_probe.py):
// is the layout right (exact integer data), how does the tensor core round when it adds products to its float32
// accumulator, and what do split operands cost in accuracy as the chain grows.
//   mode 0  float16 operands (the inputs rounded to float16)      mode 1  float16 hi + lo split, terms lo lo .. hi hi
//   mode 2  tf32 operands                                         mode 3  tf32 big + small split, three terms
#pragma once
#include <cuda_fp16.h>

#include "dia_hess_tc.cuh"

namespace dia {

constexpr int kTcProbeKC = 64;          // k elements per chunk of the operand tiles

template <int ES>                       // byte offset of element (r, k) in a tile of R rows
__device__ __forceinline__ unsigned tc_probe_off(int r, int k, int R) {
  constexpr int EPC = 16 / ES;
  return (unsigned)((k / EPC) * (R / 8 * 128) + (r / 8) * 128 + (r % 8) * 16 + (k % EPC) * ES);
}
__device__ __forceinline__ void tc_mma_tf32(unsigned tmem_d, unsigned long long ad, unsigned long long bd, unsigned idesc,
                                            unsigned accumulate) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}\n" ::"r"(tmem_d),
      "l"(ad), "l"(bd), "r"(idesc), "r"(accumulate)
      : "memory");
}

__global__ void __launch_bounds__(128, 1) tc_probe_kernel(const float* __restrict__ A, const float* __restrict__ B,
                                                          float* __restrict__ D, int K, int N, int mode) {
  extern __shared__ __align__(128) unsigned char tcp_smem[];
  __shared__ unsigned tmem_slot;
  __shared__ __align__(8) unsigned long long bar_storage;
  const int tid = threadIdx.x, warp = tid >> 5;
  const bool tf = mode >= 2, split = (mode & 1) != 0;
  const int ES = tf ? 4 : 2;
  const unsigned bar = smem_u32(&bar_storage);
  const unsigned szA = 128u * kTcProbeKC * ES, szB = (unsigned)N * kTcProbeKC * ES;
  unsigned char* const sAh = tcp_smem;
  unsigned char* const sAl = sAh + szA;
  unsigned char* const sBh = sAl + szA;
  unsigned char* const sBl = sBh + szB;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(&tmem_slot)), "r"(256u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
  }
  if (tid == 0) { mbar_init(bar, 1u);  fence_mbar_init(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const unsigned tmem = tmem_slot;
  const unsigned fmt = tf ? 2u : 0u;
  const unsigned idesc = (1u << 4) | (fmt << 7) | (fmt << 10) | ((unsigned)(N >> 3) << 17) | ((128u >> 4) << 24);
  const unsigned lboA = 128 / 8 * 128, lboB = (unsigned)N / 8 * 128, sbo = 128;
  const int KS = 32 / ES;                 // k elements per MMA
  unsigned phase = 0, first = 1;
  for (int k0 = 0; k0 < K; k0 += kTcProbeKC) {
    if (k0 > 0) { mbar_wait(bar, phase);  phase ^= 1u;  tc_fence_after(); }      // the last chunk's MMAs have read the tiles
    for (int idx = tid; idx < (128 + N) * kTcProbeKC; idx += 128) {
      const int r = idx / kTcProbeKC, k = idx - r * kTcProbeKC;
      const bool isA = r < 128;
      const int rr = isA ? r : r - 128, R = isA ? 128 : N;
      const float x = isA ? A[(size_t)rr * K + k0 + k] : B[(size_t)rr * K + k0 + k];
      unsigned char* const th = isA ? sAh : sBh;
      unsigned char* const tl = isA ? sAl : sBl;
      if (!tf) {
        __half hi = __float2half_rn(x);
        if (split) {                      // the split of tc_build_row: 8 significant bits in hi
          const unsigned short hb = (unsigned short)((*reinterpret_cast<const unsigned short*>(&hi) + (1u << (DIA_TC_HI_DROP - 1))) &
                                                     ~((1u << DIA_TC_HI_DROP) - 1u));
          hi = *reinterpret_cast<const __half*>(&hb);
        }
        *reinterpret_cast<__half*>(th + tc_probe_off<2>(rr, k, R)) = hi;
        *reinterpret_cast<__half*>(tl + tc_probe_off<2>(rr, k, R)) = __float2half_rn(x - __half2float(hi));
      } else {
        unsigned big;
        asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(big) : "f"(x));
        *reinterpret_cast<unsigned*>(th + tc_probe_off<4>(rr, k, R)) = big;
        *reinterpret_cast<float*>(tl + tc_probe_off<4>(rr, k, R)) = x - __uint_as_float(big);
      }
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    if (tid == 0) {
      tc_fence_after();
      const int n_term = split ? (tf ? 3 : 4) : 1;
      for (int term = 0; term < n_term; ++term) {      // small terms first
        const bool a_lo = split && (tf ? term == 0 : term < 2), b_lo = split && (tf ? term == 1 : (term & 1) == 0);
        const unsigned ta = smem_u32(a_lo ? sAl : sAh), tb = smem_u32(b_lo ? sBl : sBh);
        for (int s = 0; s < kTcProbeKC / KS; ++s) {
          const unsigned long long ad = tc_smem_desc(ta + s * 2 * lboA, lboA, sbo), bd = tc_smem_desc(tb + s * 2 * lboB, lboB, sbo);
          if (tf) tc_mma_tf32(tmem, ad, bd, idesc, first ? 0u : 1u);
          else tc_mma_f16(tmem, ad, bd, idesc, first ? 0u : 1u);
          first = 0;
        }
      }
      tc_commit(bar);
    }
  }
  mbar_wait(bar, phase);
  tc_fence_after();
  for (int c = 0; c < N; c += 32) {       // thread (warp, lane) owns row 32 warp + lane
    float v[32];
#pragma unroll
    for (int j = 0; j < 32; ++j) v[j] = 0.f;
    tc_flush32(tmem + ((unsigned)(warp * 32) << 16) + (unsigned)c, v);
#pragma unroll
    for (int j = 0; j < 32; ++j) D[(size_t)tid * N + c + j] = v[j];
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem), "r"(256u) : "memory");
}

// K a positive multiple of 64, N in {32, 64, ..., 256}; returns a cudaError_t
inline cudaError_t tc_probe_launch(cudaStream_t stream, const float* d_A, const float* d_B, float* d_D, int K, int N, int mode) {
  const size_t smem = (size_t)2 * (128 + N) * kTcProbeKC * (mode >= 2 ? 4 : 2);
  cudaError_t ce = cudaFuncSetAttribute(tc_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (ce != cudaSuccess) return ce;
  tc_probe_kernel<<<1, 128, smem, stream>>>(d_A, d_B, d_D, K, N, mode);
  return cudaGetLastError();
}

}  // namespace dia
