// dia_probe.cuh -- register-only FFMA microbenchmark: the measured FP32 FMA peak that the roofline of the
// fused kernel is reported against.  Every thread runs 16 independent accumulator
// chains acc[i] += k[j] * r[i + j] -- the operand pattern of the stencil's inner loop -- with no memory traffic.
#pragma once
#include <cuda_runtime.h>

namespace dia {

constexpr int kProbeAcc = 16, kProbeTaps = 8;

__global__ void __launch_bounds__(256) fp32_peak_kernel(float* out, int iters, float a0, float b0) {
  float acc[kProbeAcc], k[kProbeTaps], r[kProbeAcc + kProbeTaps];
#pragma unroll
  for (int i = 0; i < kProbeAcc; ++i) acc[i] = 0.f;
#pragma unroll
  for (int i = 0; i < kProbeTaps; ++i) k[i] = a0 + i * 1e-6f;
#pragma unroll
  for (int i = 0; i < kProbeAcc + kProbeTaps; ++i) r[i] = b0 + i * 1e-7f + threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kProbeTaps; ++j)
#pragma unroll
      for (int i = 0; i < kProbeAcc; ++i) acc[i] = fmaf(k[j], r[i + j], acc[i]);
    r[it & (kProbeTaps - 1)] += 1.0f;
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < kProbeAcc; ++i) s += acc[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// Best of `reps` timed launches; returns FMA/s (thread-level fused multiply-adds per second) or < 0 on error.
inline double measure_fp32_peak(cudaStream_t stream, int reps) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -1.0;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1.0;
  const int blocks = sms * 4, threads = 256, iters = 8192;
  float* out = nullptr;
  if (cudaMalloc(&out, sizeof(float) * blocks * threads) != cudaSuccess) return -1.0;
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  fp32_peak_kernel<<<blocks, threads, 0, stream>>>(out, iters / 8, 0.999f, 0.001f);   // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < reps; ++rep) {
    cudaEventRecord(a, stream);
    fp32_peak_kernel<<<blocks, threads, 0, stream>>>(out, iters, 0.999f, 0.001f);
    cudaEventRecord(b, stream);
    if (cudaEventSynchronize(b) != cudaSuccess) { best = -1.f; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  cudaFree(out);
  if (best <= 0.f) return -1.0;
  const double fma = (double)kProbeAcc * kProbeTaps * iters * (double)blocks * threads;
  return fma / (best * 1e-3);
}

}  // namespace dia
