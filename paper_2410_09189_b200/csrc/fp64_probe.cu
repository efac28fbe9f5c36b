// fp64_probe.cu -- calibration instrument, not part of the hot path: measures the FP64 issue-rate ceilings of the
// device the roofline fractions are quoted against ("a hand-written DMMA-issue microbenchmark and a DFMA
// one").  Register-resident operands, 16 independent accumulator chains per warp, 16 warps per SM.
#include "../../include/rt_tddft.h"
#include <cuda_runtime.h>

namespace {

constexpr int NACC = 16;

__global__ void __launch_bounds__(256) probe_dmma(double* out, int iters, double a0, double b0) {
  double acc[NACC][2];
#pragma unroll
  for (int i = 0; i < NACC; ++i) acc[i][0] = acc[i][1] = 0.0;
  const double a = a0 + threadIdx.x * 1e-9, b = b0;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < NACC; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                   : "+d"(acc[i][0]), "+d"(acc[i][1]) : "d"(a), "d"(b));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) s += acc[i][0] + acc[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) probe_dfma(double* out, int iters, double a0, double b0) {
  double acc[NACC];
#pragma unroll
  for (int i = 0; i < NACC; ++i) acc[i] = i;
  const double a = a0 + threadIdx.x * 1e-9, b = b0;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = fma(acc[i], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) s += acc[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

extern "C" int rt_probe_fp64_peak(int32_t device, double* dmma_tflops, double* dfma_tflops) {
  if (!dmma_tflops || !dfma_tflops) return RT_EINVAL;
  cudaDeviceProp p;
  if (cudaSetDevice(device) != cudaSuccess || cudaGetDeviceProperties(&p, device) != cudaSuccess) {
    cudaGetLastError();
    return RT_ECUDA;
  }
  const int blocks = p.multiProcessorCount * 2, threads = 256;
  double* out = nullptr;
  if (cudaMalloc(&out, sizeof(double) * blocks * threads) != cudaSuccess) { cudaGetLastError(); return RT_ENOMEM; }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float ms = 0;
  double best_mma = 0, best_fma = 0;
  for (int rep = 0; rep < 3; ++rep) {
    const int it_mma = 100000;            // ~50 ms
    probe_dmma<<<blocks, threads>>>(out, rep == 0 ? 1000 : it_mma, 1.0, 1e-3);
    cudaEventRecord(e0);
    probe_dmma<<<blocks, threads>>>(out, it_mma, 1.0, 1e-3);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    cudaEventElapsedTime(&ms, e0, e1);
    double tf = 2.0 * 256 * NACC * (double)it_mma * blocks * (threads / 32) / (ms * 1e9);
    if (tf > best_mma) best_mma = tf;
    const int it_fma = 400000;
    cudaEventRecord(e0);
    probe_dfma<<<blocks, threads>>>(out, it_fma, 1.0000001, 1e-3);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    cudaEventElapsedTime(&ms, e0, e1);
    tf = 2.0 * NACC * (double)it_fma * blocks * threads / (ms * 1e9);
    if (tf > best_fma) best_fma = tf;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  if (cudaGetLastError() != cudaSuccess) return RT_ECUDA;
  *dmma_tflops = best_mma;
  *dfma_tflops = best_fma;
  return RT_OK;
}
