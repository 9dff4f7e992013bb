// FP32 FMA peak of the device, measured: a register-resident FFMA chain (8 independent accumulators per thread, 8 CTAs of
// 256 threads per SM).  SURVEY.md 8(d) asks for this number beside the ALU-bound kernels' roofline; bench.py reports it
// next to the peak derived from the unit counts (148 SMs x 128 lanes x 2 flop x clock).
#include "rga_internal.h"

__global__ void __launch_bounds__(256) fma_peak_kernel(float* __restrict__ out, int iters) {
  float a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const float m = 1.0001f, c = 0.5f;
  for (int i = 0; i < iters; ++i) {
    a0 = fmaf(a0, m, c); a1 = fmaf(a1, m, c); a2 = fmaf(a2, m, c); a3 = fmaf(a3, m, c);
    a4 = fmaf(a4, m, c); a5 = fmaf(a5, m, c); a6 = fmaf(a6, m, c); a7 = fmaf(a7, m, c);
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

extern "C" rga_status rga_measure_fp32_peak(void* stream, float* tflops) {
  if (!tflops) return RGA_ERR_INVALID_ARG;
  *tflops = 0.f;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return RGA_ERR_CUDA;
  cudaStream_t s = (cudaStream_t)stream;
  float* d = nullptr;
  const int grid = sms * 8, iters = 20000;
  if (cudaMalloc(&d, (size_t)grid * 256 * sizeof(float)) != cudaSuccess) return RGA_ERR_OOM;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {                     // first repetition warms up; best of the rest
    cudaEventRecord(e0, s);
    fma_peak_kernel<<<grid, 256, 0, s>>>(d, iters);
    cudaEventRecord(e1, s);
    cudaEventSynchronize(e1);
    float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  if (cudaGetLastError() != cudaSuccess) return RGA_ERR_CUDA;
  *tflops = (float)((double)grid * 256 * iters * 8 * 2 / (best * 1e-3) / 1e12);
  return RGA_OK;
}
