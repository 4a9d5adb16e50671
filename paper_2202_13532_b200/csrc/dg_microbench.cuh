// FP64 arithmetic peak of the device, measured: the denominator of the "alu" roofline of the dense Fourier contraction
// (field_gemm_tn_kernel: DFMA; field_gemm_dmma_kernel: DMMA m8n8k4).  Register-resident dependent chains, 16 (DFMA) or
// 8 (DMMA) independent accumulators per thread, full occupancy; nothing touches memory until the final store.
#pragma once
#include <cuda_runtime.h>

namespace dgmb {

__global__ void __launch_bounds__(256) dfma_peak_kernel(double* out, int iters) {
  double a[16];
  const double x = threadIdx.x * 1e-9, y = 1.0000001;
#pragma unroll
  for (int i = 0; i < 16; ++i) a[i] = i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = fma(a[i], y, x);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += a[i];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) dmma_peak_kernel(double* out, int iters) {
  double c[8][2];
  const double a = threadIdx.x * 1e-9, b = 1.0000001;
#pragma unroll
  for (int i = 0; i < 8; ++i) c[i][0] = c[i][1] = i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                   : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// variant 0: DFMA, 1: DMMA.  Returns the elapsed device time of `iters` iterations on `blocks` CTAs of 256 threads.
inline cudaError_t run_peak(int variant, int blocks, int iters, double* scratch, cudaStream_t st, float* ms) {
  cudaEvent_t e0, e1;
  cudaError_t e = cudaEventCreate(&e0);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&e1);
  if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
  if (variant == 0) dfma_peak_kernel<<<blocks, 256, 0, st>>>(scratch, 64);
  else dmma_peak_kernel<<<blocks, 256, 0, st>>>(scratch, 64);
  cudaEventRecord(e0, st);
  if (variant == 0) dfma_peak_kernel<<<blocks, 256, 0, st>>>(scratch, iters);
  else dmma_peak_kernel<<<blocks, 256, 0, st>>>(scratch, iters);
  cudaEventRecord(e1, st);
  e = cudaEventSynchronize(e1);
  if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return e;
}

}  // namespace dgmb
