// alu_peak.cu — FMA-chain microbenchmark behind mg_measure_alu_peak(): the measured denominator of
// the "alu" roofline ("confirm with a DFMA/FFMA-chain microbenchmark on the box").
// Every thread runs 16 independent accumulator chains of a*x+b; nothing is read from memory.
#include "mg_internal.h"

namespace mg {
namespace {

template <class T> __device__ __forceinline__ T fma_t(T a, T b, T c);
template <> __device__ __forceinline__ double fma_t(double a, double b, double c) { return fma(a, b, c); }
template <> __device__ __forceinline__ float fma_t(float a, float b, float c) { return fmaf(a, b, c); }

template <class T, int CHAINS>
__global__ void __launch_bounds__(256) fma_chain_kernel(T a, T b, int iters, T* __restrict__ out) {
  T x[CHAINS];
#pragma unroll
  for (int i = 0; i < CHAINS; ++i) x[i] = (T)(threadIdx.x + i) * (T)1e-3;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int i = 0; i < CHAINS; ++i) x[i] = fma_t<T>(x[i], a, b);
  }
  T s = 0;
#pragma unroll
  for (int i = 0; i < CHAINS; ++i) s += x[i];
  if (s == (T)123456789) out[0] = s;  // never true; keeps the chains alive
}

template <class T>
cudaError_t run(int sm_count, double* tflops) {
  constexpr int CHAINS = 16;
  const int blocks = sm_count * 8, threads = 256, iters = 4096;
  T* d = nullptr;
  cudaError_t e = cudaMalloc(&d, sizeof(T));
  if (e != cudaSuccess) return e;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0);
    fma_chain_kernel<T, CHAINS><<<blocks, threads>>>((T)0.999999, (T)1e-7, iters, d);
    cudaEventRecord(e1);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    const double flops = 2.0 * CHAINS * 8.0 * iters * (double)blocks * threads;
    if (rep > 0 && ms > 0) best = fmax(best, flops / (ms * 1e-3) * 1e-12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  *tflops = best;
  return e == cudaSuccess ? cudaGetLastError() : e;
}

}  // namespace

cudaError_t measure_alu_peak(int precision, int device, double* tflops) {
  cudaDeviceProp prop;
  cudaError_t e = cudaGetDeviceProperties(&prop, device);
  if (e != cudaSuccess) return e;
  return precision == MG_FP64 ? run<double>(prop.multiProcessorCount, tflops) : run<float>(prop.multiProcessorCount, tflops);
}

}  // namespace mg
