// alu_peak.cu — FMA microbenchmarks behind include/mg_probe.h (libmg_probe.so, NOT part of the product library):
// the measured denominators of the "alu" roofline ("confirm with a DFMA/FFMA-chain microbenchmark
// on the box").  Every thread runs independent accumulator chains; nothing is read from memory.
#include <cuda_runtime.h>
#include "../../include/mg_probe.h"

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

// mode 1: every FMA reads THREE distinct registers (what products of two loaded operands accumulate into).
// On B200 the FP64 FMA then issues once per 3 cycles instead of 2 (three 64-bit operands through a two-bank
// register file; the operand-reuse cache and constant operands avoid it) — DESIGN.md §6.
template <class T, int N>
__global__ void __launch_bounds__(256) fma3_kernel(int iters, T* __restrict__ out) {
  T x[N];
#pragma unroll
  for (int i = 0; i < N; ++i) x[i] = (T)1 + (T)(threadIdx.x + i) * (T)1e-9;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < N; ++i) x[i] = fma_t<T>(x[(i + 5) % N], x[(i + 11) % N], x[i]);
  }
  T s = 0;
#pragma unroll
  for (int i = 0; i < N; ++i) s += x[i];
  if (s == (T)123456789) out[0] = s;
}

// mode 2: FP64 tensor-core path, mma.sync m8n8k4 (DMMA): 256 FMA per warp instruction, 8 independent accumulators
__global__ void __launch_bounds__(256) dmma_kernel(int iters, double* __restrict__ out) {
  double c[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i] = threadIdx.x * 1e-4 + i;
  const double a = 1.0000001, b = 0.5;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[2 * i]), "+d"(c[2 * i + 1]) : "d"(a), "d"(b));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i];
  if (s == 123456789.0) out[0] = s;
}

template <class T>
cudaError_t run_mode(int sm_count, int mode, double* tflops) {
  const int blocks = sm_count * 8, threads = 256, iters = 4096;
  T* d = nullptr;
  cudaError_t e = cudaMalloc(&d, sizeof(T));
  if (e != cudaSuccess) return e;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0);
    double flops;
    if (mode == 1) {
      fma3_kernel<T, 24><<<blocks, threads>>>(iters, d);
      flops = 2.0 * 24 * iters * (double)blocks * threads;
    } else {
      dmma_kernel<<<blocks, threads>>>(iters, reinterpret_cast<double*>(d));
      flops = 2.0 * 8 * 8 * 4 * 8.0 * iters * (double)blocks * threads / 32;
    }
    cudaEventRecord(e1);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms > 0) best = fmax(best, flops / (ms * 1e-3) * 1e-12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  *tflops = best;
  return e == cudaSuccess ? cudaGetLastError() : e;
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

cudaError_t measure_alu_peak(int precision, int device, int mode, double* tflops) {
  cudaDeviceProp prop;
  cudaError_t e = cudaGetDeviceProperties(&prop, device);
  if (e != cudaSuccess) return e;
  if (mode == 1) return precision == 0 ? run_mode<double>(prop.multiProcessorCount, 1, tflops) : run_mode<float>(prop.multiProcessorCount, 1, tflops);
  if (mode == 2) return run_mode<double>(prop.multiProcessorCount, 2, tflops);
  return precision == 0 ? run<double>(prop.multiProcessorCount, tflops) : run<float>(prop.multiProcessorCount, tflops);
}

}  // namespace mg

extern "C" int mg_probe_alu(int precision, int device, int mode, double* h_tflops_out) {
  if (!h_tflops_out || device < 0 || (precision != 0 && precision != 1) || mode < 0 || mode > 2) return -1;
  if (mode == 2 && precision != 0) return -1;
  int ndev = 0, prev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device >= ndev) { cudaGetLastError(); return -3; }
  cudaGetDevice(&prev);
  cudaSetDevice(device);
  const cudaError_t e = mg::measure_alu_peak(precision, device, mode, h_tflops_out);
  cudaSetDevice(prev);
  return e == cudaSuccess ? 0 : -3;
}
