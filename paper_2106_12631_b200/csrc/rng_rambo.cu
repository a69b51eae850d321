// rng_rambo.cu — steps A1-A4 of the hot path: Philox4x32-10 words, uniforms,
// RAMBO massless generation and massive rescaling.  One thread per event; every global access is
// a row of the SoA arrays indexed by the event, so a warp reads/writes 32 consecutive elements
// (coalesced access).  Both kernels are HBM-bound.
//
// RAMBO follows Kleiss, Stirling, Ellis, CPC 40 (1986) 359 ("RAMBO [39]"), readings
// R5-R8 of DESIGN.md; the paper prints no equations.
#include "mg_internal.h"
#include "philox.cuh"
#include "rambo.cuh"

namespace mg {

namespace {

constexpr int kThreads = 256;
constexpr int kMinBlocks = 3;      // RAMBO kernels: 24 warps per SM (80 registers) hide the sqrt / division / log chains better than 16 at 124


__global__ void __launch_bounds__(kThreads) rng_words_kernel(uint64_t seed, uint64_t first, int64_t n, int64_t ld,
                                                             int nf, uint32_t* __restrict__ out) {
  const int64_t e = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (e >= n) return;
  for (int i = 0; i < nf; ++i) {
    const u32x4 r = philox_event_particle(seed, first + (uint64_t)e, (uint32_t)i);
    uint32_t* o = out + (int64_t)(4 * i) * ld + e;
    o[0] = r.x; o[ld] = r.y; o[2 * ld] = r.z; o[3 * ld] = r.w;
  }
}

template <class T, int NF>
__global__ void __launch_bounds__(kThreads) rng_kernel(uint64_t seed, uint64_t first, int64_t n, int64_t ld,
                                                       T* __restrict__ out) {
  const int64_t e = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (e >= n) return;
#pragma unroll
  for (int i = 0; i < NF; ++i) {
    const u32x4 r = philox_event_particle(seed, first + (uint64_t)e, (uint32_t)i);
    T* o = out + (int64_t)(4 * i) * ld + e;
    __stcs(o, u32_to_uniform<T>(r.x));
    __stcs(o + ld, u32_to_uniform<T>(r.y));
    __stcs(o + 2 * ld, u32_to_uniform<T>(r.z));
    __stcs(o + 3 * ld, u32_to_uniform<T>(r.w));
  }
}

template <class T, int NF, bool MASSIVE>
__device__ __forceinline__ void rambo_event(const T (&rho)[4 * NF], const Consts& k, int64_t e, int64_t ld,
                                            T* __restrict__ mom, T* __restrict__ wout) {
  T p[NF][4];
  const T w = rambo_core<T, NF, MASSIVE>(rho, k, p);
  // beams (R5)
  const T hs = (T)0.5 * (T)k.sqrt_s;
  T* o = mom + e;
  __stcs(o + 0 * ld, hs); __stcs(o + 1 * ld, (T)0); __stcs(o + 2 * ld, (T)0); __stcs(o + 3 * ld, hs);
  __stcs(o + 4 * ld, hs); __stcs(o + 5 * ld, (T)0); __stcs(o + 6 * ld, (T)0); __stcs(o + 7 * ld, -hs);
#pragma unroll
  for (int i = 0; i < NF; ++i)
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) __stcs(o + (int64_t)(8 + 4 * i + mu) * ld, p[i][mu]);
  if (wout) __stcs(wout + e, w);
}

template <class T, int NF, bool MASSIVE>
__global__ void __launch_bounds__(kThreads, kMinBlocks) rambo_kernel(Consts k, const T* __restrict__ rnd, int64_t n, int64_t ld,
                                                         T* __restrict__ mom, T* __restrict__ wout) {
  const int64_t e = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (e >= n) return;
  T rho[4 * NF];
#pragma unroll
  for (int j = 0; j < 4 * NF; ++j) rho[j] = __ldcs(rnd + (int64_t)j * ld + e);
  rambo_event<T, NF, MASSIVE>(rho, k, e, ld, mom, wout);
}

// A1-A4 fused: the uniforms stay in registers.
template <class T, int NF, bool MASSIVE>
__global__ void __launch_bounds__(kThreads, kMinBlocks) generate_kernel(Consts k, uint64_t seed, uint64_t first, int64_t n,
                                                            int64_t ld, T* __restrict__ mom, T* __restrict__ wout) {
  const int64_t e = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (e >= n) return;
  T rho[4 * NF];
#pragma unroll
  for (int i = 0; i < NF; ++i) {
    const u32x4 r = philox_event_particle(seed, first + (uint64_t)e, (uint32_t)i);
    rho[4 * i + 0] = u32_to_uniform<T>(r.x);
    rho[4 * i + 1] = u32_to_uniform<T>(r.y);
    rho[4 * i + 2] = u32_to_uniform<T>(r.z);
    rho[4 * i + 3] = u32_to_uniform<T>(r.w);
  }
  rambo_event<T, NF, MASSIVE>(rho, k, e, ld, mom, wout);
}

inline unsigned blocks_for(int64_t n) { return (unsigned)((n + kThreads - 1) / kThreads); }

template <class T>
cudaError_t rng_dispatch(int nf, uint64_t seed, uint64_t first, int64_t n, int64_t ld, T* out, cudaStream_t s) {
  const unsigned g = blocks_for(n);
  switch (nf) {
    case 2: rng_kernel<T, 2><<<g, kThreads, 0, s>>>(seed, first, n, ld, out); break;
    case 3: rng_kernel<T, 3><<<g, kThreads, 0, s>>>(seed, first, n, ld, out); break;
    case 4: rng_kernel<T, 4><<<g, kThreads, 0, s>>>(seed, first, n, ld, out); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

template <class T>
cudaError_t rambo_dispatch(const mg_process* p, const T* rnd, int64_t n, int64_t ld, T* mom, T* w, cudaStream_t s) {
  const unsigned g = blocks_for(n);
  const bool massive = p->par.process != MG_EEMUMU;
  switch (p->n_final) {
    case 2:
      if (massive) rambo_kernel<T, 2, true><<<g, kThreads, 0, s>>>(p->k, rnd, n, ld, mom, w);
      else rambo_kernel<T, 2, false><<<g, kThreads, 0, s>>>(p->k, rnd, n, ld, mom, w);
      break;
    case 3: rambo_kernel<T, 3, true><<<g, kThreads, 0, s>>>(p->k, rnd, n, ld, mom, w); break;
    case 4: rambo_kernel<T, 4, true><<<g, kThreads, 0, s>>>(p->k, rnd, n, ld, mom, w); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

template <class T>
cudaError_t generate_dispatch(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, int64_t ld, T* mom, T* w,
                              cudaStream_t s) {
  const unsigned g = blocks_for(n);
  const bool massive = p->par.process != MG_EEMUMU;
  switch (p->n_final) {
    case 2:
      if (massive) generate_kernel<T, 2, true><<<g, kThreads, 0, s>>>(p->k, seed, first, n, ld, mom, w);
      else generate_kernel<T, 2, false><<<g, kThreads, 0, s>>>(p->k, seed, first, n, ld, mom, w);
      break;
    case 3: generate_kernel<T, 3, true><<<g, kThreads, 0, s>>>(p->k, seed, first, n, ld, mom, w); break;
    case 4: generate_kernel<T, 4, true><<<g, kThreads, 0, s>>>(p->k, seed, first, n, ld, mom, w); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_rng_words(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, int64_t ld,
                             uint32_t* d_words, cudaStream_t s) {
  rng_words_kernel<<<blocks_for(n), kThreads, 0, s>>>(seed, first, n, ld, p->n_final, d_words);
  return cudaGetLastError();
}

cudaError_t launch_rng(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, int64_t ld, void* d_rnd,
                       cudaStream_t s) {
  if (p->par.precision == MG_FP64) return rng_dispatch<double>(p->n_final, seed, first, n, ld, (double*)d_rnd, s);
  return rng_dispatch<float>(p->n_final, seed, first, n, ld, (float*)d_rnd, s);
}

cudaError_t launch_rambo(const mg_process* p, const void* d_rnd, int64_t n, int64_t ld, void* d_mom, void* d_w,
                         cudaStream_t s) {
  if (p->par.precision == MG_FP64)
    return rambo_dispatch<double>(p, (const double*)d_rnd, n, ld, (double*)d_mom, (double*)d_w, s);
  return rambo_dispatch<float>(p, (const float*)d_rnd, n, ld, (float*)d_mom, (float*)d_w, s);
}

cudaError_t launch_generate(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, int64_t ld, void* d_mom,
                            void* d_w, cudaStream_t s) {
  if (p->par.precision == MG_FP64) return generate_dispatch<double>(p, seed, first, n, ld, (double*)d_mom, (double*)d_w, s);
  return generate_dispatch<float>(p, seed, first, n, ld, (float*)d_mom, (float*)d_w, s);
}

}  // namespace mg
