// rng_rambo.cu — steps A1-A4 of the hot path: Philox4x32-10 words, uniforms,
// RAMBO massless generation and massive rescaling.  One thread per event; every global access is
// a row of the SoA arrays indexed by the event, so a warp reads/writes 32 consecutive elements
// (coalesced access).  Both kernels are HBM-bound.
//
// RAMBO follows Kleiss, Stirling, Ellis, CPC 40 (1986) 359 ("RAMBO [39]"), readings
// R5-R8 of DESIGN.md; the paper prints no equations.
#include "mg_internal.h"
#include "philox.cuh"

namespace mg {

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ void sincospi_(double x, double* s, double* c) { sincospi(x, s, c); }
__device__ __forceinline__ void sincospi_(float x, float* s, float* c) { sincospif(x, s, c); }
__device__ __forceinline__ double log_(double x) { return log(x); }
__device__ __forceinline__ float log_(float x) { return logf(x); }

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

// One event of RAMBO.  rho[4*i+k]; writes momenta rows (beams + NF finals) and the weight.
//   massless (KSE eq. for q_i, boost b, scale x);  c = 2 rho1 - 1, sqrt(1-c^2) = 2 sqrt(rho1 (1-rho1))
//   (same value, no cancellation near |c| = 1: R19).
//   massive: Newton on f(xi) = sum_i sqrt(m_i^2 + xi^2 p_i0^2) - sqrt_s, fixed iteration count
//   (lock-step; converged to rounding well before the last step, R7).
template <class T, int NF, bool MASSIVE>
__device__ __forceinline__ void rambo_event(const T (&rho)[4 * NF], const Consts& k, int64_t e, int64_t ld,
                                            T* __restrict__ mom, T* __restrict__ wout) {
  T q[NF][4];
  T Q0 = 0, Q1 = 0, Q2 = 0, Q3 = 0;
#pragma unroll
  for (int i = 0; i < NF; ++i) {
    const T r1 = rho[4 * i + 0], r2 = rho[4 * i + 1], r3 = rho[4 * i + 2], r4 = rho[4 * i + 3];
    const T c = fma_<T>((T)2, r1, (T)-1);
    const T st = (T)2 * sqrt_<T>(r1 * ((T)1 - r1));
    T sp, cp;
    sincospi_((T)2 * r2, &sp, &cp);
    const T q0 = -log_(r3 * r4);
    q[i][0] = q0;
    q[i][1] = q0 * st * cp;
    q[i][2] = q0 * st * sp;
    q[i][3] = q0 * c;
    Q0 += q[i][0]; Q1 += q[i][1]; Q2 += q[i][2]; Q3 += q[i][3];
  }
  const T sqrt_s = (T)k.sqrt_s;
  const T M2 = Q0 * Q0 - Q1 * Q1 - Q2 * Q2 - Q3 * Q3;
  const T M = sqrt_<T>(M2);
  const T iM = (T)1 / M;
  const T b1 = -Q1 * iM, b2 = -Q2 * iM, b3 = -Q3 * iM;
  const T x = sqrt_s * iM;
  const T gamma = Q0 * iM;
  const T a = (T)1 / ((T)1 + gamma);
  T p[NF][4];
#pragma unroll
  for (int i = 0; i < NF; ++i) {
    const T bq = b1 * q[i][1] + b2 * q[i][2] + b3 * q[i][3];
    p[i][0] = x * (gamma * q[i][0] + bq);
    const T abq = a * bq;
    p[i][1] = x * (q[i][1] + b1 * q[i][0] + abq * b1);
    p[i][2] = x * (q[i][2] + b2 * q[i][0] + abq * b2);
    p[i][3] = x * (q[i][3] + b3 * q[i][0] + abq * b3);
  }
  T w = (T)k.w0;
  if (MASSIVE) {
    T m[NF], m2[NF], p02[NF];
    T summ = 0;
#pragma unroll
    for (int i = 0; i < NF; ++i) { m[i] = (T)k.mass[i]; m2[i] = m[i] * m[i]; p02[i] = p[i][0] * p[i][0]; summ += m[i]; }
    const T r = summ / sqrt_s;
    T xi = sqrt_<T>((T)1 - r * r);
    constexpr int kNewton = sizeof(T) == 8 ? 5 : 4;
#pragma unroll 1
    for (int it = 0; it < kNewton; ++it) {
      T f = -sqrt_s, df = 0;
#pragma unroll
      for (int i = 0; i < NF; ++i) {
        const T E = sqrt_<T>(fma_<T>(xi * xi, p02[i], m2[i]));
        f += E;
        df += xi * p02[i] / E;
      }
      xi -= f / df;
    }
    T prod = 1, sum2 = 0;
#pragma unroll
    for (int i = 0; i < NF; ++i) {
      const T kabs = xi * p[i][0];
      const T E = sqrt_<T>(fma_<T>(kabs, kabs, m2[i]));
      p[i][0] = E;
      p[i][1] *= xi; p[i][2] *= xi; p[i][3] *= xi;
      prod *= kabs / E;
      sum2 += kabs * kabs / E;
    }
    T xipow = 1;
#pragma unroll
    for (int i = 0; i < 2 * NF - 3; ++i) xipow *= xi;
    w = w * xipow * prod * sqrt_s / sum2;
  }
  // beams (R5)
  const T hs = (T)0.5 * sqrt_s;
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
__global__ void __launch_bounds__(kThreads) rambo_kernel(Consts k, const T* __restrict__ rnd, int64_t n, int64_t ld,
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
__global__ void __launch_bounds__(kThreads) generate_kernel(Consts k, uint64_t seed, uint64_t first, int64_t n,
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
