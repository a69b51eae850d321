// fused.cuh — A1-A13 in ONE kernel for the one-thread-per-event processes: Philox words ->
// uniforms -> RAMBO momenta -> sigmaKin -> event weight, all in registers; nothing but the results (8-24 bytes per
// event) touches HBM.  PAPER.md:112-118 measures the copy:compute balance of the three separate components (1:1 for
// e+ e- -> mu+ mu-): for that process the momenta round trip through memory is the larger part of the step.
// Same device functions as the separate kernels (philox.cuh, rambo.cuh, the Proc structs), so the results agree
// with mg_generate + mg_sigmakin to rounding.
#pragma once
#include "me_common.cuh"
#include "philox.cuh"
#include "rambo.cuh"

namespace mg {

template <class Proc, class T, int NF, bool MASSIVE>
__global__ void __launch_bounds__(kMeThreads, Proc::MINB) fused_kernel(Consts k, uint64_t seed, uint64_t first, int64_t n,
                                                           T* __restrict__ me, T* __restrict__ psw, T* __restrict__ evw,
                                                           uint64_t mask) {
  static_assert(Proc::NPAR == NF + 2, "two beams + NF final particles");
  const int64_t e = (int64_t)blockIdx.x * kMeThreads + threadIdx.x;
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
  T pf[NF][4];
  const T w = rambo_core<T, NF, MASSIVE>(rho, k, pf);
  typename Proc::template Event<T> ev;
  const T hs = (T)0.5 * (T)k.sqrt_s;                      // beams (R5), as rambo_event writes them
  ev.p[0] = Mom<T>{{hs, (T)0, (T)0, hs}};
  ev.p[1] = Mom<T>{{hs, (T)0, (T)0, -hs}};
#pragma unroll
  for (int i = 0; i < NF; ++i) ev.p[2 + i] = Mom<T>{{pf[i][0], pf[i][1], pf[i][2], pf[i][3]}};
  Proc::template finish<T>(ev, k);
  T sum = 0;
#pragma unroll 1
  for (uint64_t m = flip_half<Proc>(mask); m; m &= m - 1) {
    const int h = __ffsll((long long)m) - 1;
    const T v = Proc::template helicity<T>(ev, h, k);
    sum += Proc::FLIP ? (T)flip_weight<Proc>(mask, h) * v : v;
  }
  const T r = sum * (T)k.me_norm;
  __stcs(me + e, r);
  if (psw != nullptr) __stcs(psw + e, w);
  if (evw != nullptr) __stcs(evw + e, w * r);
}

template <class Proc, int NF, bool MASSIVE>
cudaError_t launch_fused(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw,
                         cudaStream_t s) {
  const unsigned g = (unsigned)((n + kMeThreads - 1) / kMeThreads);
  if (p->par.precision == MG_FP64)
    fused_kernel<Proc, double, NF, MASSIVE><<<g, kMeThreads, 0, s>>>(p->k, seed, first, n, (double*)me, (double*)psw, (double*)evw, p->hel_mask);
  else
    fused_kernel<Proc, float, NF, MASSIVE><<<g, kMeThreads, 0, s>>>(p->k, seed, first, n, (float*)me, (float*)psw, (float*)evw, p->hel_mask);
  return cudaGetLastError();
}

}  // namespace mg
