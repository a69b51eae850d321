// me_common.cuh — pieces shared by the per-process sigmaKin kernels: momentum loads (A5), the
// helicity loop driver (A11), the optional event weight (A13) and the launch wrapper.
#pragma once
#include "mg_internal.h"
#include "helas.cuh"

namespace mg {

// A5: particle i of event e from the SoA array (row stride ld); one coalesced row access per component.
template <class T> __device__ __forceinline__ Mom<T> load_mom(const T* __restrict__ mom, int64_t ld, int64_t e, int i) {
  Mom<T> p;
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) p.v[mu] = __ldg(mom + (int64_t)(4 * i + mu) * ld + e);
  return p;
}

constexpr int kMeThreads = 128;

// Helicity-flip symmetry (R35).  For the QCD processes (parity-conserving couplings, tree level, real momenta)
// the amplitude with every helicity flipped is, up to a sign, the complex conjugate of the original one, so the
// colour-summed |M|^2 of helicity combination h equals that of its complement NHEL-1-h at the SAME momenta.  Proc::FLIP
// processes evaluate one member of each pair (the one with the last particle at helicity -1) and count it once per
// member that the good-helicity mask keeps.  Not for e+ e- -> mu+ mu- (the Z couplings are chiral).
template <class Proc> MG_HD uint64_t flip_half(uint64_t mask) {
  if (!Proc::FLIP) return mask;
  uint64_t rev = 0;
  for (int h = 0; h < Proc::NHEL / 2; ++h) rev |= ((mask >> (Proc::NHEL - 1 - h)) & 1ull) << h;
  return (mask | rev) & ((1ull << (Proc::NHEL / 2)) - 1ull);
}
template <class Proc> MG_HD int flip_weight(uint64_t mask, int h) {
  return (int)((mask >> h) & 1ull) + (int)((mask >> (Proc::NHEL - 1 - h)) & 1ull);
}

// Generic one-thread-per-event kernel.  Proc supplies
//   struct Event<T> { Mom<T> p[NPAR]; ... }   per-event data that does not depend on the helicity
//   static void   finish(Event&, consts)      fills the rest of Event from p[]
//   static T      helicity(const Event&, int ihel, consts)     |M|^2 of one helicity combination (no norm)
//   static int    NHEL, NPAR
// mask: good helicities (bit h).  me = norm * sum_h.  PER_HEL: write every helicity, ignore mask.
template <class Proc, class T, bool PER_HEL>
__global__ void __launch_bounds__(kMeThreads, Proc::MINB) sigmakin_kernel(Consts k, const T* __restrict__ mom, int64_t n, int64_t ld,
                                                              T* __restrict__ me, const T* __restrict__ psw,
                                                              T* __restrict__ evw, T* __restrict__ hel_out, uint64_t mask) {
  const int64_t e = (int64_t)blockIdx.x * kMeThreads + threadIdx.x;
  if (e >= n) return;
  typename Proc::template Event<T> ev;
#pragma unroll
  for (int i = 0; i < Proc::NPAR; ++i) ev.p[i] = load_mom<T>(mom, ld, e, i);
  Proc::template finish<T>(ev, k);
  if (PER_HEL) {
#pragma unroll 1
    for (int h = 0; h < (Proc::FLIP ? Proc::NHEL / 2 : Proc::NHEL); ++h) {
      const T v = Proc::template helicity<T>(ev, h, k);
      hel_out[(int64_t)h * ld + e] = v;
      if (Proc::FLIP) hel_out[(int64_t)(Proc::NHEL - 1 - h) * ld + e] = v;
    }
    return;
  }
  T sum = 0;
#pragma unroll 1
  for (uint64_t m = flip_half<Proc>(mask); m; m &= m - 1) {
    const int h = __ffsll((long long)m) - 1;
    const T v = Proc::template helicity<T>(ev, h, k);
    sum += Proc::FLIP ? (T)flip_weight<Proc>(mask, h) * v : v;
  }
  const T r = sum * (T)k.me_norm;
  me[e] = r;
  if (evw != nullptr) evw[e] = psw[e] * r;
}

template <class Proc>
cudaError_t launch_sigmakin(const mg_process* p, const MeArgs& a, cudaStream_t s) {
  const unsigned g = (unsigned)((a.n + kMeThreads - 1) / kMeThreads);
  const bool f64 = p->par.precision == MG_FP64;
  if (a.hel_out) {
    if (f64) sigmakin_kernel<Proc, double, true><<<g, kMeThreads, 0, s>>>(p->k, (const double*)a.mom, a.n, a.ld, nullptr, nullptr, nullptr, (double*)a.hel_out, 0);
    else sigmakin_kernel<Proc, float, true><<<g, kMeThreads, 0, s>>>(p->k, (const float*)a.mom, a.n, a.ld, nullptr, nullptr, nullptr, (float*)a.hel_out, 0);
  } else {
    if (f64) sigmakin_kernel<Proc, double, false><<<g, kMeThreads, 0, s>>>(p->k, (const double*)a.mom, a.n, a.ld, (double*)a.me, (const double*)a.psw, (double*)a.evw, nullptr, a.mask);
    else sigmakin_kernel<Proc, float, false><<<g, kMeThreads, 0, s>>>(p->k, (const float*)a.mom, a.n, a.ld, (float*)a.me, (const float*)a.psw, (float*)a.evw, nullptr, a.mask);
  }
  return cudaGetLastError();
}

}  // namespace mg
