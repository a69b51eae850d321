// rambo.cuh — one event of RAMBO (steps A3, A4): massless generation and massive rescaling.
// PAPER.md:78 ("a simple phase space sampling algorithm, RAMBO [39]"), PAPER.md:92 (momenta and a
// sampling weight).  Equations: Kleiss, Stirling, Ellis, CPC 40 (1986) 359; readings R5-R8.
//
// The KSE map is  q_i = q_i0 (1, n_i),  Q = sum q_i,  M = sqrt(Q^2),  p_i = x * Boost_{-Q/M}(q_i),  x = sqrt_s/M.
// Written as in the paper (b = -Q/M, gamma = Q0/M, a = 1/(1+gamma)) it loses a factor gamma^2 of
// precision when the q_i are nearly parallel (M << Q0), and in FP32 Q0^2 - |Q|^2 can even come out
// negative (the NaN events of PAPER.md:182).  The SAME map is evaluated here through Minkowski
// products of the massless q's, which are sums of non-negative terms:
//     h_ij = (1 - n_i.n_j) = |n_i - n_j|^2 / 2,        q_i.q_j = q_i0 q_j0 h_ij,
//     g_i  = (q_i.Q)/q_i0 = sum_{j != i} q_j0 h_ij,     M^2 = sum_i q_i0 g_i,
//     p_i0 = sqrt_s q_i0 g_i / M^2,
//     p_i  = x D q_i0 sum_{j != i} q_j0 [ (M + g_j)(n_i - n_j) + (g_j - g_i) n_j ],   D = 1/(M (M + Q0)),
// (uses sum_i c_i = 1 for c_i = (q_i0 M + q_i.Q) D, the coefficient of -Q in the boosted 3-vector).
// Rounding is then amplified by gamma, the conditioning of the map itself, not by gamma^2.
#pragma once
#include "consts.h"
#include "cx.cuh"

namespace mg {

MG_HD void sincos2pi_(double x, double* s, double* c) {
#ifdef __CUDA_ARCH__
  sincospi(2.0 * x, s, c);
#else
  *s = sin(6.283185307179586476925286766559 * x); *c = cos(6.283185307179586476925286766559 * x);
#endif
}
MG_HD void sincos2pi_(float x, float* s, float* c) {
#ifdef __CUDA_ARCH__
  sincospif(2.0f * x, s, c);
#else
  *s = sinf(6.28318530717958647692f * x); *c = cosf(6.28318530717958647692f * x);
#endif
}
MG_HD double log_(double x) { return log(x); }
MG_HD float log_(float x) { return logf(x); }

// One massless direction and energy from four uniforms (R6): c = 2 rho1 - 1, phi = 2 pi rho2, q0 = -ln(rho3 rho4).
// The only transcendental part of RAMBO; per particle, so that a kernel may spread it over threads (recycle.cuh, M_GEN).
template <class T> MG_HD void rambo_direction(T r1, T r2, T r3, T r4, T& q0, T& nx, T& ny, T& nz) {
  const T c = fma_<T>((T)2, r1, (T)-1);                    // cos(theta) = 2 rho1 - 1
  const T st = (T)2 * sqrt_<T>(r1 * ((T)1 - r1));          // sqrt(1 - c^2), no cancellation (R19)
  T sp, cp;
  sincos2pi_(r2, &sp, &cp);                                 // phi = 2 pi rho2
  // FP32: the rounded product r3*r4 near 1 would lose the small q0; two logs do not (R19)
  q0 = sizeof(T) == 8 ? -log_(r3 * r4) : -(log_(r3) + log_(r4));
  nx = st * cp; ny = st * sp; nz = c;
}

template <class T, int NF, bool MASSIVE>
MG_HD T rambo_finish(const T (&q0)[NF], const T (&nx)[NF], const T (&ny)[NF], const T (&nz)[NF], const Consts& k, T (&p)[NF][4]);

// rho[4*i+k] -> p[i][mu] (final particles only); returns the phase-space weight.
template <class T, int NF, bool MASSIVE>
MG_HD T rambo_core(const T (&rho)[4 * NF], const Consts& k, T (&p)[NF][4]) {
  T q0[NF], nx[NF], ny[NF], nz[NF];
#pragma unroll
  for (int i = 0; i < NF; ++i) rambo_direction<T>(rho[4 * i + 0], rho[4 * i + 1], rho[4 * i + 2], rho[4 * i + 3], q0[i], nx[i], ny[i], nz[i]);
  return rambo_finish<T, NF, MASSIVE>(q0, nx, ny, nz, k, p);
}

// boost and scale to (sqrt_s, 0), massive rescaling, weight: everything after the directions
template <class T, int NF, bool MASSIVE>
MG_HD T rambo_finish(const T (&q0)[NF], const T (&nx)[NF], const T (&ny)[NF], const T (&nz)[NF], const Consts& k, T (&p)[NF][4]) {
  T Q0 = 0;
#pragma unroll
  for (int i = 0; i < NF; ++i) Q0 += q0[i];
  T h[NF][NF];
#pragma unroll
  for (int i = 0; i < NF; ++i)
#pragma unroll
    for (int j = i + 1; j < NF; ++j) {
      const T dx = nx[i] - nx[j], dy = ny[i] - ny[j], dz = nz[i] - nz[j];
      h[i][j] = h[j][i] = (T)0.5 * fma_<T>(dx, dx, fma_<T>(dy, dy, dz * dz));
    }
  T g[NF];
  T M2 = 0;
#pragma unroll
  for (int i = 0; i < NF; ++i) {
    T s = 0;
#pragma unroll
    for (int j = 0; j < NF; ++j) if (j != i) s = fma_<T>(q0[j], h[i][j], s);
    g[i] = s;
    M2 = fma_<T>(q0[i], s, M2);
  }
  const T sqrt_s = (T)k.sqrt_s;
  const T M = sqrt_<T>(M2);
  const T x = sqrt_s / M;
  const T xD = x / (M * (M + Q0));
  const T e0 = sqrt_s / M2;
#pragma unroll
  for (int i = 0; i < NF; ++i) {
    T sx = 0, sy = 0, sz = 0;
#pragma unroll
    for (int j = 0; j < NF; ++j) {
      if (j == i) continue;
      const T a = q0[j] * (M + g[j]), b = q0[j] * (g[j] - g[i]);
      sx = fma_<T>(a, nx[i] - nx[j], fma_<T>(b, nx[j], sx));
      sy = fma_<T>(a, ny[i] - ny[j], fma_<T>(b, ny[j], sy));
      sz = fma_<T>(a, nz[i] - nz[j], fma_<T>(b, nz[j], sz));
    }
    const T f = xD * q0[i];
    p[i][0] = e0 * q0[i] * g[i];
    p[i][1] = f * sx; p[i][2] = f * sy; p[i][3] = f * sz;
  }
  T w = (T)k.w0;
  if (MASSIVE) {
    // Newton on f(xi) = sum_i sqrt(m_i^2 + xi^2 p_i0^2) - sqrt_s from xi0 = sqrt(1 - (sum m / sqrt_s)^2) (R7).  An event
    // stops updating once |f| <= 16 eps sqrt_s (its own residual only: the result is a function of the event, not of
    // the batch); the loop ends when every event of the warp has stopped: 3 updates for the BASELINE masses, at most 8.
    // Inside the iteration E_i and 1/E_i come from one reciprocal square root (the iteration corrects its own
    // rounding); the energies that are stored are recomputed below with a correctly rounded square root.
    T m2[NF], p02[NF];
    T summ = 0;
#pragma unroll
    for (int i = 0; i < NF; ++i) { const T m = (T)k.mass[i]; m2[i] = m * m; p02[i] = p[i][0] * p[i][0]; summ += m; }
    const T r = summ / sqrt_s;
    T xi = sqrt_<T>((T)1 - r * r);
    const T tol = (sizeof(T) == 8 ? (T)3.6e-15 : (T)1.9e-6) * sqrt_s;
#pragma unroll 1
    for (int it = 0; it < 8; ++it) {
      T f = -sqrt_s, df = 0;
#pragma unroll
      for (int i = 0; i < NF; ++i) {
        const T arg = fma_<T>(xi * xi, p02[i], m2[i]);
        const T inv = rsqrt_<T>(arg);
        f = fma_<T>(arg, inv, f);
        df = fma_<T>(xi * p02[i], inv, df);
      }
      const bool done = abs_<T>(f) <= tol;
      if (!done) xi -= f / df;
#ifdef __CUDA_ARCH__
      if (__all_sync(__activemask(), done)) break;
#else
      if (done) break;
#endif
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
  return w;
}


#ifdef __CUDACC__
// rambo_finish spread over the final particles of an event: FOUR consecutive lanes of a warp hold one event, lane i < NF
// owns particle i (its direction and energy from rambo_direction; lanes i >= NF carry a copy of particle 0 and only take
// part in the exchanges).  Everything that depends on one particle — its reciprocal square root in every Newton step, its
// boosted momentum, its final square root and divisions — is evaluated by its lane only; the sums over particles are
// gathered with shuffles and added IN THE ORDER OF rambo_finish, so the momenta and the weight are the same bits as
// mg_generate's.  Used by the shared-memory kernels in M_GEN mode (recycle.cuh), where the CTA waits for this chain:
// a third of the instructions of the one-thread form on the critical path.  All 32 lanes of the warp must call it.
// p: the lane's particle (E, px, py, pz); returns the phase-space weight (the same in the four lanes of an event).
template <class T, int NF>
__device__ __forceinline__ T rambo_finish_lanes(int i, T q0m, T nxm, T nym, T nzm, const Consts& k, T (&p)[4]) {
  static_assert(NF <= 4, "four lanes per event");
  const unsigned full = 0xffffffffu;
  T q0[NF], nx[NF], ny[NF], nz[NF];
#pragma unroll
  for (int j = 0; j < NF; ++j) {
    q0[j] = __shfl_sync(full, q0m, j, 4); nx[j] = __shfl_sync(full, nxm, j, 4);
    ny[j] = __shfl_sync(full, nym, j, 4); nz[j] = __shfl_sync(full, nzm, j, 4);
  }
  T Q0 = 0;
#pragma unroll
  for (int j = 0; j < NF; ++j) Q0 += q0[j];
  // h_ij of the lane's particle with every other one ((-a)^2 = a^2: the value rambo_finish uses for either order of i, j)
  T hm[NF];
#pragma unroll
  for (int j = 0; j < NF; ++j) {
    const T dx = nxm - nx[j], dy = nym - ny[j], dz = nzm - nz[j];
    hm[j] = (T)0.5 * fma_<T>(dx, dx, fma_<T>(dy, dy, dz * dz));
  }
  T gm = 0;
#pragma unroll
  for (int j = 0; j < NF; ++j) gm = (j != i) ? fma_<T>(q0[j], hm[j], gm) : gm;
  T g[NF];
  T M2 = 0;
#pragma unroll
  for (int j = 0; j < NF; ++j) { g[j] = __shfl_sync(full, gm, j, 4); M2 = fma_<T>(q0[j], g[j], M2); }
  const T sqrt_s = (T)k.sqrt_s;
  const T M = sqrt_<T>(M2);
  const T x = sqrt_s / M;
  const T xD = x / (M * (M + Q0));
  const T e0 = sqrt_s / M2;
  T sx = 0, sy = 0, sz = 0;
#pragma unroll
  for (int j = 0; j < NF; ++j) {
    const T a = q0[j] * (M + g[j]), b = q0[j] * (g[j] - gm);
    const T tx = fma_<T>(a, nxm - nx[j], fma_<T>(b, nx[j], sx));
    const T ty = fma_<T>(a, nym - ny[j], fma_<T>(b, ny[j], sy));
    const T tz = fma_<T>(a, nzm - nz[j], fma_<T>(b, nz[j], sz));
    if (j != i) { sx = tx; sy = ty; sz = tz; }
  }
  const T f0 = xD * q0m;
  p[0] = e0 * q0m * gm;
  p[1] = f0 * sx; p[2] = f0 * sy; p[3] = f0 * sz;
  // massive rescaling: Newton as in rambo_finish; the lane contributes sqrt(m^2 + xi^2 p0^2) of its particle
  T summ = 0;
#pragma unroll
  for (int j = 0; j < NF; ++j) summ += (T)k.mass[j];
  T mm = 0;
#pragma unroll
  for (int j = 0; j < NF; ++j) mm = (j == i) ? (T)k.mass[j] : mm;
  const T m2m = mm * mm, p02m = p[0] * p[0];
  const T r = summ / sqrt_s;
  T xi = sqrt_<T>((T)1 - r * r);
  const T tol = (sizeof(T) == 8 ? (T)3.6e-15 : (T)1.9e-6) * sqrt_s;
#pragma unroll 1
  for (int it = 0; it < 8; ++it) {
    const T argm = fma_<T>(xi * xi, p02m, m2m);
    const T invm = rsqrt_<T>(argm);
    const T dm = xi * p02m;
    T f = -sqrt_s, df = 0;
#pragma unroll
    for (int j = 0; j < NF; ++j) {
      const T arg = __shfl_sync(full, argm, j, 4), inv = __shfl_sync(full, invm, j, 4), d = __shfl_sync(full, dm, j, 4);
      f = fma_<T>(arg, inv, f);
      df = fma_<T>(d, inv, df);
    }
    const bool done = abs_<T>(f) <= tol;
    if (!done) xi -= f / df;
    if (__all_sync(full, done)) break;
  }
  const T kabsm = xi * p[0];
  const T Em = sqrt_<T>(fma_<T>(kabsm, kabsm, m2m));
  p[0] = Em;
  p[1] *= xi; p[2] *= xi; p[3] *= xi;
  const T ratm = kabsm / Em, s2m = kabsm * kabsm / Em;
  T prod = 1, sum2 = 0;
#pragma unroll
  for (int j = 0; j < NF; ++j) { prod *= __shfl_sync(full, ratm, j, 4); sum2 += __shfl_sync(full, s2m, j, 4); }
  T xipow = 1;
#pragma unroll
  for (int j = 0; j < 2 * NF - 3; ++j) xipow *= xi;
  return (T)k.w0 * xipow * prod * sqrt_s / sum2;
}
#endif

}  // namespace mg
