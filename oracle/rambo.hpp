// ORACLE — test infrastructure only (see philox.hpp header).
//
// RAMBO flat phase-space sampler: massless generation, then the massive rescaling.
//
// Serves PAPER.md:78 (§3: "a simple phase space sampling algorithm, RAMBO [39]") and PAPER.md:92
// (§4: momenta "as well as a sampling weight").  The paper gives no equations; the steps below
// follow Kleiss, Stirling, Ellis, Comput. Phys. Commun. 40 (1986) 359, in its notation
// (readings R5-R8 in DESIGN.md).
#pragma once
#include <cmath>
#include <vector>
#include "common.hpp"

namespace oracle {

// Closed-form massless RAMBO weight (north_star):
//   W0 = (pi/2)^(n-1) s^(n-2) / ((n-1)!(n-2)!) * (2 pi)^(4-3n)
template <class T>
T rambo_w0(int n, T sqrt_s) {
  T s = sqrt_s * sqrt_s;
  T w = 1;
  for (int i = 0; i < n - 1; ++i) w *= pi_v<T>() / 2;
  for (int i = 0; i < n - 2; ++i) w *= s;
  for (int i = 2; i <= n - 1; ++i) w /= (T)i;  // (n-1)!
  for (int i = 2; i <= n - 2; ++i) w /= (T)i;  // (n-2)!
  int e = 4 - 3 * n;                          // (2 pi)^(4-3n), e <= -2
  for (int i = 0; i < -e; ++i) w /= 2 * pi_v<T>();
  return w;
}

// KSE massless step.  rho[4*i+0..3] = (rho1..rho4) of final particle i; p[i][mu], mu = (E,x,y,z).
//   c = 2 rho1 - 1, phi = 2 pi rho2, q0 = -ln(rho3 rho4), q = q0 (1, sqrt(1-c^2) cos phi, sqrt(1-c^2) sin phi, c)
//   Q = sum q, M = sqrt(Q^2), b = -Qvec/M, x = sqrt_s/M, gamma = Q0/M, a = 1/(1+gamma)
//   p0 = x (gamma q0 + b.q),  pvec = x (qvec + b q0 + a (b.q) b)
template <class T>
void rambo_massless(int n, const T* rho, T sqrt_s, T (*p)[4]) {
  std::vector<T> q(4 * n);
  T Q[4] = {0, 0, 0, 0};
  for (int i = 0; i < n; ++i) {
    T c = 2 * rho[4 * i + 0] - 1;
    T phi = 2 * pi_v<T>() * rho[4 * i + 1];
    T q0 = -std::log(rho[4 * i + 2] * rho[4 * i + 3]);
    T st = std::sqrt(1 - c * c);
    q[4 * i + 0] = q0;
    q[4 * i + 1] = q0 * st * std::cos(phi);
    q[4 * i + 2] = q0 * st * std::sin(phi);
    q[4 * i + 3] = q0 * c;
    for (int mu = 0; mu < 4; ++mu) Q[mu] += q[4 * i + mu];
  }
  T M = std::sqrt(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
  T b[3] = {-Q[1] / M, -Q[2] / M, -Q[3] / M};
  T x = sqrt_s / M;
  T gamma = Q[0] / M;
  T a = 1 / (1 + gamma);
  for (int i = 0; i < n; ++i) {
    const T* qi = &q[4 * i];
    T bq = b[0] * qi[1] + b[1] * qi[2] + b[2] * qi[3];
    p[i][0] = x * (gamma * qi[0] + bq);
    for (int k = 0; k < 3; ++k) p[i][1 + k] = x * (qi[1 + k] + b[k] * qi[0] + a * bq * b[k]);
  }
}

// KSE massive step (reading R7).  Input: massless p[i]; output k[i] with k_i^2 = m_i^2, weight.
//   solve f(xi) = sum_i sqrt(m_i^2 + xi^2 p_i0^2) - sqrt_s = 0 by Newton from
//   xi0 = sqrt(1 - (sum m_i / sqrt_s)^2),  f' = sum xi p_i0^2 / E_i,  until |f| <= tol * sqrt_s
//   kvec_i = xi pvec_i, E_i = sqrt(m_i^2 + xi^2 p_i0^2)
//   W = W0 * xi^(2n-3) * prod_i(|k_i|/E_i) * sqrt_s / sum_i(|k_i|^2/E_i),  |k_i| = xi p_i0
// Returns xi through *xi_out when non-null.
template <class T>
T rambo_massive(int n, const T* m, T sqrt_s, T (*p)[4], T tol, T* xi_out = nullptr) {
  T summ = 0;
  bool any = false;
  for (int i = 0; i < n; ++i) { summ += m[i]; any = any || (m[i] != 0); }
  T w0 = rambo_w0<T>(n, sqrt_s);
  if (!any) { if (xi_out) *xi_out = 1; return w0; }
  T xi = std::sqrt(1 - (summ / sqrt_s) * (summ / sqrt_s));
  for (int it = 0; it < 100; ++it) {
    T f = -sqrt_s, df = 0;
    for (int i = 0; i < n; ++i) {
      T E = std::sqrt(m[i] * m[i] + xi * xi * p[i][0] * p[i][0]);
      f += E;
      df += xi * p[i][0] * p[i][0] / E;
    }
    if (std::fabs(f) <= tol * sqrt_s) break;
    xi -= f / df;
  }
  T prod = 1, sum2 = 0;
  for (int i = 0; i < n; ++i) {
    T kabs = xi * p[i][0];
    T E = std::sqrt(m[i] * m[i] + kabs * kabs);
    p[i][0] = E;
    for (int k = 1; k < 4; ++k) p[i][k] *= xi;
    prod *= kabs / E;
    sum2 += kabs * kabs / E;
  }
  T xipow = 1;
  for (int i = 0; i < 2 * n - 3; ++i) xipow *= xi;
  if (xi_out) *xi_out = xi;
  return w0 * xipow * prod * sqrt_s / sum2;
}

// One whole event: beams (reading R5: p1 = (sqrt_s/2,0,0,+sqrt_s/2), p2 = (sqrt_s/2,0,0,-sqrt_s/2))
// followed by the n final momenta.  mom[(2+n)][4].  Returns the phase-space weight.
template <class T>
T rambo_event(int n, const T* rho, const T* masses, T sqrt_s, T (*mom)[4], T tol, T* xi_out = nullptr) {
  mom[0][0] = sqrt_s / 2; mom[0][1] = 0; mom[0][2] = 0; mom[0][3] = sqrt_s / 2;
  mom[1][0] = sqrt_s / 2; mom[1][1] = 0; mom[1][2] = 0; mom[1][3] = -sqrt_s / 2;
  rambo_massless<T>(n, rho, sqrt_s, mom + 2);
  return rambo_massive<T>(n, masses, sqrt_s, mom + 2, tol, xi_out);
}

}  // namespace oracle
