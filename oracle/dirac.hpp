// ORACLE — test infrastructure only (see philox.hpp header).
//
// Explicit Dirac algebra for the textbook Feynman rules: 4x4 gamma matrices in the DIRAC
// (standard) representation, helicity spinors u, v, polarisation vectors.  Nothing here is in the
// paper (it only names the routines IXXXXX/OXXXXX/FFV..., Fig. 1 caption, PAPER.md:37
// §2); the definitions are the Peskin-Schroeder ones collected in SURVEY.md Appendix A and
// restated in DESIGN.md ("Conventions").  The CUDA path uses a different (chiral, 2x2 block)
// formulation; per-helicity |M|^2 does not depend on that choice (reading R22).
#pragma once
#include <cmath>
#include <complex>

namespace oracle {

template <class T> using cx = std::complex<T>;

template <class T> struct Vec4 {  // contravariant components V^mu, mu = (0,1,2,3), complex
  cx<T> v[4];
};
template <class T> struct Col4 { cx<T> c[4]; };  // column spinor
template <class T> struct Row4 { cx<T> r[4]; };  // row spinor (psi-bar)
template <class T> struct Mat4 { cx<T> m[4][4]; };

// Minkowski product a.b = a0 b0 - a1 b1 - a2 b2 - a3 b3 (no complex conjugation).
template <class T> cx<T> mdot(const Vec4<T>& a, const Vec4<T>& b) {
  return a.v[0] * b.v[0] - a.v[1] * b.v[1] - a.v[2] * b.v[2] - a.v[3] * b.v[3];
}
template <class T> Vec4<T> real_vec(const T* p, T sign = 1) {
  Vec4<T> r;
  for (int i = 0; i < 4; ++i) r.v[i] = cx<T>(sign * p[i], 0);
  return r;
}
template <class T> Vec4<T> vadd(const Vec4<T>& a, const Vec4<T>& b) {
  Vec4<T> r; for (int i = 0; i < 4; ++i) r.v[i] = a.v[i] + b.v[i]; return r;
}
template <class T> Vec4<T> vsub(const Vec4<T>& a, const Vec4<T>& b) {
  Vec4<T> r; for (int i = 0; i < 4; ++i) r.v[i] = a.v[i] - b.v[i]; return r;
}
template <class T> Vec4<T> vscale(const Vec4<T>& a, cx<T> s) {
  Vec4<T> r; for (int i = 0; i < 4; ++i) r.v[i] = a.v[i] * s; return r;
}
template <class T> Vec4<T> vconj(const Vec4<T>& a) {
  Vec4<T> r; for (int i = 0; i < 4; ++i) r.v[i] = std::conj(a.v[i]); return r;
}

// gamma^mu, Dirac representation:  gamma^0 = diag(1,1,-1,-1),  gamma^i = [[0, s_i],[-s_i, 0]].
template <class T> Mat4<T> gamma_mu(int mu) {
  Mat4<T> g{};
  const cx<T> I(0, 1);
  if (mu == 0) { g.m[0][0] = 1; g.m[1][1] = 1; g.m[2][2] = -1; g.m[3][3] = -1; return g; }
  cx<T> s[2][2];
  if (mu == 1) { s[0][0] = 0; s[0][1] = 1; s[1][0] = 1; s[1][1] = 0; }
  if (mu == 2) { s[0][0] = 0; s[0][1] = -I; s[1][0] = I; s[1][1] = 0; }
  if (mu == 3) { s[0][0] = 1; s[0][1] = 0; s[1][0] = 0; s[1][1] = -1; }
  for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b) { g.m[a][2 + b] = s[a][b]; g.m[2 + a][b] = -s[a][b]; }
  return g;
}
// gamma^5 = i g0 g1 g2 g3 = [[0,1],[1,0]] in this representation.
template <class T> Mat4<T> gamma_5() {
  Mat4<T> g{};
  g.m[0][2] = 1; g.m[1][3] = 1; g.m[2][0] = 1; g.m[3][1] = 1;
  return g;
}
template <class T> Mat4<T> identity4() {
  Mat4<T> g{}; for (int i = 0; i < 4; ++i) g.m[i][i] = 1; return g;
}
template <class T> Mat4<T> madd(const Mat4<T>& a, const Mat4<T>& b) {
  Mat4<T> r; for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) r.m[i][j] = a.m[i][j] + b.m[i][j]; return r;
}
template <class T> Mat4<T> mscale(const Mat4<T>& a, cx<T> s) {
  Mat4<T> r; for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) r.m[i][j] = a.m[i][j] * s; return r;
}
template <class T> Mat4<T> mmul(const Mat4<T>& a, const Mat4<T>& b) {
  Mat4<T> r{};
  for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) for (int k = 0; k < 4; ++k) r.m[i][j] += a.m[i][k] * b.m[k][j];
  return r;
}
template <class T> Col4<T> mul(const Mat4<T>& a, const Col4<T>& x) {
  Col4<T> r{}; for (int i = 0; i < 4; ++i) for (int k = 0; k < 4; ++k) r.c[i] += a.m[i][k] * x.c[k]; return r;
}
template <class T> Row4<T> mul(const Row4<T>& x, const Mat4<T>& a) {
  Row4<T> r{}; for (int j = 0; j < 4; ++j) for (int k = 0; k < 4; ++k) r.r[j] += x.r[k] * a.m[k][j]; return r;
}
template <class T> cx<T> mul(const Row4<T>& x, const Col4<T>& y) {
  cx<T> r = 0; for (int k = 0; k < 4; ++k) r += x.r[k] * y.c[k]; return r;
}
// V-slash = gamma^mu V_mu = g0 V^0 - g1 V^1 - g2 V^2 - g3 V^3.
template <class T> Mat4<T> slash(const Vec4<T>& V) {
  Mat4<T> r{};
  for (int mu = 0; mu < 4; ++mu) {
    Mat4<T> g = gamma_mu<T>(mu);
    cx<T> s = (mu == 0) ? V.v[0] : -V.v[mu];
    r = madd(r, mscale(g, s));
  }
  return r;
}
// psi-bar = psi^dagger gamma^0.
template <class T> Row4<T> bar(const Col4<T>& x) {
  Row4<T> r;
  r.r[0] = std::conj(x.c[0]); r.r[1] = std::conj(x.c[1]);
  r.r[2] = -std::conj(x.c[2]); r.r[3] = -std::conj(x.c[3]);
  return r;
}

// Helicity 2-spinors chi_lambda for 3-momentum (px,py,pz), P = |p|:
//   chi_+ = (P+pz, px+i py)/sqrt(2P(P+pz)),  chi_- = (-px+i py, P+pz)/sqrt(2P(P+pz));
//   pz = -P (pT = 0): chi_+ = (0,1), chi_- = (-1,0).
// P+pz is evaluated as pT^2/(P-pz) when pz<0 (no cancellation).
template <class T> void chi(const T* p, int lambda, cx<T> out[2]) {
  T px = p[1], py = p[2], pz = p[3];
  T pt2 = px * px + py * py;
  T P = std::sqrt(pt2 + pz * pz);
  if (pt2 == 0 && pz < 0) {
    if (lambda > 0) { out[0] = 0; out[1] = 1; } else { out[0] = -1; out[1] = 0; }
    return;
  }
  T Ppz = (pz >= 0) ? (P + pz) : pt2 / (P - pz);
  T nrm = 1 / std::sqrt(2 * P * Ppz);
  if (lambda > 0) { out[0] = cx<T>(Ppz * nrm, 0); out[1] = cx<T>(px * nrm, py * nrm); }
  else { out[0] = cx<T>(-px * nrm, py * nrm); out[1] = cx<T>(Ppz * nrm, 0); }
}

// u(p,lambda) = ( sqrt(E+m) chi, lambda P/sqrt(E+m) chi )   [ = lambda sqrt(E-m) chi ]
template <class T> Col4<T> spinor_u(const T* p, T m, int lambda) {
  cx<T> x[2]; chi<T>(p, lambda, x);
  T P = std::sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  T up = std::sqrt(p[0] + m);
  T lo = (T)lambda * P / up;
  Col4<T> u;
  u.c[0] = up * x[0]; u.c[1] = up * x[1]; u.c[2] = lo * x[0]; u.c[3] = lo * x[1];
  return u;
}
// v(p,lambda) = i gamma^2 u(p,lambda)^*   (antiparticle of helicity lambda)
template <class T> Col4<T> spinor_v(const T* p, T m, int lambda) {
  Col4<T> u = spinor_u<T>(p, m, lambda);
  Col4<T> v;
  v.c[0] = std::conj(u.c[3]);
  v.c[1] = -std::conj(u.c[2]);
  v.c[2] = -std::conj(u.c[1]);
  v.c[3] = std::conj(u.c[0]);
  return v;
}

// Polarisation vector of helicity lambda = +-1 for a massless vector of momentum p:
//   eps = (0; -l cos(th) cos(ph) + i sin(ph), -l cos(th) sin(ph) - i cos(ph), l sin(th))/sqrt(2);
//   pT = 0: (0; -l sgn(pz), -i, 0)/sqrt(2).
template <class T> Vec4<T> polvec(const T* p, int lambda) {
  T px = p[1], py = p[2], pz = p[3];
  T pt = std::sqrt(px * px + py * py);
  T P = std::sqrt(px * px + py * py + pz * pz);
  T l = (T)lambda;
  T r2 = 1 / std::sqrt((T)2);
  Vec4<T> e;
  e.v[0] = 0;
  if (pt == 0) {
    T sg = (pz >= 0) ? (T)1 : (T)-1;
    e.v[1] = cx<T>(-l * sg * r2, 0); e.v[2] = cx<T>(0, -r2); e.v[3] = 0;
    return e;
  }
  T ct = pz / P, st = pt / P, cp = px / pt, sp = py / pt;
  e.v[1] = cx<T>(-l * ct * cp * r2, sp * r2);
  e.v[2] = cx<T>(-l * ct * sp * r2, -cp * r2);
  e.v[3] = cx<T>(l * st * r2, 0);
  return e;
}

}  // namespace oracle
