// helas.cuh — helicity wavefunctions and vertex routines of the sm_100a path (steps A6-A8 of
// SURVEY.md §8(a); Fig. 1 and PAPER.md:37 §2 name the routine families IXXXXX/OXXXXX,
// FFV*_0 (amplitude), FFV*_1/_2/_3 (off-shell wavefunction incl. propagator) without printing a
// formula).  Everything here is derived from the textbook Feynman rules of DESIGN.md
// "Conventions" in the CHIRAL (Weyl) representation,
//     gamma^mu = [[0, sigma^mu],[sigmabar^mu, 0]],  sigma^mu = (1, sigma),  sigmabar^mu = (1, -sigma),
// so that a fermion wavefunction is two 2-component blocks ("two for the
// chirality-left spinor, two for the chirality-right spinor"), V-slash is two 2x2 products and the
// vanishing chirality of a massless fermion is an exact zero.
//
// REDUCED rules: all couplings and all factors of i are stripped from vertices and propagators:
//     q qbar g vertex -> gamma^mu,  quark propagator -> (qslash+m)/(q^2-m^2),  gluon propagator -> 1/k^2,
//     ggg vertex -> V3^{mu nu rho},  gggg vertex -> the three metric-tensor structures.
// DESIGN.md "Phase bookkeeping" shows that for gg -> t t~ + gluons every diagram then carries the
// SAME global factor (-i)(-1)^{n_g} g_s^{n_g}, so the colour-flow coefficients are +-1 and g_s^{2 n_g}
// is applied once per event.
//
// A 4-momentum that enters a routine is REAL (a signed sum of external momenta); wavefunctions do
// not carry their momentum (HELAS stores it in two extra complex slots; here it is recomputed).
//
// Everything is __host__ __device__ so that a developer probe can run the same code on the host.
#pragma once
#include "cx.cuh"
#include "consts.h"

namespace mg {

template <class T> struct Vec4 { cx<T> v[4]; };          // V^mu, mu = 0..3 (contravariant)
template <class T> struct Spinor { cx<T> l[2], r[2]; };  // column: (psi_L, psi_R); row: (a | b) = (first two | last two)
template <class T> struct Mom { T v[4]; };               // real 4-momentum (E, px, py, pz)

template <class T> MG_HD Mom<T> operator+(Mom<T> a, Mom<T> b) { return Mom<T>{{a.v[0] + b.v[0], a.v[1] + b.v[1], a.v[2] + b.v[2], a.v[3] + b.v[3]}}; }
template <class T> MG_HD Mom<T> operator-(Mom<T> a, Mom<T> b) { return Mom<T>{{a.v[0] - b.v[0], a.v[1] - b.v[1], a.v[2] - b.v[2], a.v[3] - b.v[3]}}; }
template <class T> MG_HD Mom<T> operator-(Mom<T> a) { return Mom<T>{{-a.v[0], -a.v[1], -a.v[2], -a.v[3]}}; }
template <class T> MG_HD T mdot(Mom<T> a, Mom<T> b) {
  return fma_<T>(a.v[0], b.v[0], fma_<T>(-a.v[1], b.v[1], fma_<T>(-a.v[2], b.v[2], -a.v[3] * b.v[3])));
}
// Minkowski products (no conjugation)
template <class T> MG_HD cx<T> mdot(const Vec4<T>& a, const Vec4<T>& b) {
  cx<T> r = a.v[0] * b.v[0];
  r = cfms(a.v[1], b.v[1], r);
  r = cfms(a.v[2], b.v[2], r);
  r = cfms(a.v[3], b.v[3], r);
  return r;
}
template <class T> MG_HD cx<T> mdot(const Vec4<T>& a, Mom<T> k) {
  cx<T> r = k.v[0] * a.v[0];
  r = rfma(-k.v[1], a.v[1], r);
  r = rfma(-k.v[2], a.v[2], r);
  r = rfma(-k.v[3], a.v[3], r);
  return r;
}

// ---------------------------------------------------------------------------------------------
// External wavefunctions (A6).  Helicity 2-spinors chi_lambda of the 3-momentum (|p| = P):
//   chi_+ = (P+pz, px+i py)/sqrt(2P(P+pz)),  chi_- = (-px+i py, P+pz)/sqrt(2P(P+pz));
//   pz = -P: chi_+ = (0,1), chi_- = (-1,0).     P+pz is evaluated as pT^2/(P-pz) for pz < 0 (R19).
// ---------------------------------------------------------------------------------------------
template <class T> struct Chi { cx<T> c[2]; };

template <class T> MG_HD Chi<T> chi(Mom<T> p, T P, int lambda) {
  const T px = p.v[1], py = p.v[2], pz = p.v[3];
  const T pt2 = fma_<T>(px, px, py * py);
  Chi<T> x;
  if (pt2 == (T)0) {  // along the z axis
    const bool up = (pz >= (T)0) == (lambda > 0);
    // pz>=0: chi_+ = (1,0), chi_- = (0,1);  pz<0: chi_+ = (0,1), chi_- = (-1,0)
    x.c[0] = cx<T>(up ? (pz >= (T)0 ? (T)1 : (T)-1) : (T)0, (T)0);
    x.c[1] = cx<T>(up ? (T)0 : (T)1, (T)0);
    return x;
  }
  const T Ppz = (pz >= (T)0) ? (P + pz) : pt2 / (P - pz);
  const T nrm = rsqrt_<T>((T)2 * P * Ppz);
  if (lambda > 0) { x.c[0] = cx<T>(Ppz * nrm, (T)0); x.c[1] = cx<T>(px * nrm, py * nrm); }
  else            { x.c[0] = cx<T>(-px * nrm, py * nrm); x.c[1] = cx<T>(Ppz * nrm, (T)0); }
  return x;
}

// omega_+ = sqrt(E+P), omega_- = sqrt(E-P).  For m = 0 the energy is taken as |p| (not the stored E): omega_- is
// exactly 0 and the spinor solves the Dirac equation of the 3-momentum exactly even when the event generator left E
// and |p| a few ulps apart.  For m > 0 the pair is evaluated as
//     omega_+- = ((E+m) +- P) / sqrt(2 (E+m)),
// which equals sqrt(E +- P) on the mass shell and has no cancellation (E + m - P >= m).  Off the mass shell by
// rounding (momenta stored in FP32: E^2 - P^2 - m^2 ~ 1e-7 E^2) sqrt(E+P) and m/sqrt(E+P) would be a different
// function of (E, p, m) than the textbook u = (sqrt(E+m) chi, lambda P/sqrt(E+m) chi) of the plain definition
// (omega_- differs by ~1e-7 E^2/m^2), and the gauge cancellations of soft and collinear events amplify that
// difference; this form is the chiral rotation of the textbook spinor, term by term.
template <class T> MG_HD void omegas(T E, T P, T m, T& wp, T& wm) {
  if (m == (T)0) { wp = sqrt_<T>(P + P); wm = (T)0; return; }
  const T em = E + m;
  const T inv = rsqrt_<T>(em + em);
  wp = (em + P) * inv; wm = (em - P) * inv;
}
// u(p,l)    = (omega_{-l} chi_l ; omega_{l} chi_l)            incoming fermion   (IXXXXX)
// v(p,l)    = (omega_{l} chi_{-l} ; -omega_{-l} chi_{-l})     outgoing antifermion (IXXXXX)
// ubar, vbar = psi^dagger gamma^0 = (psi_R^dagger | psi_L^dagger)   outgoing fermion / incoming antifermion (OXXXXX)
template <class T> MG_HD Spinor<T> spinor_u(Mom<T> p, T m, int lambda) {
  const T P = sqrt_<T>(fma_<T>(p.v[1], p.v[1], fma_<T>(p.v[2], p.v[2], p.v[3] * p.v[3])));
  T wp, wm;
  omegas<T>(p.v[0], P, m, wp, wm);
  const Chi<T> x = chi<T>(p, P, lambda);
  const T wl = lambda > 0 ? wm : wp, wr = lambda > 0 ? wp : wm;
  Spinor<T> s;
  s.l[0] = wl * x.c[0]; s.l[1] = wl * x.c[1];
  s.r[0] = wr * x.c[0]; s.r[1] = wr * x.c[1];
  return s;
}
template <class T> MG_HD Spinor<T> spinor_v(Mom<T> p, T m, int lambda) {
  const T P = sqrt_<T>(fma_<T>(p.v[1], p.v[1], fma_<T>(p.v[2], p.v[2], p.v[3] * p.v[3])));
  T wp, wm;
  omegas<T>(p.v[0], P, m, wp, wm);
  const Chi<T> x = chi<T>(p, P, -lambda);
  const T wl = lambda > 0 ? wp : wm, wr = lambda > 0 ? -wm : -wp;
  Spinor<T> s;
  s.l[0] = wl * x.c[0]; s.l[1] = wl * x.c[1];
  s.r[0] = wr * x.c[0]; s.r[1] = wr * x.c[1];
  return s;
}
// row spinor of a column spinor: (a | b) = (psi_R^* | psi_L^*), stored as l = a, r = b.
template <class T> MG_HD Spinor<T> bar(const Spinor<T>& s) {
  Spinor<T> b;
  b.l[0] = conj_(s.r[0]); b.l[1] = conj_(s.r[1]);
  b.r[0] = conj_(s.l[0]); b.r[1] = conj_(s.l[1]);
  return b;
}

// Polarisation vector of helicity lambda = +-1 of a massless vector (VXXXXX):
//   eps = (0; -l cos(th)cos(ph) + i sin(ph), -l cos(th)sin(ph) - i cos(ph), l sin(th))/sqrt(2);
//   pT = 0: (0; -l sgn(pz), -i, 0)/sqrt(2).   Outgoing: complex conjugate.
template <class T> MG_HD Vec4<T> polvec(Mom<T> p, int lambda, bool outgoing) {
  const T px = p.v[1], py = p.v[2], pz = p.v[3];
  const T pt2 = fma_<T>(px, px, py * py);
  const T l = (T)lambda;
  const T r2 = (T)0.70710678118654752440084436210485;
  const T cj = outgoing ? (T)-1 : (T)1;
  Vec4<T> e;
  e.v[0] = cx<T>((T)0, (T)0);
  if (pt2 == (T)0) {
    const T sg = pz >= (T)0 ? (T)1 : (T)-1;
    e.v[1] = cx<T>(-l * sg * r2, (T)0);
    e.v[2] = cx<T>((T)0, -cj * r2);
    e.v[3] = cx<T>((T)0, (T)0);
    return e;
  }
  const T ipt = rsqrt_<T>(pt2);
  const T iP = rsqrt_<T>(fma_<T>(pz, pz, pt2));
  const T ct = pz * iP, st = pt2 * ipt * iP, cp = px * ipt, sp = py * ipt;
  e.v[1] = cx<T>(-l * ct * cp * r2, cj * sp * r2);
  e.v[2] = cx<T>(-l * ct * sp * r2, -cj * cp * r2);
  e.v[3] = cx<T>(l * st * r2, (T)0);
  return e;
}

// ---------------------------------------------------------------------------------------------
// Fermion-line algebra.  S(V) = V0 - sigma.V (acts on R, result L), Sb(V) = V0 + sigma.V.
//   Vslash psi      = ( S(V) psi_R ; Sb(V) psi_L )
//   psibar Vslash   = ( b Sb(V) | a S(V) )
// ---------------------------------------------------------------------------------------------
template <class T> struct Slash { cx<T> p03, m03, p12, m12; };  // V0+V3, V0-V3, V1+iV2, V1-iV2
template <class T> MG_HD Slash<T> slash_parts(const Vec4<T>& V) {
  Slash<T> s;
  s.p03 = V.v[0] + V.v[3];
  s.m03 = V.v[0] - V.v[3];
  s.p12 = cx<T>(V.v[1].re - V.v[2].im, V.v[1].im + V.v[2].re);
  s.m12 = cx<T>(V.v[1].re + V.v[2].im, V.v[1].im - V.v[2].re);
  return s;
}
// column: out = Vslash psi
template <class T> MG_HD Spinor<T> slash_col(const Slash<T>& s, const Spinor<T>& x) {
  Spinor<T> o;
  o.l[0] = cfms(s.m12, x.r[1], s.m03 * x.r[0]);   // (V0-V3) r0 - (V1-iV2) r1
  o.l[1] = cfms(s.p12, x.r[0], s.p03 * x.r[1]);   // -(V1+iV2) r0 + (V0+V3) r1
  o.r[0] = cfma(s.m12, x.l[1], s.p03 * x.l[0]);   // (V0+V3) l0 + (V1-iV2) l1
  o.r[1] = cfma(s.p12, x.l[0], s.m03 * x.l[1]);   // (V1+iV2) l0 + (V0-V3) l1
  return o;
}
// row: out = psibar Vslash,  (a|b) = (x.l | x.r)
template <class T> MG_HD Spinor<T> slash_row(const Slash<T>& s, const Spinor<T>& x) {
  Spinor<T> o;
  o.l[0] = cfma(x.r[1], s.p12, x.r[0] * s.p03);   // b0 (V0+V3) + b1 (V1+iV2)
  o.l[1] = cfma(x.r[0], s.m12, x.r[1] * s.m03);   // b0 (V1-iV2) + b1 (V0-V3)
  o.r[0] = cfms(x.l[1], s.p12, x.l[0] * s.m03);   // a0 (V0-V3) - a1 (V1+iV2)
  o.r[1] = cfms(x.l[0], s.m12, x.l[1] * s.p03);   // -a0 (V1-iV2) + a1 (V0+V3)
  return o;
}
// (qslash + m) acting on a column, q real
template <class T> MG_HD Spinor<T> qslash_m_col(Mom<T> q, T m, const Spinor<T>& x) {
  const T p03 = q.v[0] + q.v[3], m03 = q.v[0] - q.v[3];
  const cx<T> p12(q.v[1], q.v[2]), m12(q.v[1], -q.v[2]);
  Spinor<T> o;
  o.l[0] = rfma(m, x.l[0], cfms(m12, x.r[1], m03 * x.r[0]));
  o.l[1] = rfma(m, x.l[1], cfms(p12, x.r[0], p03 * x.r[1]));
  o.r[0] = rfma(m, x.r[0], cfma(m12, x.l[1], p03 * x.l[0]));
  o.r[1] = rfma(m, x.r[1], cfma(p12, x.l[0], m03 * x.l[1]));
  return o;
}
// row times (qslash + m)
template <class T> MG_HD Spinor<T> qslash_m_row(Mom<T> q, T m, const Spinor<T>& x) {
  const T p03 = q.v[0] + q.v[3], m03 = q.v[0] - q.v[3];
  const cx<T> p12(q.v[1], q.v[2]), m12(q.v[1], -q.v[2]);
  Spinor<T> o;
  o.l[0] = rfma(m, x.l[0], cfma(x.r[1], p12, p03 * x.r[0]));
  o.l[1] = rfma(m, x.l[1], cfma(x.r[0], m12, m03 * x.r[1]));
  o.r[0] = rfma(m, x.r[0], cfms(x.l[1], p12, m03 * x.l[0]));
  o.r[1] = rfma(m, x.r[1], cfms(x.l[0], m12, p03 * x.l[1]));
  return o;
}
template <class T> MG_HD Spinor<T> scale(T s, const Spinor<T>& x) {
  Spinor<T> o;
  o.l[0] = s * x.l[0]; o.l[1] = s * x.l[1]; o.r[0] = s * x.r[0]; o.r[1] = s * x.r[1];
  return o;
}
template <class T> MG_HD Vec4<T> scale(T s, const Vec4<T>& x) {
  Vec4<T> o;
  o.v[0] = s * x.v[0]; o.v[1] = s * x.v[1]; o.v[2] = s * x.v[2]; o.v[3] = s * x.v[3];
  return o;
}

// FFV1_1-type (reduced): psibar' = psibar Vslash (qslash+m) * iden,   iden = 1/(q^2-m^2)
template <class T> MG_HD Spinor<T> ffv_row_prop(const Spinor<T>& psibar, const Vec4<T>& V, Mom<T> q, T m, T iden) {
  return scale(iden, qslash_m_row(q, m, slash_row(slash_parts(V), psibar)));
}
// FFV1_2-type (reduced): psi' = (qslash+m) Vslash psi * iden
template <class T> MG_HD Spinor<T> ffv_col_prop(const Spinor<T>& psi, const Vec4<T>& V, Mom<T> q, T m, T iden) {
  return scale(iden, qslash_m_col(q, m, slash_col(slash_parts(V), psi)));
}
// row . column
template <class T> MG_HD cx<T> row_col(const Spinor<T>& b, const Spinor<T>& x) {
  cx<T> r = b.l[0] * x.l[0];
  r = cfma(b.l[1], x.l[1], r);
  r = cfma(b.r[0], x.r[0], r);
  r = cfma(b.r[1], x.r[1], r);
  return r;
}
// FFV1_0-type (reduced): psibar Vslash psi
template <class T> MG_HD cx<T> ffv_amp(const Spinor<T>& psibar, const Vec4<T>& V, const Spinor<T>& psi) {
  return row_col(psibar, slash_col(slash_parts(V), psi));
}
// FFV1P0_3-type (reduced, no propagator): J^mu = psibar gamma^mu psi = a sigma^mu psi_R + b sigmabar^mu psi_L
template <class T> MG_HD Vec4<T> ff_current(const Spinor<T>& bq, const Spinor<T>& x) {
  const cx<T> a0r0 = bq.l[0] * x.r[0], a1r1 = bq.l[1] * x.r[1], a0r1 = bq.l[0] * x.r[1], a1r0 = bq.l[1] * x.r[0];
  const cx<T> b0l0 = bq.r[0] * x.l[0], b1l1 = bq.r[1] * x.l[1], b0l1 = bq.r[0] * x.l[1], b1l0 = bq.r[1] * x.l[0];
  Vec4<T> J;
  J.v[0] = (a0r0 + a1r1) + (b0l0 + b1l1);
  J.v[3] = (a0r0 - a1r1) - (b0l0 - b1l1);
  const cx<T> s = (a0r1 + a1r0) - (b0l1 + b1l0);     // sigma^1
  const cx<T> d = (a1r0 - a0r1) - (b1l0 - b0l1);     // sigma^2 = i * d
  J.v[1] = s;
  J.v[2] = times_i(d);
  return J;
}

// ---------------------------------------------------------------------------------------------
// Gluon self-couplings (reduced).
//   V3^{mu nu rho}(k1,k2,k3) J1_mu J2_nu = (J1.J2)(k1-k2)^rho + (J1.(k2-k3)) J2^rho + (J2.(k3-k1)) J1^rho,
//   k3 = -(k1+k2)  =>  k2-k3 = k1+2 k2,  k3-k1 = -(2 k1+k2).
// vvv_cur ADDS sign * that vector to acc (VVV1P0_1 without the 1/K^2); vvv_amp contracts with J3.
// ---------------------------------------------------------------------------------------------
template <class T, bool INIT> MG_HD void vvv_cur(Vec4<T>& acc, T sign, const Vec4<T>& J1, Mom<T> k1, const Vec4<T>& J2, Mom<T> k2) {
  Mom<T> d, e, f;
#pragma unroll
  for (int i = 0; i < 4; ++i) { d.v[i] = k1.v[i] - k2.v[i]; e.v[i] = fma_<T>((T)2, k2.v[i], k1.v[i]); f.v[i] = -fma_<T>((T)2, k1.v[i], k2.v[i]); }
  const cx<T> j12 = sign * mdot(J1, J2);
  const cx<T> a = sign * mdot(J1, e);
  const cx<T> b = sign * mdot(J2, f);
#pragma unroll
  for (int i = 0; i < 4; ++i) acc.v[i] = cfma(b, J1.v[i], cfma(a, J2.v[i], INIT ? d.v[i] * j12 : rfma(d.v[i], j12, acc.v[i])));
}
// full contraction V3(k1,k2,k3) J1 J2 J3 with k3 = -(k1+k2)
template <class T> MG_HD cx<T> vvv_amp(const Vec4<T>& J1, Mom<T> k1, const Vec4<T>& J2, Mom<T> k2, const Vec4<T>& J3) {
  Mom<T> d, e, f;
#pragma unroll
  for (int i = 0; i < 4; ++i) { d.v[i] = k1.v[i] - k2.v[i]; e.v[i] = fma_<T>((T)2, k2.v[i], k1.v[i]); f.v[i] = -fma_<T>((T)2, k1.v[i], k2.v[i]); }
  cx<T> r = mdot(J1, J2) * mdot(J3, d);
  r = cfma(mdot(J2, J3), mdot(J1, e), r);
  r = cfma(mdot(J3, J1), mdot(J2, f), r);
  return r;
}
// Four-gluon structures for legs A,B,C -> open index (VVVV{1,3,4}P0_1 without 1/K^2):
//   s1 = (A.C) B - (B.C) A   [colour [[A,B],C]]
//   s2 = (A.B) C - (B.C) A   [colour [[A,C],B]]
//   s3 = (A.B) C - (A.C) B   [colour [[B,C],A]]
template <class T, bool INIT> MG_HD void vvvv_cur(Vec4<T>& acc, T sign, int which, const Vec4<T>& A, const Vec4<T>& B, const Vec4<T>& C) {
  if (which == 1) {
    const cx<T> ac = sign * mdot(A, C), bc = sign * mdot(B, C);
#pragma unroll
    for (int i = 0; i < 4; ++i) acc.v[i] = cfms(bc, A.v[i], INIT ? ac * B.v[i] : cfma(ac, B.v[i], acc.v[i]));
  } else if (which == 2) {
    const cx<T> ab = sign * mdot(A, B), bc = sign * mdot(B, C);
#pragma unroll
    for (int i = 0; i < 4; ++i) acc.v[i] = cfms(bc, A.v[i], INIT ? ab * C.v[i] : cfma(ab, C.v[i], acc.v[i]));
  } else {
    const cx<T> ab = sign * mdot(A, B), ac = sign * mdot(A, C);
#pragma unroll
    for (int i = 0; i < 4; ++i) acc.v[i] = cfms(ac, B.v[i], INIT ? ab * C.v[i] : cfma(ab, C.v[i], acc.v[i]));
  }
}
template <class T> MG_HD cx<T> vvvv_amp(int which, const Vec4<T>& A, const Vec4<T>& B, const Vec4<T>& C, const Vec4<T>& D) {
  if (which == 1) return cfms(mdot(B, C), mdot(A, D), mdot(A, C) * mdot(B, D));
  if (which == 2) return cfms(mdot(B, C), mdot(A, D), mdot(A, B) * mdot(C, D));
  return cfms(mdot(A, C), mdot(B, D), mdot(A, B) * mdot(C, D));
}

}  // namespace mg
