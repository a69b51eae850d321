// eemumu.cuh — sigmaKin for e+ e- -> mu+ mu- (photon + Z), hand-written in the routine order of
// PAPER.md:33 (Fig. 1 caption): external wavefunctions (IXXXXX/OXXXXX) for the four fermions, then
//   FFV1P0_3 : photon off-shell wavefunction from the e+ e- gamma vertex (incl. propagator 1/s)
//   FFV1_0   : amplitude of diagram (a) from the gamma mu mu vertex
//   FFV2_4_3 : Z off-shell wavefunction from the e+ e- Z vertex (incl. propagator)
//   FFV2_4_0 : amplitude of diagram (b) from the Z mu mu vertex
// "The two amplitudes are added to each other, their sum is squared, and the result is averaged
// over all valid helicity combinations".
//
// Rules (R13-R15): l l gamma: i e gamma^mu;  l l Z: i e/(sW cW) gamma^mu (gL PL + gR PR);
// photon propagator -i g/q^2;  Z propagator -i (g - q q/mZ^2)/(q^2 - mZ^2 + i mZ GammaZ).  Both diagrams
// carry the same overall factor i^2 (-i) = i, dropped.  Massless leptons: the chirality block that
// vanishes is an exact zero, so exactly 4 of the 16 helicity combinations are non-zero.
// Particle order (R9): 0 = e+, 1 = e-, 2 = mu+, 3 = mu-.
#pragma once
#include "helas.cuh"

namespace mg {

struct Eemumu {
  static constexpr int NHEL = 16;
  static constexpr int NPAR = 4;
#ifndef MG_EE_MINB
#define MG_EE_MINB 6
#endif
  static constexpr int MINB = MG_EE_MINB;   // resident CTAs of 128 threads the register allocation aims at
  // Massless helicity spinors need three reals per particle (the "simplified" IXXXXX/OXXXXX of PAPER.md:136):
  //   omega_+ chi_+ = (a, b),  omega_+ chi_- = (-b^*, a),   a = sqrt(P+pz),  b = (px + i py)/sqrt(P+pz),
  // P+pz evaluated as pT^2/(P-pz) for pz < 0 (R19); along -z: a = 0, b = sqrt(2P) (B1).  One square root, one
  // reciprocal square root and at most one division per particle and event, shared by all 16 helicity combinations.
  template <class T> struct Event { Mom<T> p[4]; Mom<T> q; T is; cx<T> bw; T a[4]; cx<T> b[4]; };

  template <class T> static MG_HD void massless_frame(Mom<T> p, T& a, cx<T>& b) {
    const T px = p.v[1], py = p.v[2], pz = p.v[3];
    const T pt2 = fma_<T>(px, px, py * py);
    const T P = sqrt_<T>(fma_<T>(pz, pz, pt2));
    if (pt2 == (T)0 && pz < (T)0) { a = (T)0; b = cx<T>(sqrt_<T>(P + P), (T)0); return; }
    const T Ppz = (pz >= (T)0) ? (P + pz) : pt2 / (P - pz);
    const T r = rsqrt_<T>(Ppz);
    a = Ppz * r;
    b = cx<T>(px * r, py * r);
  }
  // u(p, l): incoming fermion; v(p, l): outgoing antifermion (helas.cuh spinor_u / spinor_v at m = 0)
  template <class T> static MG_HD Spinor<T> u0(T a, cx<T> b, int l) {
    Spinor<T> s;
    const cx<T> z((T)0, (T)0);
    if (l > 0) { s.l[0] = z; s.l[1] = z; s.r[0] = cx<T>(a, (T)0); s.r[1] = b; }
    else { s.l[0] = cx<T>(-b.re, b.im); s.l[1] = cx<T>(a, (T)0); s.r[0] = z; s.r[1] = z; }
    return s;
  }
  template <class T> static MG_HD Spinor<T> v0(T a, cx<T> b, int l) {
    Spinor<T> s;
    const cx<T> z((T)0, (T)0);
    if (l > 0) { s.l[0] = cx<T>(-b.re, b.im); s.l[1] = cx<T>(a, (T)0); s.r[0] = z; s.r[1] = z; }
    else { s.l[0] = z; s.l[1] = z; s.r[0] = cx<T>(-a, (T)0); s.r[1] = -b; }
    return s;
  }

  template <class T> static MG_HD void finish(Event<T>& ev, const Consts& k) {
    ev.q = ev.p[0] + ev.p[1];
    const T s = mdot(ev.q, ev.q);
    ev.is = (T)1 / s;
    // 1/(s - mZ^2 + i mZ GZ)
    const T dr = s - (T)k.mZ2, di = (T)k.mZgZ;
    const T inv = (T)1 / fma_<T>(dr, dr, di * di);
    ev.bw = cx<T>(dr * inv, -di * inv);
#pragma unroll
    for (int i = 0; i < 4; ++i) massless_frame<T>(ev.p[i], ev.a[i], ev.b[i]);
  }

  template <class T> static MG_HD T helicity(const Event<T>& ev, int ihel, const Consts& k) {
    const int h0 = (ihel & 1) ? 1 : -1, h1 = (ihel & 2) ? 1 : -1, h2 = (ihel & 4) ? 1 : -1, h3 = (ihel & 8) ? 1 : -1;
    // OXXXXX / IXXXXX: incoming e+ -> vbar, incoming e- -> u, outgoing mu+ -> v, outgoing mu- -> ubar
    const Spinor<T> vbar_ep = bar(v0<T>(ev.a[0], ev.b[0], h0));
    const Spinor<T> u_em = u0<T>(ev.a[1], ev.b[1], h1);
    const Spinor<T> v_mup = v0<T>(ev.a[2], ev.b[2], h2);
    const Spinor<T> ubar_mum = bar(u0<T>(ev.a[3], ev.b[3], h3));
    const T e = (T)k.ee, gzl = (T)k.gzl, gzr = (T)k.gzr;

    // chirality-split current of the electron line: J_R = a sigma^mu psi_R, J_L = b sigmabar^mu psi_L
    Spinor<T> onlyR = vbar_ep, onlyL = vbar_ep;
    onlyR.r[0] = onlyR.r[1] = cx<T>(0, 0);   // keep a (couples to psi_R)
    onlyL.l[0] = onlyL.l[1] = cx<T>(0, 0);   // keep b (couples to psi_L)
    const Vec4<T> JR = ff_current(onlyR, u_em);
    const Vec4<T> JL = ff_current(onlyL, u_em);

    // FFV1P0_3: A^mu = e (J_L + J_R)^mu / s
    Vec4<T> A;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) A.v[mu] = (e * ev.is) * (JL.v[mu] + JR.v[mu]);
    // FFV1_0: e ubar Aslash v
    const cx<T> amp_a = e * ffv_amp(ubar_mum, A, v_mup);

    // FFV2_4_3: Z^mu = [Jz^mu - q^mu (Jz.q)/mZ^2] / (s - mZ^2 + i mZ GZ),  Jz = gzl J_L + gzr J_R
    Vec4<T> Jz;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) Jz.v[mu] = rfma(gzr, JR.v[mu], gzl * JL.v[mu]);
    const cx<T> jq = ((T)1 / (T)k.mZ2) * mdot(Jz, ev.q);
    Vec4<T> Z;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) Z.v[mu] = ev.bw * rfma(-ev.q.v[mu], jq, Jz.v[mu]);
    // FFV2_4_0: ubar Zslash (gzl PL + gzr PR) v = gzl b.Sb(Z) v_L + gzr a.S(Z) v_R
    const Spinor<T> zv = slash_col(slash_parts(Z), v_mup);   // (S(Z) v_R ; Sb(Z) v_L)
    cx<T> aR = cfma(ubar_mum.l[1], zv.l[1], ubar_mum.l[0] * zv.l[0]);
    cx<T> bL = cfma(ubar_mum.r[1], zv.r[1], ubar_mum.r[0] * zv.r[0]);
    const cx<T> amp_b = rfma(gzr, aR, gzl * bL);

    return norm2(amp_a + amp_b);
  }
};

}  // namespace mg
