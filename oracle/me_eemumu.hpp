// ORACLE — test infrastructure only (see philox.hpp header).
//
// e+ e- -> mu+ mu- at tree level: photon + Z exchange, helicity by helicity, from the plain Feynman
// rules with explicit 4x4 Dirac matrices.
//
// Serves PAPER.md:33 (Fig. 1 caption: two diagrams, (a) photon and (b) Z exchange; "The two
// amplitudes are added to each other, their sum is squared, and the result is averaged over all
// valid helicity combinations"; "sixteen helicity combinations ... only four of those are allowed")
// and PAPER.md:35 (§2).  The paper prints no formula; rules as in DESIGN.md "Conventions"
// (readings R13-R15): vertex l l gamma = i e gamma^mu (charge -1), l l Z = i e/(sW cW) gamma^mu
// (gL PL + gR PR), gL = -1/2 + sW^2, gR = sW^2, sW^2 = 1 - mW^2/mZ^2, e = sqrt(4 pi alpha);
// photon propagator -i g/q^2, Z propagator -i (g - q q/mZ^2)/(q^2 - mZ^2 + i mZ GammaZ).
// Particle order (reading R9): 0 = e+ (beam +z), 1 = e- (beam -z), 2 = mu+, 3 = mu-.
// Helicity combination index: bit k = helicity of particle k (0 <-> -1, 1 <-> +1).
#pragma once
#include "common.hpp"
#include "dirac.hpp"

namespace oracle {

// |M|^2 for ONE helicity combination (no averaging factor).
template <class T>
T eemumu_hel(const Params& par, const T (*p)[4], int ihel) {
  const cx<T> I(0, 1);
  const T pi = pi_v<T>();
  const T e = std::sqrt(4 * pi / (T)par.alpha_em_inv);
  const T mZ = (T)par.mZ, gZ = (T)par.gammaZ, mW = (T)par.mW;
  const T sw2 = 1 - (mW * mW) / (mZ * mZ);
  const T cw2 = 1 - sw2;
  const T gL = -(T)0.5 + sw2, gR = sw2;
  int h[4];
  for (int k = 0; k < 4; ++k) h[k] = ((ihel >> k) & 1) ? +1 : -1;

  // external wavefunctions: incoming e+ -> vbar, incoming e- -> u, outgoing mu+ -> v, outgoing mu- -> ubar
  Row4<T> vbar_ep = bar(spinor_v<T>(p[0], 0, h[0]));
  Col4<T> u_em = spinor_u<T>(p[1], 0, h[1]);
  Col4<T> v_mup = spinor_v<T>(p[2], 0, h[2]);
  Row4<T> ubar_mum = bar(spinor_u<T>(p[3], 0, h[3]));

  // chiral projectors and the Z vertex matrix (gL PL + gR PR)
  Mat4<T> one = identity4<T>(), g5 = gamma_5<T>();
  Mat4<T> PL = mscale(madd(one, mscale(g5, cx<T>(-1, 0))), cx<T>((T)0.5, 0));
  Mat4<T> PR = mscale(madd(one, g5), cx<T>((T)0.5, 0));
  Mat4<T> chir = madd(mscale(PL, cx<T>(gL, 0)), mscale(PR, cx<T>(gR, 0)));
  const cx<T> cg = I * e;                                // photon vertex coefficient
  const cx<T> cz = I * e / std::sqrt(sw2 * cw2);         // Z vertex coefficient

  Vec4<T> Je_g, Jm_g, Je_z, Jm_z;
  for (int mu = 0; mu < 4; ++mu) {
    Mat4<T> g = gamma_mu<T>(mu);
    Je_g.v[mu] = cg * mul(vbar_ep, mul(g, u_em));
    Jm_g.v[mu] = cg * mul(ubar_mum, mul(g, v_mup));
    Mat4<T> gz = mmul(g, chir);
    Je_z.v[mu] = cz * mul(vbar_ep, mul(gz, u_em));
    Jm_z.v[mu] = cz * mul(ubar_mum, mul(gz, v_mup));
  }
  Vec4<T> q = vadd(real_vec<T>(p[0]), real_vec<T>(p[1]));
  cx<T> s = mdot(q, q);
  cx<T> Mg = mdot(Je_g, Jm_g) * (-I) / s;
  cx<T> Mz = (mdot(Je_z, Jm_z) - mdot(Je_z, q) * mdot(Jm_z, q) / (mZ * mZ)) * (-I) /
             (s - mZ * mZ + I * mZ * gZ);
  cx<T> M = Mg + Mz;
  return std::norm(M);
}

// ME = (1/4) sum over the 16 helicity combinations (reading R11); hel_out[16] optional.
template <class T>
T eemumu_me(const Params& par, const T (*p)[4], T* hel_out = nullptr) {
  T sum = 0;
  for (int ihel = 0; ihel < 16; ++ihel) {
    T m2 = eemumu_hel<T>(par, p, ihel);
    if (hel_out) hel_out[ihel] = m2;
    sum += m2;
  }
  return sum / 4;
}

}  // namespace oracle
