// ORACLE — test infrastructure only (see philox.hpp header).
//
// u u~ -> t t~ (+ g) at tree level: the quark-initiated channel of SURVEY.md §8(f) N4 (§2: the generator is
// validated on "more complex QCD processes ... more directly relevant to LHC physics"), as the PLAIN DEFINITION
//     ME = (1/36) sum_helicities sum_{every colour assignment} | sum of Feynman diagrams |^2
// with the textbook QCD rules written out in me_qcd.hpp's header (q q g: i gs gamma^mu T^a; quark propagator
// i(qslash + m)/(q^2 - m^2); gluon propagator -i g^{mu nu} delta^{ab}/k^2; three-gluon vertex, all momenta incoming,
// gs f^{abc}[g^{mu nu}(k1-k2)^rho + g^{nu rho}(k2-k3)^mu + g^{rho mu}(k3-k1)^nu]), explicit 4x4 Dirac matrices
// (dirac.hpp) and explicit Gell-Mann matrices and structure constants (Su3 of me_qcd.hpp).  Colours are summed by
// brute force: 3^4 (x 8) assignments, no colour basis, no colour matrix.  The paper prints none of this.
//
// Particle order: 0 = u (incoming, colour k), 1 = u~ (incoming, colour l), 2 = t (colour i), 3 = t~ (colour j),
// 4 = g (colour a).  Massless u, helicity +-1 for everyone (R10); helicity index: bit k = helicity of particle k.
// Averaging: 1/4 spins x 1/9 colours = 1/36.
//
//   u u~ -> t t~ :   M = [vbar1 (i gs gamma^mu T^c) u0] (-i / s) [ubar2 (i gs gamma_mu T^c) v3]
//   u u~ -> t t~ g, with J^mu = vbar1 gamma^mu u0, G^mu = ubar2 gamma^mu v3, s_q = (p0+p1)^2, s_t = (p2+p3)^2, k = p4:
//     D1 (g off t)    -i gs^3 (T^a T^c)_ij (T^c)_lk  ubar2 eps-slash (p2-slash + k-slash + m) gamma_mu v3 J^mu / ((p2+k)^2 - m^2) / s_q
//     D2 (g off t~)   -i gs^3 (T^c T^a)_ij (T^c)_lk  ubar2 gamma_mu (-p3-slash - k-slash + m) eps-slash v3 J^mu / ((p3+k)^2 - m^2) / s_q
//     D3 (g off u)    -i gs^3 (T^c)_ij (T^c T^a)_lk  vbar1 gamma_mu (p0-slash - k-slash) eps-slash u0 G^mu / (p0-k)^2 / s_t
//     D4 (g off u~)   -i gs^3 (T^c)_ij (T^a T^c)_lk  vbar1 eps-slash (k-slash - p1-slash) gamma_mu u0 G^mu / (p1-k)^2 / s_t
//     D5 (g g g)         gs^3 f^{bca} (T^b)_lk (T^c)_ij  V3(J, p0+p1; G, -(p2+p3); eps, -k) / (s_q s_t)
//   (three vertices i gs each and one quark and one gluon propagator, i and -i, give -i gs^3; D5: (i gs)^2 (-i)^2 gs).
//
// Pins (tests/test_oracle_me.py): the closed form (4 gs^4/9)(tau1^2 + tau2^2 + rho/2) of q q~ -> Q Q~; gauge invariance
// (eps -> k gives zero for every colour assignment) and Lorentz invariance of u u~ -> t t~ g; its absolute normalisation
// through the initial-state collinear limit  ME -> (2 gs^2 / (2 p0.k)) (1/z) C_F (1+z^2)/(1-z) ME(u u~ -> t t~)(z p0, p1).
#pragma once
#include <vector>
#include "common.hpp"
#include "dirac.hpp"
#include "me_qcd.hpp"

namespace oracle {

// psibar gamma^mu psi as a contravariant vector
template <class T> Vec4<T> bilinear(const Row4<T>& a, const Col4<T>& b) {
  Vec4<T> r;
  for (int mu = 0; mu < 4; ++mu) r.v[mu] = mul(a, mul(gamma_mu<T>(mu), b));
  return r;
}
// psibar M gamma^mu psi and psibar gamma^mu M psi as contravariant vectors
template <class T> Vec4<T> bilinear_left(const Row4<T>& a, const Mat4<T>& M, const Col4<T>& b) {
  Vec4<T> r;
  const Row4<T> aM = mul(a, M);
  for (int mu = 0; mu < 4; ++mu) r.v[mu] = mul(aM, mul(gamma_mu<T>(mu), b));
  return r;
}
template <class T> Vec4<T> bilinear_right(const Row4<T>& a, const Mat4<T>& M, const Col4<T>& b) {
  Vec4<T> r;
  const Col4<T> Mb = mul(M, b);
  for (int mu = 0; mu < 4; ++mu) r.v[mu] = mul(a, mul(gamma_mu<T>(mu), Mb));
  return r;
}

// Colour factors of the five diagrams of u u~ -> t t~ g for every colour assignment, written out from the rules above:
// C[d][a][((i*3+j)*3+k)*3+l], d = 0..4 for D1..D5 (tables only so that the sums over c, b are not redone per event).
template <class T> struct QqColour {
  cx<T> C[5][8][81];
  QqColour() {
    const Su3<T> su3;
    for (int a = 0; a < 8; ++a) {
      cx<T> TaTc[8][3][3] = {}, TcTa[8][3][3] = {};
      for (int c = 0; c < 8; ++c) for (int x = 0; x < 3; ++x) for (int y = 0; y < 3; ++y) for (int z = 0; z < 3; ++z) {
        TaTc[c][x][y] += su3.Ta[a][x][z] * su3.Ta[c][z][y];
        TcTa[c][x][y] += su3.Ta[c][x][z] * su3.Ta[a][z][y];
      }
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k) for (int l = 0; l < 3; ++l) {
        const int x = ((i * 3 + j) * 3 + k) * 3 + l;
        for (int d = 0; d < 5; ++d) C[d][a][x] = 0;
        for (int c = 0; c < 8; ++c) {
          C[0][a][x] += TaTc[c][i][j] * su3.Ta[c][l][k];
          C[1][a][x] += TcTa[c][i][j] * su3.Ta[c][l][k];
          C[2][a][x] += su3.Ta[c][i][j] * TcTa[c][l][k];
          C[3][a][x] += su3.Ta[c][i][j] * TaTc[c][l][k];
          for (int b = 0; b < 8; ++b) C[4][a][x] += su3.f[b][c][a] * su3.Ta[b][l][k] * su3.Ta[c][i][j];
        }
      }
    }
  }
};

// ng = 0: u u~ -> t t~; ng = 1: u u~ -> t t~ g.  hel_out[2^(4+ng)] optional: colour-summed |M|^2 of every helicity
// combination (couplings included, before the 1/36).  gauge: the gluon polarisation is replaced by its momentum / energy.
// max_colour_amp (optional): largest |M| over colour assignments and helicities (for the gauge-invariance pin).
template <class T>
T qq_me(int ng, const Params& par, const T (*p)[4], T* hel_out = nullptr, bool gauge = false, T* max_colour_amp = nullptr) {
  static const Su3<T> su3;
  static const QqColour<T> col;
  const int npar = 4 + ng, nhel = 1 << npar;
  const T gs = std::sqrt(4 * pi_v<T>() * (T)par.alpha_s), m = (T)par.mt;
  const cx<T> I(0, 1);
  T P01[4], P23[4];
  for (int mu = 0; mu < 4; ++mu) { P01[mu] = p[0][mu] + p[1][mu]; P23[mu] = p[2][mu] + p[3][mu]; }
  auto sq = [](const T* q) { return q[0] * q[0] - q[1] * q[1] - q[2] * q[2] - q[3] * q[3]; };
  const T s_q = sq(P01), s_t = sq(P23);
  T total = 0, amax = 0;
  for (int ihel = 0; ihel < nhel; ++ihel) {
    auto hel = [&](int k) { return ((ihel >> k) & 1) ? 1 : -1; };
    const Col4<T> u0 = spinor_u<T>(p[0], (T)0, hel(0));
    const Row4<T> vb1 = bar(spinor_v<T>(p[1], (T)0, hel(1)));
    const Row4<T> ub2 = bar(spinor_u<T>(p[2], m, hel(2)));
    const Col4<T> v3 = spinor_v<T>(p[3], m, hel(3));
    const Vec4<T> J = bilinear(vb1, u0), G = bilinear(ub2, v3);
    T sum = 0;
    if (ng == 0) {
      const cx<T> lor = I * gs * gs * mdot(J, G) / s_q;
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k) for (int l = 0; l < 3; ++l) {
        cx<T> col = 0;
        for (int c = 0; c < 8; ++c) col += su3.Ta[c][l][k] * su3.Ta[c][i][j];
        const cx<T> M = col * lor;
        sum += std::norm(M);
        amax = std::max(amax, std::abs(M));
      }
    } else {
      const T* k = p[4];
      Vec4<T> eps = vconj(polvec<T>(k, hel(4)));                       // outgoing gluon
      if (gauge) for (int mu = 0; mu < 4; ++mu) eps.v[mu] = cx<T>(k[mu] / k[0], 0);
      const Mat4<T> E = slash(eps);
      T q1[4], q2[4], q3[4], q4[4];
      for (int mu = 0; mu < 4; ++mu) {
        q1[mu] = p[2][mu] + k[mu]; q2[mu] = -p[3][mu] - k[mu]; q3[mu] = p[0][mu] - k[mu]; q4[mu] = k[mu] - p[1][mu];
      }
      const Mat4<T> S1 = madd(slash(real_vec<T>(q1)), mscale(identity4<T>(), cx<T>(m, 0)));
      const Mat4<T> S2 = madd(slash(real_vec<T>(q2)), mscale(identity4<T>(), cx<T>(m, 0)));
      const Mat4<T> S3 = slash(real_vec<T>(q3)), S4 = slash(real_vec<T>(q4));
      const cx<T> A1 = mdot(bilinear_left(ub2, mmul(E, S1), v3), J) / ((sq(q1) - m * m) * s_q);
      const cx<T> A2 = mdot(bilinear_right(ub2, mmul(S2, E), v3), J) / ((sq(q2) - m * m) * s_q);
      const cx<T> A3 = mdot(bilinear_right(vb1, mmul(S3, E), u0), G) / (sq(q3) * s_t);
      const cx<T> A4 = mdot(bilinear_left(vb1, mmul(E, S4), u0), G) / (sq(q4) * s_t);
      Vec4<T> k1 = real_vec<T>(P01), k2 = real_vec<T>(P23, (T)-1), k3 = real_vec<T>(k, (T)-1);
      const cx<T> A5 = mdot(v3_contract(J, k1, G, k2, k3), eps) / (s_q * s_t);
      const cx<T> f14 = -I * gs * gs * gs, f5 = gs * gs * gs;
      for (int a = 0; a < 8; ++a)
        for (int x = 0; x < 81; ++x) {
          const cx<T> M = f14 * (col.C[0][a][x] * A1 + col.C[1][a][x] * A2 + col.C[2][a][x] * A3 + col.C[3][a][x] * A4) + f5 * col.C[4][a][x] * A5;
          sum += std::norm(M);
          amax = std::max(amax, std::abs(M));
        }
    }
    if (hel_out) hel_out[ihel] = sum;
    total += sum;
  }
  if (max_colour_amp) *max_colour_amp = amax;
  return total / 36;
}

}  // namespace oracle
