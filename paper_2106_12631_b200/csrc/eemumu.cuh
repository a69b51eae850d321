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
  static constexpr bool FLIP = false;   // chiral Z couplings: |M(h)|^2 != |M(-h)|^2
  static constexpr int MINB = 6;            // resident CTAs of 128 threads the register allocation aims at
  // Where the two single-chirality currents of a helicity combination are evaluated.  Each line has ONE non-zero helicity
  // assignment per chirality, so the 16 combinations share four currents and their four contractions with q.  FP32 evaluates
  // them once per event (696 -> 504 flops per event: 0.47 -> 0.41 ms per 2^24 events).  FP64 keeps them inside the
  // helicity loop: four currents are 64 registers in double, which costs a resident CTA or spills — measured in bench.py's
  // step 0.77 (5 CTAs, 96 registers) / 0.82 ms (4 CTAs, 122) against 0.76 ms with the currents in the loop (6 CTAs, 80).
  template <class T> static constexpr bool per_event_currents() { return sizeof(T) == 4; }
  // Massless helicity spinors need three reals per particle (the "simplified" IXXXXX/OXXXXX of PAPER.md:136):
  //   omega_+ chi_+ = (a, b),  omega_+ chi_- = (-b^*, a),   a = sqrt(P+pz),  b = (px + i py)/sqrt(P+pz),
  // P+pz evaluated as pT^2/(P-pz) for pz < 0 (R19); along -z: a = 0, b = sqrt(2P) (B1).  One square root, one
  // reciprocal square root and at most one division per particle and event, shared by all 16 helicity combinations.
  // Each of the two currents has ONE non-zero helicity assignment per chirality, so all 16 helicity combinations share
  // four currents and their four contractions with q: they are evaluated once per event (finish), and a helicity
  // combination only selects one of each and does the final contraction (helicity)
  template <class T> struct Event { Mom<T> p[4]; Mom<T> q; T is; cx<T> bw; T a[4]; cx<T> b[4]; Vec4<T> JeR, JeL, JmR, JmL; cx<T> qeR, qeL, qmR, qmL; };

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
  // helas.cuh spinor_u / spinor_v at m = 0 in terms of (a, b):
  //   u(p, +) = (0 ; (a, b))        u(p, -) = ((-b^*, a) ; 0)          incoming fermion
  //   v(p, +) = ((-b^*, a) ; 0)     v(p, -) = (0 ; (-a, -b))           outgoing antifermion
  //   psibar = (psi_R^* | psi_L^*): the a-block meets psi_R, the b-block meets psi_L

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
    if (!per_event_currents<T>()) return;
    const T a0 = ev.a[0], a1 = ev.a[1], a2 = ev.a[2], a3 = ev.a[3];
    const cx<T> b0 = ev.b[0], b1 = ev.b[1], b2 = ev.b[2], b3 = ev.b[3];
    // the e+ e- current and the mu+ mu- current vanish unless the two helicities of a line are opposite, and each is a
    // single chirality block:
    //   vbar(e+, h0) gamma^mu u(e-, h1):   h1 = +1: a = (-a0, -b0^*), psi_R = (a1, b1)       h1 = -1: b = (-b0, a0), psi_L = (-b1^*, a1)
    //   ubar(mu-, h3) gamma^mu v(mu+, h2): h3 = +1: a = (a3, b3^*),  psi_R = (-a2, -b2)      h3 = -1: b = (-b3, a3), psi_L = (-b2^*, a2)
    ev.JeR = cur_R<T>(cx<T>(-a0, (T)0), -conj_(b0), cx<T>(a1, (T)0), b1);
    ev.JeL = cur_L<T>(-b0, cx<T>(a0, (T)0), -conj_(b1), cx<T>(a1, (T)0));
    ev.JmR = cur_R<T>(cx<T>(a3, (T)0), conj_(b3), cx<T>(-a2, (T)0), -b2);
    ev.JmL = cur_L<T>(-b3, cx<T>(a3, (T)0), -conj_(b2), cx<T>(a2, (T)0));
    ev.qeR = mdot(ev.JeR, ev.q); ev.qeL = mdot(ev.JeL, ev.q); ev.qmR = mdot(ev.JmR, ev.q); ev.qmL = mdot(ev.JmL, ev.q);
  }

  // psibar gamma^mu psi of a massless line: only one chirality block of each spinor is non-zero, so the current is ONE of
  //   R:  J^mu = a sigma^mu psi_R        L:  J^mu = b sigmabar^mu psi_L        (helas.cuh ff_current, one half each)
  template <class T> static MG_HD Vec4<T> cur_R(cx<T> a0, cx<T> a1, cx<T> r0, cx<T> r1) {
    const cx<T> a0r0 = a0 * r0, a1r1 = a1 * r1, a0r1 = a0 * r1, a1r0 = a1 * r0;
    Vec4<T> J;
    J.v[0] = a0r0 + a1r1; J.v[3] = a0r0 - a1r1; J.v[1] = a0r1 + a1r0; J.v[2] = times_i(a1r0 - a0r1);
    return J;
  }
  template <class T> static MG_HD Vec4<T> cur_L(cx<T> b0, cx<T> b1, cx<T> l0, cx<T> l1) {
    const cx<T> b0l0 = b0 * l0, b1l1 = b1 * l1, b0l1 = b0 * l1, b1l0 = b1 * l0;
    Vec4<T> J;
    J.v[0] = b0l0 + b1l1; J.v[3] = b1l1 - b0l0; J.v[1] = -(b0l1 + b1l0); J.v[2] = times_i(b0l1 - b1l0);
    return J;
  }

  // |M|^2 of one helicity combination.  The helicity index is the same for every thread of the launch (the loop over the
  // good-helicity mask is uniform), so the selections below are uniform, not divergence.  With the
  // currents J_e, J_m of the combination and the chiral Z couplings g_e, g_m of their blocks:
  //   FFV1P0_3 + FFV1_0 :   amp_a = e^2 (J_e . J_m) / s
  //   FFV2_4_3 + FFV2_4_0:  amp_b = g_e g_m [ (J_e . J_m) - (J_e . q)(J_m . q)/mZ^2 ] / (s - mZ^2 + i mZ GZ)      (R13)
  template <class T> static MG_HD T helicity(const Event<T>& ev, int ihel, const Consts& k) {
    const bool h0 = (ihel & 1) != 0, h1 = (ihel & 2) != 0, h2 = (ihel & 4) != 0, h3 = (ihel & 8) != 0;
    if (h0 == h1 || h2 == h3) return (T)0;
    Vec4<T> Je, Jm;
    cx<T> jeq, jmq;
    if (per_event_currents<T>()) {
      // selected value by value: a reference into the event would force it into local memory
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        Je.v[i] = cx<T>(h1 ? ev.JeR.v[i].re : ev.JeL.v[i].re, h1 ? ev.JeR.v[i].im : ev.JeL.v[i].im);
        Jm.v[i] = cx<T>(h3 ? ev.JmR.v[i].re : ev.JmL.v[i].re, h3 ? ev.JmR.v[i].im : ev.JmL.v[i].im);
      }
      jeq = cx<T>(h1 ? ev.qeR.re : ev.qeL.re, h1 ? ev.qeR.im : ev.qeL.im);
      jmq = cx<T>(h3 ? ev.qmR.re : ev.qmL.re, h3 ? ev.qmR.im : ev.qmL.im);
    } else {
      const T a0 = ev.a[0], a1 = ev.a[1], a2 = ev.a[2], a3 = ev.a[3];
      const cx<T> b0 = ev.b[0], b1 = ev.b[1], b2 = ev.b[2], b3 = ev.b[3];
      if (h1) Je = cur_R<T>(cx<T>(-a0, (T)0), -conj_(b0), cx<T>(a1, (T)0), b1);
      else Je = cur_L<T>(-b0, cx<T>(a0, (T)0), -conj_(b1), cx<T>(a1, (T)0));
      if (h3) Jm = cur_R<T>(cx<T>(a3, (T)0), conj_(b3), cx<T>(-a2, (T)0), -b2);
      else Jm = cur_L<T>(-b3, cx<T>(a3, (T)0), -conj_(b2), cx<T>(a2, (T)0));
      jeq = mdot(Je, ev.q); jmq = mdot(Jm, ev.q);
    }
    const T ge = h1 ? (T)k.gzr : (T)k.gzl, gm = h3 ? (T)k.gzr : (T)k.gzl;
    const T e = (T)k.ee;
    const cx<T> jj = mdot(Je, Jm);
    const cx<T> zc = (ge * gm) * ev.bw;                                    // Z exchange: couplings x Breit-Wigner
    const cx<T> coef = cx<T>(fma_<T>(e * e, ev.is, zc.re), zc.im);          // photon + Z on the g^{mu nu} part
    const cx<T> amp = coef * jj - (zc * ((T)1 / (T)k.mZ2)) * (jeq * jmq);
    return norm2(amp);
  }
};

}  // namespace mg
