// ORACLE — test infrastructure only (see philox.hpp header).
//
// g g -> t t~ (+ g, + g g) at tree level, as the PLAIN DEFINITION
//     ME = (1/denom) sum_helicities sum_colours | sum of Feynman diagrams |^2 ,
// evaluated two ways that share only the Dirac algebra of dirac.hpp:
//   (1) qcd_me():       colour-ordered off-shell recursion  M = sum_sigma (T^{a_s1}...T^{a_sn})_ij A_sigma
//                       and the colour matrix C built by brute force from explicit Gell-Mann
//                       matrices;  ME = (1/denom) sum_hel A^dagger C A.
//   (2) qcd_me_dressed(): colour-DRESSED recursion with explicit f^{abc}, T^a and open colour
//                       indices, |M|^2 summed over every colour assignment (tiny inputs only).
// Neither needs a diagram list, so both are independent of the CUDA path's generator.
//
// Serves PAPER.md:29 and PAPER.md:35 (§2: amplitudes of all diagrams for one helicity combination
// are summed per colour flow into dual amplitudes; |M|^2 is a quadratic form with a constant
// colour matrix; sum over helicities, average) and PAPER.md:64 (§2, the gg -> t t~ (+g,+gg)
// processes).  The paper prints no Feynman rule; those used are the textbook QCD rules
// (after SURVEY.md Appendix A):
//   q q g: i gs gamma^mu T^a;   quark propagator i(q-slash + m)/(q^2 - m^2)   (Gamma_t = 0, R12);
//   g g g (all incoming): gs f^{abc}[g^{mu nu}(k1-k2)^rho + g^{nu rho}(k2-k3)^mu + g^{rho mu}(k3-k1)^nu];
//   g g g g: -i gs^2 [f^{abe}f^{cde}(g^{mu rho}g^{nu sigma} - g^{mu sigma}g^{nu rho}) + (2 more)];
//   gluon propagator -i g^{mu nu} delta^{ab}/k^2 (Feynman gauge).
// Colour-ordered rules implied by f^{abc}T^c = -i[T^a,T^b]: 3-vertex -i gs V3, 4-vertex
//   i gs^2 [2 g^{mu rho}g^{nu sigma} - g^{mu nu}g^{rho sigma} - g^{mu sigma}g^{nu rho}].
// Particle order (R9): 0,1 = beam gluons, 2 = t, 3 = t~, 4.. = final gluons.  All external
// particles have helicity +-1 (R10).  Helicity index: bit k = helicity of particle k (0 <-> -1).
// Colour-flow basis: permutations of the gluons (in particle order) in lexicographic order,
// strings ordered from the t end.
#pragma once
#include <algorithm>
#include <vector>
#include "common.hpp"
#include "dirac.hpp"

namespace oracle {

struct QcdProcess {
  int ng;            // number of gluons: 2, 3, 4
  int npar;          // ng + 2
  int gl[4];         // particle index of gluon g
  int it, itbar;     // particle index of t, t~
  int denom;         // 4 * 64 * (ng-2)!  (R11)
};
inline QcdProcess qcd_process(int ng) {
  QcdProcess P;
  P.ng = ng; P.npar = ng + 2; P.it = 2; P.itbar = 3;
  P.gl[0] = 0; P.gl[1] = 1; P.gl[2] = 4; P.gl[3] = 5;
  int fact = 1; for (int i = 2; i <= ng - 2; ++i) fact *= i;
  P.denom = 256 * fact;
  return P;
}
inline int factorial(int n) { int f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; }

// ---------------------------------------------------------------------------------------------
// Gell-Mann matrices, T^a = lambda^a/2, f^{abc} = -2i Tr([T^a,T^b]T^c).
// ---------------------------------------------------------------------------------------------
template <class T> struct Su3 {
  cx<T> Ta[8][3][3];
  T f[8][8][8];
  Su3() {
    const cx<T> I(0, 1);
    for (int a = 0; a < 8; ++a) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Ta[a][i][j] = 0;
    cx<T> l[8][3][3] = {};
    l[0][0][1] = 1; l[0][1][0] = 1;
    l[1][0][1] = -I; l[1][1][0] = I;
    l[2][0][0] = 1; l[2][1][1] = -1;
    l[3][0][2] = 1; l[3][2][0] = 1;
    l[4][0][2] = -I; l[4][2][0] = I;
    l[5][1][2] = 1; l[5][2][1] = 1;
    l[6][1][2] = -I; l[6][2][1] = I;
    T r3 = 1 / std::sqrt((T)3);
    l[7][0][0] = r3; l[7][1][1] = r3; l[7][2][2] = -2 * r3;
    for (int a = 0; a < 8; ++a) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Ta[a][i][j] = l[a][i][j] / (T)2;
    for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) {
      cx<T> tr = 0;
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k)
        tr += (Ta[a][i][j] * Ta[b][j][k] - Ta[b][i][j] * Ta[a][j][k]) * Ta[c][k][i];
      cx<T> v = cx<T>(0, -2) * tr;
      f[a][b][c] = (std::fabs(v.real()) < (T)1e-12) ? (T)0 : v.real();
    }
  }
};

// Colour matrix C_{sigma tau} = sum_{a_1..a_n, i, j} (T^{a_s1}...T^{a_sn})_{ij} conj((T^{a_t1}...T^{a_tn})_{ij}),
// brute force over all 8^n colour assignments.  out is nperm x nperm, row-major, real.
template <class T> void colour_matrix(int ng, std::vector<T>& out) {
  Su3<T> su3;
  int nperm = factorial(ng);
  std::vector<std::vector<int>> perms;
  std::vector<int> pr(ng);
  for (int i = 0; i < ng; ++i) pr[i] = i;
  do { perms.push_back(pr); } while (std::next_permutation(pr.begin(), pr.end()));
  std::vector<cx<T>> acc((size_t)nperm * nperm, cx<T>(0, 0));
  int ncol = 1; for (int i = 0; i < ng; ++i) ncol *= 8;
  std::vector<cx<T>> str((size_t)nperm * 9);
  for (int ca = 0; ca < ncol; ++ca) {
    int a[4]; int t = ca;
    for (int g = 0; g < ng; ++g) { a[g] = t % 8; t /= 8; }
    for (int s = 0; s < nperm; ++s) {
      cx<T> M[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
      for (int pos = 0; pos < ng; ++pos) {
        const auto& Tm = su3.Ta[a[perms[s][pos]]];
        cx<T> R[3][3] = {};
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k) R[i][j] += M[i][k] * Tm[k][j];
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) M[i][j] = R[i][j];
      }
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) str[(size_t)s * 9 + i * 3 + j] = M[i][j];
    }
    for (int s = 0; s < nperm; ++s) for (int u = 0; u < nperm; ++u) {
      cx<T> z = 0;
      for (int k = 0; k < 9; ++k) z += str[(size_t)s * 9 + k] * std::conj(str[(size_t)u * 9 + k]);
      acc[(size_t)s * nperm + u] += z;
    }
  }
  out.resize((size_t)nperm * nperm);
  for (size_t k = 0; k < out.size(); ++k) out[k] = acc[k].real();
}

// ---------------------------------------------------------------------------------------------
// Kinematic building blocks.
// ---------------------------------------------------------------------------------------------
// V3^{mu nu rho}(k1,k2,k3) J1_mu J2_nu = (J1.J2)(k1-k2)^rho + (J1.(k2-k3)) J2^rho + (J2.(k3-k1)) J1^rho
template <class T>
Vec4<T> v3_contract(const Vec4<T>& J1, const Vec4<T>& k1, const Vec4<T>& J2, const Vec4<T>& k2, const Vec4<T>& k3) {
  cx<T> j12 = mdot(J1, J2);
  cx<T> a = mdot(J1, vsub(k2, k3));
  cx<T> b = mdot(J2, vsub(k3, k1));
  Vec4<T> r;
  for (int mu = 0; mu < 4; ++mu) r.v[mu] = j12 * (k1.v[mu] - k2.v[mu]) + a * J2.v[mu] + b * J1.v[mu];
  return r;
}

template <class T> struct QcdExternal {
  Vec4<T> eps[4];   // per gluon: eps (incoming) or eps* (outgoing)
  Vec4<T> kin[4];   // per gluon: incoming momentum (+p beams, -p final)
  Row4<T> ubar_t;   // outgoing top
  Col4<T> v_tbar;   // outgoing anti-top
  Vec4<T> pt;       // top momentum (real)
};

// External wavefunctions for helicity combination ihel.  gauge_gluon >= 0 replaces that gluon's
// polarisation by its momentum divided by its energy (gauge-invariance probe).
template <class T>
QcdExternal<T> qcd_external(const QcdProcess& P, const Params& par, const T (*p)[4], int ihel, int gauge_gluon = -1) {
  QcdExternal<T> X;
  T mt = (T)par.mt;
  for (int g = 0; g < P.ng; ++g) {
    int ip = P.gl[g];
    int h = ((ihel >> ip) & 1) ? +1 : -1;
    bool incoming = (ip < 2);
    Vec4<T> e = polvec<T>(p[ip], h);
    X.eps[g] = incoming ? e : vconj(e);
    X.kin[g] = real_vec<T>(p[ip], incoming ? (T)1 : (T)-1);
    if (g == gauge_gluon) X.eps[g] = vscale(real_vec<T>(p[ip]), cx<T>(1 / p[ip][0], 0));
  }
  int ht = ((ihel >> P.it) & 1) ? +1 : -1;
  int htb = ((ihel >> P.itbar) & 1) ? +1 : -1;
  X.ubar_t = bar(spinor_u<T>(p[P.it], mt, ht));
  X.v_tbar = spinor_v<T>(p[P.itbar], mt, htb);
  X.pt = real_vec<T>(p[P.it]);
  return X;
}

// Colour-ordered partial amplitude A_sigma for the ordered gluon list ord[0..ng-1] (from the t end).
//   J(i..j)^rho = (-i/K^2)[ sum_l (-i gs) V3(K_A,K_B,-K) J_A J_B
//                          + sum_{l<m} (i gs^2)(2 (J_A.J_C) J_B - (J_A.J_B) J_C - (J_B.J_C) J_A) ]
//   psibar(m)  = sum_{l<m} psibar(l) (i gs slash(J(l+1..m))) i(qslash_m + mt)/(q_m^2 - mt^2),
//                q_m = p_t - sum_{k<=m} k_k,   psibar(0) = ubar(p_t)
//   A_sigma    = [ sum_{l<n} psibar(l) (i gs slash(J(l+1..n))) ] v(p_tbar)
template <class T>
cx<T> ordered_amplitude(const QcdProcess& P, const Params& par, const QcdExternal<T>& X, const int* ord) {
  const cx<T> I(0, 1);
  const int n = P.ng;
  const T gs = std::sqrt(4 * pi_v<T>() * (T)par.alpha_s);
  const T mt = (T)par.mt;
  Vec4<T> J[4][4], K[4][4];
  for (int i = 0; i < n; ++i) { J[i][i] = X.eps[ord[i]]; K[i][i] = X.kin[ord[i]]; }
  for (int len = 2; len <= n; ++len)
    for (int i = 0; i + len - 1 < n; ++i) {
      int j = i + len - 1;
      K[i][j] = vadd(K[i][j - 1], K[j][j]);
      Vec4<T> Kout = vscale(K[i][j], cx<T>(-1, 0));
      Vec4<T> acc{};
      for (int l = i; l < j; ++l) {  // A = (i..l), B = (l+1..j)
        Vec4<T> t = v3_contract<T>(J[i][l], K[i][l], J[l + 1][j], K[l + 1][j], Kout);
        acc = vadd(acc, vscale(t, -I * gs));
      }
      for (int l = i; l < j; ++l)
        for (int m = l + 1; m < j; ++m) {  // A = (i..l), B = (l+1..m), C = (m+1..j)
          const Vec4<T>&A = J[i][l], &B = J[l + 1][m], &C = J[m + 1][j];
          cx<T> ac = mdot(A, C), ab = mdot(A, B), bc = mdot(B, C);
          Vec4<T> t;
          for (int mu = 0; mu < 4; ++mu) t.v[mu] = cx<T>(2, 0) * ac * B.v[mu] - ab * C.v[mu] - bc * A.v[mu];
          acc = vadd(acc, vscale(t, I * gs * gs));
        }
      J[i][j] = vscale(acc, -I / mdot(K[i][j], K[i][j]));
    }
  // quark line from the t end
  Row4<T> psib[5];
  psib[0] = X.ubar_t;
  Vec4<T> q = X.pt;
  for (int m = 1; m <= n - 1; ++m) {  // psibar after absorbing positions 0..m-1
    q = vsub(q, X.kin[ord[m - 1]]);
    Row4<T> acc{};
    for (int l = 0; l < m; ++l) {  // psibar(l) absorbs J(l..m-1)
      Row4<T> t = mul(psib[l], mscale(slash(J[l][m - 1]), I * gs));
      for (int c = 0; c < 4; ++c) acc.r[c] += t.r[c];
    }
    Mat4<T> prop = mscale(madd(slash(q), mscale(identity4<T>(), cx<T>(mt, 0))), I / (mdot(q, q) - mt * mt));
    psib[m] = mul(acc, prop);
  }
  cx<T> A = 0;
  for (int l = 0; l < n; ++l) A += mul(mul(psib[l], mscale(slash(J[l][n - 1]), I * gs)), X.v_tbar);
  return A;
}

template <class T> std::vector<std::vector<int>> qcd_perms(int ng) {
  std::vector<std::vector<int>> perms;
  std::vector<int> pr(ng);
  for (int i = 0; i < ng; ++i) pr[i] = i;
  do { perms.push_back(pr); } while (std::next_permutation(pr.begin(), pr.end()));
  return perms;
}

// All partial amplitudes of one helicity combination (lexicographic permutation order).
template <class T>
void qcd_partial_amplitudes(const QcdProcess& P, const Params& par, const T (*p)[4], int ihel,
                            std::vector<cx<T>>& A, int gauge_gluon = -1) {
  auto perms = qcd_perms<T>(P.ng);
  QcdExternal<T> X = qcd_external<T>(P, par, p, ihel, gauge_gluon);
  A.resize(perms.size());
  for (size_t s = 0; s < perms.size(); ++s) A[s] = ordered_amplitude<T>(P, par, X, perms[s].data());
}

// ME = (1/denom) sum_hel A^dagger C A.  C: nperm x nperm colour matrix (colour_matrix()).
// hel_out[2^npar] optional: |M|^2 of each helicity combination (before the 1/denom).
template <class T>
T qcd_me(const QcdProcess& P, const Params& par, const std::vector<T>& C, const T (*p)[4], T* hel_out = nullptr) {
  int nhel = 1 << P.npar;
  int nperm = factorial(P.ng);
  T sum = 0;
  std::vector<cx<T>> A;
  for (int ihel = 0; ihel < nhel; ++ihel) {
    qcd_partial_amplitudes<T>(P, par, p, ihel, A);
    T m2 = 0;
    for (int s = 0; s < nperm; ++s)
      for (int u = 0; u < nperm; ++u) m2 += (std::conj(A[s]) * C[(size_t)s * nperm + u] * A[u]).real();
    if (hel_out) hel_out[ihel] = m2;
    sum += m2;
  }
  return sum / (T)P.denom;
}

// ---------------------------------------------------------------------------------------------
// Colour-dressed brute force: full amplitude M_{ij}(a_1..a_n) from explicit f^{abc}, T^a.
// Gluon currents J_S^{rho,c} for every subset S (bitmask) of the gluons, open colour c:
//   J_S^c = (-i/K_S^2)[ sum_{unordered {A,B}} sum_{cA,cB} gs f^{cA cB c} V3(K_A,K_B,-K_S) J_A^{cA} J_B^{cB}
//                     + sum_{unordered {A,B,C}} sum_{cA,cB,cC} (-i gs^2)( f^{cA cB e}f^{cC c e}[(A.C)B - (B.C)A]
//                         + f^{cA cC e}f^{cB c e}[(A.B)C - (B.C)A] + f^{cA c e}f^{cB cC e}[(A.B)C - (A.C)B] ) ]
// Quark line (row spinor x colour row), subset S absorbed, t colour i:
//   Psi_S = sum_{A subset S, A != 0} Psi_{S\A} (i gs slash(J_A^c) T^c) i(qslash_S + mt)/(q_S^2 - mt^2)
//   M_ij  = [ sum_{A != 0} Psi_{all\A} (i gs slash(J_A^c) T^c) ]_j v
// ---------------------------------------------------------------------------------------------
template <class T>
T qcd_me_dressed(const QcdProcess& P, const Params& par, const T (*p)[4]) {
  const cx<T> I(0, 1);
  Su3<T> su3;
  const int n = P.ng, full = (1 << n) - 1;
  const T gs = std::sqrt(4 * pi_v<T>() * (T)par.alpha_s);
  const T mt = (T)par.mt;
  int nhel = 1 << P.npar;
  int ncol = 1; for (int i = 0; i < n; ++i) ncol *= 8;
  T total = 0;
  for (int ihel = 0; ihel < nhel; ++ihel) {
    QcdExternal<T> X = qcd_external<T>(P, par, p, ihel);
    Vec4<T> K[16];
    for (int S = 1; S <= full; ++S) {
      Vec4<T> k{};
      for (int g = 0; g < n; ++g) if (S & (1 << g)) k = vadd(k, X.kin[g]);
      K[S] = k;
    }
    for (int ca = 0; ca < ncol; ++ca) {
      int a[4]; int t = ca;
      for (int g = 0; g < n; ++g) { a[g] = t % 8; t /= 8; }
      // gluon currents
      std::vector<Vec4<T>> J((size_t)16 * 8);
      std::vector<char> nz((size_t)16 * 8, 0);
      for (int S = 1; S <= full; ++S) {
        int pc = __builtin_popcount(S);
        if (pc == 1) {
          int g = __builtin_ctz(S);
          for (int c = 0; c < 8; ++c) { J[S * 8 + c] = Vec4<T>{}; }
          J[S * 8 + a[g]] = X.eps[g]; nz[S * 8 + a[g]] = 1;
          continue;
        }
        Vec4<T> Kout = vscale(K[S], cx<T>(-1, 0));
        Vec4<T> acc[8] = {};
        // unordered 2-splits: A contains the lowest bit of S
        int low = S & (-S);
        for (int A = (S - 1) & S; A > 0; A = (A - 1) & S) {
          if (!(A & low)) continue;
          int B = S ^ A;
          if (B == 0) continue;
          for (int cA = 0; cA < 8; ++cA) {
            if (!nz[A * 8 + cA]) continue;
            for (int cB = 0; cB < 8; ++cB) {
              if (!nz[B * 8 + cB]) continue;
              Vec4<T> v = v3_contract<T>(J[A * 8 + cA], K[A], J[B * 8 + cB], K[B], Kout);
              for (int c = 0; c < 8; ++c) {
                T ff = su3.f[cA][cB][c];
                if (ff == 0) continue;
                acc[c] = vadd(acc[c], vscale(v, cx<T>(gs * ff, 0)));
              }
            }
          }
        }
        // unordered 3-splits: A contains the lowest bit; B contains the lowest bit of the rest
        for (int A = (S - 1) & S; A > 0; A = (A - 1) & S) {
          if (!(A & low)) continue;
          int R = S ^ A;
          if (R == 0) continue;
          int lowR = R & (-R);
          for (int B = (R - 1) & R; B > 0; B = (B - 1) & R) {
            if (!(B & lowR)) continue;
            int Cc = R ^ B;
            if (Cc == 0) continue;
            for (int cA = 0; cA < 8; ++cA) { if (!nz[A * 8 + cA]) continue;
              for (int cB = 0; cB < 8; ++cB) { if (!nz[B * 8 + cB]) continue;
                for (int cC = 0; cC < 8; ++cC) { if (!nz[Cc * 8 + cC]) continue;
                  const Vec4<T>&JA = J[A * 8 + cA], &JB = J[B * 8 + cB], &JC = J[Cc * 8 + cC];
                  cx<T> ab = mdot(JA, JB), ac = mdot(JA, JC), bc = mdot(JB, JC);
                  Vec4<T> s1, s2, s3;
                  for (int mu = 0; mu < 4; ++mu) {
                    s1.v[mu] = ac * JB.v[mu] - bc * JA.v[mu];
                    s2.v[mu] = ab * JC.v[mu] - bc * JA.v[mu];
                    s3.v[mu] = ab * JC.v[mu] - ac * JB.v[mu];
                  }
                  for (int c = 0; c < 8; ++c) {
                    T f1 = 0, f2 = 0, f3 = 0;
                    for (int e = 0; e < 8; ++e) {
                      f1 += su3.f[cA][cB][e] * su3.f[cC][c][e];
                      f2 += su3.f[cA][cC][e] * su3.f[cB][c][e];
                      f3 += su3.f[cA][c][e] * su3.f[cB][cC][e];
                    }
                    if (f1 == 0 && f2 == 0 && f3 == 0) continue;
                    Vec4<T> v;
                    for (int mu = 0; mu < 4; ++mu) v.v[mu] = f1 * s1.v[mu] + f2 * s2.v[mu] + f3 * s3.v[mu];
                    acc[c] = vadd(acc[c], vscale(v, -I * gs * gs));
                  }
                } } }
          }
        }
        cx<T> prop = -I / mdot(K[S], K[S]);
        for (int c = 0; c < 8; ++c) {
          J[S * 8 + c] = vscale(acc[c], prop);
          bool any = false;
          for (int mu = 0; mu < 4; ++mu) any = any || (J[S * 8 + c].v[mu] != cx<T>(0, 0));
          nz[S * 8 + c] = any ? 1 : 0;
        }
      }
      // quark line, for each top colour i
      for (int i = 0; i < 3; ++i) {
        Row4<T> Psi[16][3];
        for (int S = 0; S <= full; ++S) for (int j = 0; j < 3; ++j) Psi[S][j] = Row4<T>{};
        Psi[0][i] = X.ubar_t;
        cx<T> Mj[3] = {0, 0, 0};
        for (int S = 1; S <= full; ++S) {
          Row4<T> acc[3] = {};
          for (int A = S; A > 0; A = (A - 1) & S) {
            int Rm = S ^ A;
            for (int c = 0; c < 8; ++c) {
              if (!nz[A * 8 + c]) continue;
              Mat4<T> V = mscale(slash(J[A * 8 + c]), I * gs);
              for (int j1 = 0; j1 < 3; ++j1) {
                Row4<T> t = mul(Psi[Rm][j1], V);
                for (int j2 = 0; j2 < 3; ++j2) {
                  cx<T> tc = su3.Ta[c][j1][j2];
                  if (tc == cx<T>(0, 0)) continue;
                  for (int d = 0; d < 4; ++d) acc[j2].r[d] += t.r[d] * tc;
                }
              }
            }
          }
          if (S == full) {
            for (int j = 0; j < 3; ++j) Mj[j] = mul(acc[j], X.v_tbar);
          } else {
            Vec4<T> q = vsub(X.pt, K[S]);
            Mat4<T> prop = mscale(madd(slash(q), mscale(identity4<T>(), cx<T>(mt, 0))), I / (mdot(q, q) - mt * mt));
            for (int j = 0; j < 3; ++j) Psi[S][j] = mul(acc[j], prop);
          }
        }
        for (int j = 0; j < 3; ++j) total += std::norm(Mj[j]);
      }
    }
  }
  return total / (T)P.denom;
}

}  // namespace oracle
