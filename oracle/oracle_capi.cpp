// ORACLE — test infrastructure only (see philox.hpp header).
//
// Plain C entry points over the oracle templates so that tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs can call it through ctypes.  Event-major (AoS)
// arrays throughout: rho[n][n_final][4], mom[n][npar][4].  Nothing here is used by the product.
//
// process ids: 0 = e+e- -> mu+mu-, 1 = gg -> tt~, 2 = gg -> tt~g, 3 = gg -> tt~gg, 4 = u u~ -> t t~, 5 = u u~ -> t t~ g.
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>
#include "philox.hpp"
#include "rambo.hpp"
#include "me_eemumu.hpp"
#include "me_qcd.hpp"
#include "me_qq.hpp"

using namespace oracle;

namespace {

int n_final_of(int process) { return process <= 1 ? 2 : (process <= 3 ? process + 1 : process - 2); }    // 2,2,3,4,2,3
int n_par_of(int process) { return n_final_of(process) + 2; }
void masses_of(int process, const Params& par, double* m) {
  int nf = n_final_of(process);
  for (int i = 0; i < nf; ++i) m[i] = 0;
  if (process >= 1) { m[0] = par.mt; m[1] = par.mt; }
}

template <class T>
void me_batch(int process, const Params& par, const double* mom, int64_t n, double* me_out, double* hel_out,
              int64_t lo, int64_t hi) {
  int np = n_par_of(process);
  int nhel = 1 << np;
  std::vector<T> C;
  QcdProcess P{};
  if (process >= 1 && process <= 3) { P = qcd_process(process + 1); colour_matrix<T>(P.ng, C); }
  std::vector<T> hel(nhel);
  for (int64_t e = lo; e < hi; ++e) {
    T p[6][4];
    for (int i = 0; i < np; ++i) for (int mu = 0; mu < 4; ++mu) p[i][mu] = (T)mom[(e * np + i) * 4 + mu];
    T me;
    if (process == 0) me = eemumu_me<T>(par, p, hel.data());
    else if (process >= 4) me = qq_me<T>(process - 4, par, p, hel.data());
    else me = qcd_me<T>(P, par, C, p, hel.data());
    me_out[e] = (double)me;
    if (hel_out) for (int h = 0; h < nhel; ++h) hel_out[e * nhel + h] = (double)hel[h];
  }
  (void)n;
}

template <class F> void run_threads(int64_t n, int nthreads, F f) {
  if (nthreads <= 1 || n < 2) { f(0, n); return; }
  std::vector<std::thread> th;
  int64_t chunk = (n + nthreads - 1) / nthreads;
  for (int t = 0; t < nthreads; ++t) {
    int64_t lo = t * chunk, hi = std::min<int64_t>(n, lo + chunk);
    if (lo >= hi) break;
    th.emplace_back([=] { f(lo, hi); });
  }
  for (auto& t : th) t.join();
}

}  // namespace

extern "C" {

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

// words[n][n_final][4]
void oracle_rng_words(uint64_t seed, uint64_t first_event, int64_t n, int n_final, uint32_t* words) {
  for (int64_t e = 0; e < n; ++e)
    for (int i = 0; i < n_final; ++i) philox_event_particle(seed, first_event + (uint64_t)e, (uint32_t)i, words + (e * n_final + i) * 4);
}
void oracle_uniforms_f64(uint64_t seed, uint64_t first_event, int64_t n, int n_final, double* rho) {
  for (int64_t e = 0; e < n; ++e)
    for (int i = 0; i < n_final; ++i) {
      uint32_t w[4]; philox_event_particle(seed, first_event + (uint64_t)e, (uint32_t)i, w);
      for (int k = 0; k < 4; ++k) rho[(e * n_final + i) * 4 + k] = u32_to_uniform_f64(w[k]);
    }
}
void oracle_uniforms_f32(uint64_t seed, uint64_t first_event, int64_t n, int n_final, float* rho) {
  for (int64_t e = 0; e < n; ++e)
    for (int i = 0; i < n_final; ++i) {
      uint32_t w[4]; philox_event_particle(seed, first_event + (uint64_t)e, (uint32_t)i, w);
      for (int k = 0; k < 4; ++k) rho[(e * n_final + i) * 4 + k] = u32_to_uniform_f32(w[k]);
    }
}

double oracle_rambo_w0(int n_final, double sqrt_s) { return rambo_w0<double>(n_final, sqrt_s); }

// rho[n][n_final][4] -> mom[n][2+n_final][4], weight[n], xi[n] (nullable).  use_ld: long double arithmetic.
void oracle_rambo(int n_final, const double* masses, double sqrt_s, const double* rho, int64_t n,
                  double* mom, double* weight, double* xi, int use_ld) {
  int np = n_final + 2;
  for (int64_t e = 0; e < n; ++e) {
    if (use_ld) {
      long double r[16], m[4], p[6][4], x;
      for (int k = 0; k < 4 * n_final; ++k) r[k] = rho[e * 4 * n_final + k];
      for (int k = 0; k < n_final; ++k) m[k] = masses[k];
      long double w = rambo_event<long double>(n_final, r, m, (long double)sqrt_s, p, 1e-17L, &x);
      for (int i = 0; i < np; ++i) for (int mu = 0; mu < 4; ++mu) mom[(e * np + i) * 4 + mu] = (double)p[i][mu];
      weight[e] = (double)w; if (xi) xi[e] = (double)x;
    } else {
      double p[6][4], x;
      double w = rambo_event<double>(n_final, rho + e * 4 * n_final, masses, sqrt_s, p, 1e-14, &x);
      for (int i = 0; i < np; ++i) for (int mu = 0; mu < 4; ++mu) mom[(e * np + i) * 4 + mu] = p[i][mu];
      weight[e] = w; if (xi) xi[e] = x;
    }
  }
}

// mom[n][npar][4] -> me[n]; hel_out[n][2^npar] nullable.
void oracle_me(int process, const Params* par, const double* mom, int64_t n, double* me_out, double* hel_out,
               int use_ld, int nthreads) {
  run_threads(n, nthreads, [=](int64_t lo, int64_t hi) {
    if (use_ld) me_batch<long double>(process, *par, mom, n, me_out, hel_out, lo, hi);
    else me_batch<double>(process, *par, mom, n, me_out, hel_out, lo, hi);
  });
}

// Colour-dressed brute force (processes 1..3), tiny n only.
void oracle_me_dressed(int process, const Params* par, const double* mom, int64_t n, double* me_out, int nthreads) {
  QcdProcess P = qcd_process(process + 1);
  int np = P.npar;
  run_threads(n, nthreads, [=](int64_t lo, int64_t hi) {
    for (int64_t e = lo; e < hi; ++e) {
      double p[6][4];
      for (int i = 0; i < np; ++i) for (int mu = 0; mu < 4; ++mu) p[i][mu] = mom[(e * np + i) * 4 + mu];
      me_out[e] = qcd_me_dressed<double>(P, *par, p);
    }
  });
}

// out[nperm*nperm], row-major, lexicographic permutation order.
void oracle_colour_matrix(int ng, double* out) {
  std::vector<double> C; colour_matrix<double>(ng, C);
  std::memcpy(out, C.data(), C.size() * sizeof(double));
}

// Partial amplitudes A_sigma (re,im interleaved, nperm of them) of one event and helicity combination;
// gauge_gluon >= 0 replaces that gluon's polarisation by p/E.
void oracle_partial_amplitudes(int process, const Params* par, const double* mom, int ihel, int gauge_gluon, double* out, int use_ld) {
  QcdProcess P = qcd_process(process + 1);
  if (use_ld) {
    long double p[6][4];
    for (int i = 0; i < P.npar; ++i) for (int mu = 0; mu < 4; ++mu) p[i][mu] = mom[i * 4 + mu];
    std::vector<cx<long double>> A; qcd_partial_amplitudes<long double>(P, *par, p, ihel, A, gauge_gluon);
    for (size_t s = 0; s < A.size(); ++s) { out[2 * s] = (double)A[s].real(); out[2 * s + 1] = (double)A[s].imag(); }
  } else {
    double p[6][4];
    for (int i = 0; i < P.npar; ++i) for (int mu = 0; mu < 4; ++mu) p[i][mu] = mom[i * 4 + mu];
    std::vector<cx<double>> A; qcd_partial_amplitudes<double>(P, *par, p, ihel, A, gauge_gluon);
    for (size_t s = 0; s < A.size(); ++s) { out[2 * s] = A[s].real(); out[2 * s + 1] = A[s].imag(); }
  }
}

// Whole path for events [first_event, first_event+n): Philox -> uniforms -> RAMBO -> ME, FP64.
// me[n], weight[n]; mom (nullable) [n][npar][4].  Used for the timed CPU baseline.
void oracle_pipeline(int process, const Params* par, uint64_t seed, uint64_t first_event, int64_t n,
                     double* me_out, double* weight, double* mom_out, int nthreads) {
  int nf = n_final_of(process), np = nf + 2;
  run_threads(n, nthreads, [=](int64_t lo, int64_t hi) {
    std::vector<double> C;
    QcdProcess P{};
    if (process >= 1 && process <= 3) { P = qcd_process(process + 1); colour_matrix<double>(P.ng, C); }
    double masses[4]; masses_of(process, *par, masses);
    for (int64_t e = lo; e < hi; ++e) {
      double rho[16], p[6][4];
      for (int i = 0; i < nf; ++i) {
        uint32_t w[4]; philox_event_particle(seed, first_event + (uint64_t)e, (uint32_t)i, w);
        for (int k = 0; k < 4; ++k) rho[4 * i + k] = u32_to_uniform_f64(w[k]);
      }
      weight[e] = rambo_event<double>(nf, rho, masses, par->sqrt_s, p, 1e-14);
      if (mom_out) for (int i = 0; i < np; ++i) for (int mu = 0; mu < 4; ++mu) mom_out[(e * np + i) * 4 + mu] = p[i][mu];
      me_out[e] = (process == 0) ? eemumu_me<double>(*par, p) : (process >= 4 ? qq_me<double>(process - 4, *par, p) : qcd_me<double>(P, *par, C, p));
    }
  });
}

// u u~ -> t t~ g with the gluon polarisation replaced by its momentum / energy: largest |M| over colour assignments and
// helicities (out[0]) next to the same with the physical polarisations (out[1])  -- gauge-invariance pin
void oracle_qq_gauge(const Params* par, const double* mom, double* out) {
  double p[5][4];
  for (int i = 0; i < 5; ++i) for (int mu = 0; mu < 4; ++mu) p[i][mu] = mom[i * 4 + mu];
  qq_me<double>(1, *par, p, nullptr, true, &out[0]);
  qq_me<double>(1, *par, p, nullptr, false, &out[1]);
}

int oracle_hardware_threads() { return (int)std::thread::hardware_concurrency(); }

}  // extern "C"
