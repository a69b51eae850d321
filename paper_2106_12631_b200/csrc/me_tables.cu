// me_tables.cu — generated tables (flop tallies, colour matrices) behind mg_flops_per_event / mg_colour_matrix.
#include "mg_internal.h"
#include "gen_tables.cuh"
#include "gen_rc_tables.cuh"
#include "gen_qq_tables.cuh"

namespace mg {

// e+ e- -> mu+ mu-: hand tally of eemumu.cuh.  The two single-chirality currents of a
// helicity combination (4 complex products + 4 complex sums = 32 each) and their contractions with q (14 each) are inside
// the helicity loop in FP64 and per event (four currents, four contractions) in FP32 (eemumu.cuh per_event_currents).
// Per NON-VANISHING helicity combination besides: J_e.J_m (30), the photon + Z coefficient (2 + 3 + 1), the two terms of the
// amplitude (6 + 2 + 6 + 6 + 2), the square (3).  Per event: s, 1/s, Breit-Wigner (20) and 4 massless spinor frames
// (pT^2 3, P 4, P+pz 2, rsqrt 2, 3 products = 14 each).
static const int kFlopsPerHelicity_ee = 30 + 6 + 22 + 3;
static const int kFlopsCurrents_ee = 2 * 32 + 2 * 14;      // one pair of currents with their q contractions
static const int kFlopsFixed_ee = 4 + 7 + 1 + 1 + 4 + 3 + 4 * 14;

int64_t me_flops_per_helicity(int process, bool fp64) {
  switch (process) {
    case MG_EEMUMU: return kFlopsPerHelicity_ee + (fp64 ? kFlopsCurrents_ee : 0);
    case MG_GGTT: return kFlopsPerHelicity_2;
    case MG_GGTTG: return kFlopsPerHelicity_3;
    case MG_GGTTGG: return kFlopsPerHelicity_4;
    case MG_QQTT: return kFlopsPerHelicity_qq0;
    case MG_QQTTG: return kFlopsPerHelicity_qq1;
  }
  return 0;
}
int64_t me_flops_per_event_fixed(int process, bool fp64) {
  switch (process) {
    case MG_EEMUMU: return kFlopsFixed_ee + (fp64 ? 0 : 2 * kFlopsCurrents_ee);
    case MG_GGTT: return kFlopsFixed_2;
    case MG_GGTTG: return kFlopsFixed_3;
    case MG_GGTTGG: return kFlopsFixed_4;
    case MG_QQTT: return kFlopsFixed_qq0;
    case MG_QQTTG: return kFlopsFixed_qq1;
  }
  return 0;
}
// processes evaluated by the helicity-recycling kernel (recycle.cuh): the tally of everything that kernel
// executes per event (all helicity variants of every shared wavefunction); -1: per-helicity tally applies
int64_t me_flops_per_event_recycle(int process, bool fp64) {
  switch (process) {
    case MG_GGTTGG: return fp64 ? kFlopsRecycleFp64_4 : kFlopsRecycle_4;
    case MG_GGTTG: return fp64 ? kFlopsRecycleFp64_3 : kFlopsRecycle_3;
  }
  return -1;
}
const int* me_colour_numerators(int process, int* den) {
  switch (process) {
    case MG_GGTT: *den = kColourDen_2; return kColourNum_2;
    case MG_GGTTG: *den = kColourDen_3; return kColourNum_3;
    case MG_GGTTGG: *den = kColourDen_4; return kColourNum_4;
    case MG_QQTT: *den = kColourDen_qq0; return kColourNum_qq0;
    case MG_QQTTG: *den = kColourDen_qq1; return kColourNum_qq1;
  }
  return nullptr;
}

}  // namespace mg
