// ORACLE — test infrastructure only (see philox.hpp header).
// Shared scalar helpers of the oracle: pi and the physics-parameter record (BASELINE.json configs).
#pragma once

namespace oracle {

template <class T> inline T pi_v() { return (T)3.14159265358979323846264338327950288419716939937510L; }

// sqrt_s [GeV]; 1/alpha_EM, mZ, GammaZ, mW (e+e- -> mu+mu-); mt, alpha_s (gg -> t t~ + gluons).
struct Params {
  double sqrt_s, alpha_em_inv, mZ, gammaZ, mW, mt, alpha_s;
};

}  // namespace oracle
