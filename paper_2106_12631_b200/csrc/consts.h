// consts.h — derived physics constants handed to every kernel by value.
#pragma once
namespace mg {

// Derived physics constants, computed once on the host in double precision (constant
// parameters).  Passed to kernels by value (kernel arguments live in the constant bank).
struct Consts {
  double sqrt_s;
  double mass[4];      // final-state masses (R7)
  double w0;           // massless RAMBO weight (north_star closed form)
  // e+e- -> mu+mu- (R13-R15)
  double ee;           // e = sqrt(4 pi alpha)
  double gzl, gzr;     // Z couplings e/(sW cW) * gL, gR
  double mZ, mZ2, mZgZ;
  // QCD (R12, R15)
  double gs;           // sqrt(4 pi alpha_s)
  double mt;
  double me_norm;      // overall factor applied once per event: coupling powers / denominator
};

}  // namespace mg
