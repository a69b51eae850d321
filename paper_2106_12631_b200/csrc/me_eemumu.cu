// me_eemumu.cu — launcher of the e+ e- -> mu+ mu- sigmaKin kernel (eemumu.cuh holds the physics).
#include "me_common.cuh"
#include "eemumu.cuh"

namespace mg {

cudaError_t launch_me_eemumu(const mg_process* p, const MeArgs& a, cudaStream_t s) { return launch_sigmakin<Eemumu>(p, a, s); }

}  // namespace mg
