// me_eemumu.cu — launcher of the e+ e- -> mu+ mu- sigmaKin kernel (eemumu.cuh holds the physics).
#include "me_common.cuh"
#include "eemumu.cuh"
#include "fused.cuh"

namespace mg {

cudaError_t launch_me_eemumu(const mg_process* p, const MeArgs& a, cudaStream_t s) { return launch_sigmakin<Eemumu>(p, a, s); }

cudaError_t launch_fused_eemumu(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s) {
  return launch_fused<Eemumu, 2, false>(p, seed, first, n, me, psw, evw, s);
}

}  // namespace mg
