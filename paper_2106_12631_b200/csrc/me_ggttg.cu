// me_ggttg.cu — launcher of the generated g g -> t t~ g sigmaKin kernel (gen_ggttg.cuh, written by gen/qcdgen.py).
#include "me_common.cuh"
#include "gen_ggttg.cuh"

namespace mg {

cudaError_t launch_me_ggttg(const mg_process* p, const MeArgs& a, cudaStream_t s) { return launch_sigmakin<Ggttg>(p, a, s); }

}  // namespace mg
