// me_ggttgg.cu — launcher of the generated g g -> t t~ g g sigmaKin kernel (gen_ggttgg.cuh, written by gen/qcdgen.py).
#include "me_common.cuh"
#include "gen_ggttgg.cuh"

namespace mg {

cudaError_t launch_me_ggttgg(const mg_process* p, const MeArgs& a, cudaStream_t s) { return launch_sigmakin<Ggttgg>(p, a, s); }

}  // namespace mg
