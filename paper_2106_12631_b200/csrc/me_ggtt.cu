// me_ggtt.cu — launcher of the generated g g -> t t~ sigmaKin kernel (gen_ggtt.cuh, written by gen/qcdgen.py).
#include "me_common.cuh"
#include "gen_ggtt.cuh"

namespace mg {

cudaError_t launch_me_ggtt(const mg_process* p, const MeArgs& a, cudaStream_t s) { return launch_sigmakin<Ggtt>(p, a, s); }

}  // namespace mg
