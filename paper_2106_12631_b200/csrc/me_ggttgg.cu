// me_ggttgg.cu — launcher of the generated g g -> t t~ g g sigmaKin kernel: helicity recycling in shared
// memory (recycle.cuh + gen_rc_ggttgg.cuh, written by gen/recycle.py).
#include "gen_rc_ggttgg.cuh"

namespace mg {

cudaError_t launch_me_ggttgg(const mg_process* p, const MeArgs& a, cudaStream_t s) { return rc::launch_sigmakin_recycle<RcGgttgg>(p, a, s); }

}  // namespace mg
