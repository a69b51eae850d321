// me_ggttg.cu — launcher of the generated g g -> t t~ g sigmaKin kernel: helicity recycling in shared memory
// (recycle.cuh + gen_rc_ggttg.cuh, written by gen/recycle.py).
#include "gen_rc_ggttg.cuh"
namespace mg {
cudaError_t launch_me_ggttg(const mg_process* p, const MeArgs& a, cudaStream_t s) { return rc::launch_sigmakin_recycle<RcGgttg>(p, a, s); }
}  // namespace mg
