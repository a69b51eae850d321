// me_ggttg.cu — launcher of the generated g g -> t t~ g sigmaKin kernel: helicity recycling in shared memory
// (recycle.cuh + gen_rc_ggttg.cuh, written by gen/recycle.py): a third of the arithmetic of the one-thread-per-event
// kernel (gen_ggttg.cuh, kept for comparison through MG_GGTTG_THREAD_PER_EVENT at build time).
#ifdef MG_GGTTG_THREAD_PER_EVENT
#include "me_common.cuh"
#include "gen_ggttg.cuh"
namespace mg {
cudaError_t launch_me_ggttg(const mg_process* p, const MeArgs& a, cudaStream_t s) { return launch_sigmakin<Ggttg>(p, a, s); }
}  // namespace mg
#else
#include "gen_rc_ggttg.cuh"
namespace mg {
cudaError_t launch_me_ggttg(const mg_process* p, const MeArgs& a, cudaStream_t s) { return rc::launch_sigmakin_recycle<RcGgttg>(p, a, s); }
}  // namespace mg
#endif
