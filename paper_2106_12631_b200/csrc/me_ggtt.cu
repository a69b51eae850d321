// me_ggtt.cu — launcher of the generated g g -> t t~ sigmaKin kernel.  Default: one thread per event
// (gen_ggtt.cuh, written by gen/qcdgen.py); MG_GGTT_RECYCLE at build time selects the helicity-recycling
// kernel (recycle.cuh + gen_rc_ggtt.cuh) for comparison.
#ifdef MG_GGTT_RECYCLE
#include "gen_rc_ggtt.cuh"
namespace mg {
cudaError_t launch_me_ggtt(const mg_process* p, const MeArgs& a, cudaStream_t s) { return rc::launch_sigmakin_recycle<RcGgtt>(p, a, s); }
}  // namespace mg
#else
#include "me_common.cuh"
#include "gen_ggtt.cuh"
namespace mg {
cudaError_t launch_me_ggtt(const mg_process* p, const MeArgs& a, cudaStream_t s) { return launch_sigmakin<Ggtt>(p, a, s); }
}  // namespace mg
#endif
#include "gen_ggtt.cuh"
#include "fused.cuh"
namespace mg {
cudaError_t launch_fused_ggtt(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s) {
  return launch_fused<Ggtt, 2, true>(p, seed, first, n, me, psw, evw, s);
}
}  // namespace mg
