// me_ggtt.cu — launchers of the generated g g -> t t~ sigmaKin kernel: one thread per event (gen_ggtt.cuh, written by
// gen/qcdgen.py), alone (A5-A13) and fused with the event generation (A1-A13, fused.cuh).
#include "me_common.cuh"
#include "gen_ggtt.cuh"
#include "fused.cuh"
namespace mg {
cudaError_t launch_me_ggtt(const mg_process* p, const MeArgs& a, cudaStream_t s) { return launch_sigmakin<Ggtt>(p, a, s); }
cudaError_t launch_fused_ggtt(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s) {
  return launch_fused<Ggtt, 2, true>(p, seed, first, n, me, psw, evw, s);
}
}  // namespace mg
