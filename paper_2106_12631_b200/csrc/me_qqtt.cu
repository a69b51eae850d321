// me_qqtt.cu — launchers of the generated quark-initiated sigmaKin kernels u u~ -> t t~ and u u~ -> t t~ g
// (gen_qqtt.cuh, written by gen/qqgen.py): one thread per event, alone (A5-A13) and
// fused with the event generation (A1-A13, fused.cuh).
#include "me_common.cuh"
#include "gen_qqtt.cuh"
#include "fused.cuh"
namespace mg {
cudaError_t launch_me_qqtt(const mg_process* p, const MeArgs& a, cudaStream_t s) { return launch_sigmakin<Qqtt>(p, a, s); }
cudaError_t launch_me_qqttg(const mg_process* p, const MeArgs& a, cudaStream_t s) { return launch_sigmakin<Qqttg>(p, a, s); }
cudaError_t launch_fused_qqtt(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s) {
  return launch_fused<Qqtt, 2, true>(p, seed, first, n, me, psw, evw, s);
}
cudaError_t launch_fused_qqttg(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s) {
  return launch_fused<Qqttg, 3, true>(p, seed, first, n, me, psw, evw, s);
}
}  // namespace mg
