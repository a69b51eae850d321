// me_ggttg.cu — launcher of the generated g g -> t t~ g sigmaKin kernel: helicity recycling in shared memory
// (recycle.cuh + gen_rc_ggttg.cuh, written by gen/recycle.py).
#include "gen_rc_ggttg.cuh"
#include "split.cuh"
namespace mg {
cudaError_t launch_me_ggttg(const mg_process* p, const MeArgs& a, cudaStream_t s) { return rc::launch_sigmakin_recycle<RcGgttg>(p, a, s); }
cudaError_t prepare_split_ggttg(const mg_process* p) { return rc::prepare_split<RcGgttg>(p); }
size_t split_scratch_bytes_ggttg(const mg_process* p, int64_t chunk) { return rc::split_scratch_bytes<RcGgttg>(p, chunk); }
cudaError_t launch_split_chunk_ggttg(const mg_process* p, const MeArgs& a, void* jamp, cudaStream_t s) { return rc::launch_split_chunk<RcGgttg>(p, a, jamp, s); }

}  // namespace mg
