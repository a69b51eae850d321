// me_ggttgg.cu — launcher of the generated g g -> t t~ g g sigmaKin kernel: helicity recycling in shared
// memory (recycle.cuh + gen_rc_ggttgg.cuh, written by gen/recycle.py).
#include "gen_rc_ggttgg.cuh"
#include "split.cuh"

namespace mg {

cudaError_t launch_me_ggttgg(const mg_process* p, const MeArgs& a, cudaStream_t s) { return rc::launch_sigmakin_recycle<RcGgttgg>(p, a, s); }
cudaError_t prepare_split_ggttgg(const mg_process* p) { return rc::prepare_split<RcGgttgg>(p); }
size_t split_scratch_bytes_ggttgg(const mg_process* p, int64_t chunk) { return rc::split_scratch_bytes<RcGgttgg>(p, chunk); }
cudaError_t launch_split_chunk_ggttgg(const mg_process* p, const MeArgs& a, void* jamp, cudaStream_t s) { return rc::launch_split_chunk<RcGgttgg>(p, a, jamp, s); }

}  // namespace mg
