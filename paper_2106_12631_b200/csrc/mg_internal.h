// mg_internal.h — handle layout and the launcher entry points shared by the translation units of
// libmg_b200.so.  Not part of the public ABI (include/mg.h is).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/mg.h"
#include "consts.h"

namespace mg {

}  // namespace mg

// A device scratch region owned by the handle.  Users on different streams are ordered through `done`: acquire()
// makes the caller's stream wait for the previous user, release() records the end of the new use (mg_api.cu).
struct mg_scratch {
  void* d;
  size_t bytes;
  cudaEvent_t done;
  bool used;
};

struct mg_process {
  mg_params par;
  mg::Consts k;
  int n_ext, n_final, n_hel, n_flows, n_diag, n_amp, denom;
  int sm_count;
  uint64_t hel_mask;
  // FP32 handles of the shared-memory kernels: events with max |s / propagator denominator| above this are recomputed
  // in double (0 = never); mg_set_fp32_rescue
  double rescue_kappa;
  // device scratch, one region per kind of user, grown on demand: host-buffer calls (momenta, weights, MEs), the
  // steps after the path (partials, tile states), lists of ill-conditioned events (two: one per stream of a host call)
  mg_scratch sc_host, sc_xsec, sc_rescue[2];
  int rescue_last_mask;                   // rescue regions written by the most recent sigmaKin call
  cudaStream_t own_stream, own_stream2;   // host-buffer calls: chunks alternate between the two (copy/compute overlap)
  cudaEvent_t ev0, ev1;
  cudaEvent_t kev[16];                    // start/end of the sigmaKin launch of each chunk of a host call
  double last_kernel_ms;
  // mg_sigmakin_split: the instantiated graph, the arguments it was captured for, its scratch (two branches) and the
  // fork/join events of the capture
  mg_scratch sc_split;
  cudaGraphExec_t split_exec;
  struct { const void* mom; int64_t n, ld; void* me; const void* psw; void* evw; int64_t chunk; uint64_t mask; void* scratch; } split_key;
  cudaEvent_t split_fork, split_join;
};

namespace mg {

// rng_rambo.cu
cudaError_t launch_rng_words(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, int64_t ld,
                             uint32_t* d_words, cudaStream_t s);
cudaError_t launch_rng(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, int64_t ld,
                       void* d_rnd, cudaStream_t s);
cudaError_t launch_rambo(const mg_process* p, const void* d_rnd, int64_t n, int64_t ld, void* d_mom,
                         void* d_w, cudaStream_t s);
cudaError_t launch_generate(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, int64_t ld,
                            void* d_mom, void* d_w, cudaStream_t s);

// me_*.cu : per-process sigmaKin launchers.  hel_out != nullptr selects the per-helicity
// diagnostic kernel (mask ignored).
struct MeArgs {
  const void* mom;
  int64_t n, ld;
  void* me;
  const void* psw;
  void* evw;
  void* hel_out;
  uint64_t mask;
  // shared-memory kernels only (recycle.cuh):
  bool gen = false;                        // momenta generated in the kernel from (seed, first): mg_sigmakin_fused
  uint64_t seed = 0, first = 0;
  void* psw_out = nullptr;                 // gen: phase-space weights written here (nullable)
  int64_t* rescue_list = nullptr;          // FP32: ill-conditioned events are listed here and recomputed in double
  unsigned long long* rescue_count = nullptr;
  double rescue_kappa = 0;
};
cudaError_t launch_me_eemumu(const mg_process* p, const MeArgs& a, cudaStream_t s);
cudaError_t launch_me_ggtt(const mg_process* p, const MeArgs& a, cudaStream_t s);
cudaError_t launch_me_ggttg(const mg_process* p, const MeArgs& a, cudaStream_t s);
cudaError_t launch_me_ggttgg(const mg_process* p, const MeArgs& a, cudaStream_t s);
cudaError_t launch_me_qqtt(const mg_process* p, const MeArgs& a, cudaStream_t s);
cudaError_t launch_me_qqttg(const mg_process* p, const MeArgs& a, cudaStream_t s);
// split.cuh: the two-kernel form of the shared-memory processes (mg_sigmakin_split): attributes of kernel A (outside a
// capture), J scratch of one chunk, kernels A and B of one chunk (a = the chunk's slice of the caller's arrays)
cudaError_t prepare_split_ggttg(const mg_process* p);
cudaError_t prepare_split_ggttgg(const mg_process* p);
size_t split_scratch_bytes_ggttg(const mg_process* p, int64_t chunk);
size_t split_scratch_bytes_ggttgg(const mg_process* p, int64_t chunk);
cudaError_t launch_split_chunk_ggttg(const mg_process* p, const MeArgs& a, void* jamp, cudaStream_t s);
cudaError_t launch_split_chunk_ggttgg(const mg_process* p, const MeArgs& a, void* jamp, cudaStream_t s);
// A1-A13 in one kernel (fused.cuh) for the one-thread-per-event processes
cudaError_t launch_fused_eemumu(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s);
cudaError_t launch_fused_ggtt(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s);
cudaError_t launch_fused_qqtt(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s);
cudaError_t launch_fused_qqttg(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s);
// xsec.cu: batch sums of the event weights and hit-or-miss unweighting
int64_t weight_sums_blocks(int64_t n);
// d_part: 3 doubles per block of weight_sums_blocks(n); d_out: (sum, sum of squares, max)
cudaError_t launch_weight_sums(const mg_process* p, const void* d_w, int64_t n, double* d_part, double* d_out, cudaStream_t s);
int64_t unweight_tiles(int64_t n);
// d_state: unweight_tiles(n) + 1 words of 8 bytes (tile states of the decoupled look-back + the tile ticket), zeroed by
// the launcher; d_out: kept event indices in increasing order; d_count: their number
cudaError_t launch_unweight(const mg_process* p, uint64_t seed, uint64_t first, const void* d_w, int64_t n, double wmax,
                            unsigned long long* d_state, int64_t* d_out, int64_t* d_count, cudaStream_t s);
// explicit flop tally of one helicity combination / fixed per-event overhead (generated)
int64_t me_flops_per_helicity(int process, bool fp64);
int64_t me_flops_per_event_fixed(int process, bool fp64);
int64_t me_flops_per_event_recycle(int process, bool fp64);   // >= 0: the process runs the recycling kernel
// colour matrix numerators / denominator (generated tables), row-major n_flows x n_flows
const int* me_colour_numerators(int process, int* denom_out);

}  // namespace mg
