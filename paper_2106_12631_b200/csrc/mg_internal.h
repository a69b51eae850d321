// mg_internal.h — handle layout and the launcher entry points shared by the translation units of
// libmg_b200.so.  Not part of the public ABI (include/mg.h is).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/mg.h"
#include "consts.h"

namespace mg {

}  // namespace mg

struct mg_process {
  mg_params par;
  mg::Consts k;
  int n_ext, n_final, n_hel, n_flows, n_diag, n_amp, denom;
  uint64_t hel_mask;
  // host-call scratch (grown on demand)
  void* d_scratch;
  size_t scratch_bytes;
  void* h_pinned;
  size_t pinned_bytes;
  cudaStream_t own_stream, own_stream2;   // host-buffer calls: chunks alternate between the two (copy/compute overlap)
  cudaEvent_t ev0, ev1;
  double last_kernel_ms;
};

namespace mg {

// alu_peak.cu
cudaError_t measure_alu_peak(int precision, int device, int mode, double* tflops);

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
};
cudaError_t launch_me_eemumu(const mg_process* p, const MeArgs& a, cudaStream_t s);
cudaError_t launch_me_ggtt(const mg_process* p, const MeArgs& a, cudaStream_t s);
cudaError_t launch_me_ggttg(const mg_process* p, const MeArgs& a, cudaStream_t s);
cudaError_t launch_me_ggttgg(const mg_process* p, const MeArgs& a, cudaStream_t s);
// A1-A13 in one kernel (fused.cuh) for the one-thread-per-event processes
cudaError_t launch_fused_eemumu(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s);
cudaError_t launch_fused_ggtt(const mg_process* p, uint64_t seed, uint64_t first, int64_t n, void* me, void* psw, void* evw, cudaStream_t s);
// xsec.cu: batch sums of the event weights and hit-or-miss unweighting
int64_t weight_sums_blocks(int64_t n);
cudaError_t launch_weight_sums(const mg_process* p, const void* d_w, int64_t n, double* d_part, cudaStream_t s);
int64_t unweight_tiles(int64_t n);
cudaError_t launch_unweight(const mg_process* p, uint64_t seed, uint64_t first, const void* d_w, int64_t n, double wmax,
                            int* d_counts, unsigned* d_ballots, int64_t* d_offsets, int64_t* d_out, cudaStream_t s);
// explicit flop tally of one helicity combination / fixed per-event overhead (generated)
int64_t me_flops_per_helicity(int process);
int64_t me_flops_per_event_fixed(int process);
int64_t me_flops_per_event_recycle(int process);   // >= 0: the process runs the recycling kernel
// colour matrix numerators / denominator (generated tables), row-major n_flows x n_flows
const int* me_colour_numerators(int process, int* denom_out);

}  // namespace mg
