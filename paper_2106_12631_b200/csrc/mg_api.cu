// mg_api.cu — the C ABI of include/mg.h: argument checking, handle, stream/device plumbing,
// host-buffer (end-to-end) forms.  Every compute step is a kernel launch in rng_rambo.cu / me_*.cu;
// nothing is computed on the host (no CPU fallback).
#include <math.h>
#include <new>
#include <string.h>
#include "mg_internal.h"

using namespace mg;

namespace {

struct ProcInfo { int n_ext, n_final, n_hel, n_flows, n_diag, n_amp, denom; };
const ProcInfo kInfo[6] = {
    {4, 2, 16, 1, 2, 2, 4},        // e+e- -> mu+mu-     
    {4, 2, 16, 2, 3, 3, 256},      // gg -> tt~          (BASELINE.json configs[2])
    {5, 3, 32, 6, 16, 18, 256},    // gg -> tt~g         (configs[3])
    {6, 4, 64, 24, 123, 159, 512}, // gg -> tt~gg        (configs[4])
    {4, 2, 16, 1, 1, 1, 36},       // u u~ -> t t~       (quark-initiated channel; diagrams are the colour basis)
    {5, 3, 32, 5, 5, 5, 36},       // u u~ -> t t~ g
};

// FP32 handles of g g -> t t~ g (g): events with max |s / propagator denominator| above this go through the
// double-precision pass (mg_set_fp32_rescue, chosen from profiles/r02_fp32_accuracy.md)
const double kDefaultRescueKappa = 1000.0;

inline bool valid_handle(const mg_process* p) { return p != nullptr; }
inline size_t elem(const mg_process* p) { return p->par.precision == MG_FP64 ? 8 : 4; }
inline bool aligned(const void* q, size_t a) { return ((uintptr_t)q % a) == 0; }

struct DeviceGuard {
  int prev = -1; bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int cuda_rc(cudaError_t e) { return e == cudaSuccess ? MG_OK : (e == cudaErrorMemoryAllocation ? MG_ENOMEM : MG_ECUDA); }

double rambo_w0(int n, double sqrt_s) {  // (pi/2)^(n-1) s^(n-2) / ((n-1)!(n-2)!) (2 pi)^(4-3n)   (north_star)
  const double pi = 3.14159265358979323846;
  double w = pow(pi / 2, n - 1) * pow(sqrt_s * sqrt_s, n - 2) * pow(2 * pi, 4 - 3 * n);
  for (int i = 2; i <= n - 1; ++i) w /= i;
  for (int i = 2; i <= n - 2; ++i) w /= i;
  return w;
}

// Scratch regions (mg_internal.h).  acquire(): the region holds >= bytes and everything `stream` does from here on
// runs after the previous user of the region (on whatever stream) has finished; growing waits for that user on the
// host before the old buffer is freed.  release(): marks the end of this use on `stream`.
int acquire(mg_scratch& sc, size_t bytes, cudaStream_t stream) {
  if (bytes > sc.bytes) {
    if (sc.used && cudaEventSynchronize(sc.done) != cudaSuccess) { cudaGetLastError(); return MG_ECUDA; }
    if (sc.d) cudaFree(sc.d);
    sc.d = nullptr; sc.bytes = 0; sc.used = false;
    const size_t want = bytes + bytes / 4;                      // head room: a slightly larger batch does not reallocate
    if (cudaMalloc(&sc.d, want) != cudaSuccess) { cudaGetLastError(); return MG_ENOMEM; }
    sc.bytes = want;
  } else if (sc.used) {
    if (cudaStreamWaitEvent(stream, sc.done, 0) != cudaSuccess) { cudaGetLastError(); return MG_ECUDA; }
  }
  return MG_OK;
}
int release(mg_scratch& sc, cudaStream_t stream) {
  if (cudaEventRecord(sc.done, stream) != cudaSuccess) { cudaGetLastError(); return MG_ECUDA; }
  sc.used = true;
  return MG_OK;
}
bool scratch_init(mg_scratch& sc) {
  sc.d = nullptr; sc.bytes = 0; sc.used = false;
  return cudaEventCreateWithFlags(&sc.done, cudaEventDisableTiming) == cudaSuccess;
}
void scratch_free(mg_scratch& sc) {
  if (sc.used) cudaEventSynchronize(sc.done);
  if (sc.d) cudaFree(sc.d);
  if (sc.done) cudaEventDestroy(sc.done);
}

// processes evaluated by the shared-memory kernels (recycle.cuh)
inline bool shared_memory_kernel(const mg_process* p) { return p->par.process == MG_GGTTG || p->par.process == MG_GGTTGG; }
// list of ill-conditioned events of an FP32 batch: [count (8 B, padded to 256)] [n event indices]
inline bool wants_rescue(const mg_process* p) { return shared_memory_kernel(p) && p->par.precision == MG_FP32 && p->rescue_kappa > 0; }
inline size_t rescue_bytes(int64_t n) { return 256 + (size_t)n * sizeof(int64_t); }
inline void set_rescue(const mg_process* p, MeArgs& a, void* region) {
  a.rescue_count = (unsigned long long*)region;
  a.rescue_list = (int64_t*)((char*)region + 256);
  a.rescue_kappa = p->rescue_kappa;
}

cudaError_t launch_me(const mg_process* p, const MeArgs& a, cudaStream_t s) {
  switch (p->par.process) {
    case MG_EEMUMU: return launch_me_eemumu(p, a, s);
    case MG_GGTT: return launch_me_ggtt(p, a, s);
    case MG_GGTTG: return launch_me_ggttg(p, a, s);
    case MG_GGTTGG: return launch_me_ggttgg(p, a, s);
    case MG_QQTT: return launch_me_qqtt(p, a, s);
    case MG_QQTTG: return launch_me_qqttg(p, a, s);
  }
  return cudaErrorInvalidValue;
}

// launch_me plus, for FP32 handles of the shared-memory kernels, the list of ill-conditioned events in rescue region `slot`
int run_me(mg_process* p, MeArgs& a, cudaStream_t s, int slot) {
  if (!wants_rescue(p) || a.hel_out) return cuda_rc(launch_me(p, a, s));
  mg_scratch& sc = p->sc_rescue[slot];
  p->rescue_last_mask |= 1 << slot;
  int rc = acquire(sc, rescue_bytes(a.n), s); if (rc != MG_OK) return rc;
  set_rescue(p, a, sc.d);
  const cudaError_t e = launch_me(p, a, s);
  rc = release(sc, s);
  return e != cudaSuccess ? cuda_rc(e) : rc;
}

int check_soa(const mg_process* p, const void* ptr, int64_t n, int64_t ld) {
  if (!valid_handle(p) || n < 0) return MG_EINVAL;
  if (n == 0) return MG_OK;
  if (ptr == nullptr || ld < n || !aligned(ptr, elem(p))) return MG_EINVAL;
  return MG_OK;
}

}  // namespace

extern "C" {

int mg_default_params(int process, int precision, mg_params* out) {
  if (!out || process < 0 || process > MG_QQTTG || (precision != MG_FP64 && precision != MG_FP32)) return MG_EINVAL;
  memset(out, 0, sizeof(*out));
  out->process = process; out->precision = precision; out->device = 0;
  out->sqrt_s = 1500.0; out->alpha_em_inv = 132.507; out->mZ = 91.188; out->gammaZ = 2.441; out->mW = 80.419;
  out->mt = 173.0; out->alpha_s = 0.118;
  return MG_OK;
}

int mg_init_process(const mg_params* par, mg_process** out) {
  if (!par || !out) return MG_EINVAL;
  *out = nullptr;
  if (par->process < 0 || par->process > MG_QQTTG || (par->precision != MG_FP64 && par->precision != MG_FP32) || par->reserved != 0 || par->device < 0)
    return MG_EINVAL;
  const ProcInfo& I = kInfo[par->process];
  auto pos = [](double x) { return isfinite(x) && x > 0; };
  if (!pos(par->sqrt_s)) return MG_EPARAM;
  if (par->process == MG_EEMUMU) {
    if (!pos(par->alpha_em_inv) || !pos(par->mZ) || !pos(par->mW) || !isfinite(par->gammaZ) || par->gammaZ < 0 || par->mW >= par->mZ) return MG_EPARAM;
  } else {
    if (!pos(par->mt) || !pos(par->alpha_s) || 2 * par->mt >= par->sqrt_s) return MG_EPARAM;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || par->device >= ndev) { cudaGetLastError(); return MG_ECUDA; }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, par->device) != cudaSuccess || prop.major != 10) { cudaGetLastError(); return MG_ECUDA; }

  mg_process* p = new (std::nothrow) mg_process();
  if (!p) return MG_ENOMEM;
  memset(p, 0, sizeof(*p));
  p->par = *par;
  p->n_ext = I.n_ext; p->n_final = I.n_final; p->n_hel = I.n_hel; p->n_flows = I.n_flows;
  p->n_diag = I.n_diag; p->n_amp = I.n_amp; p->denom = I.denom;
  p->hel_mask = I.n_hel == 64 ? ~0ull : ((1ull << I.n_hel) - 1);
  Consts& k = p->k;
  const double pi = 3.14159265358979323846;
  k.sqrt_s = par->sqrt_s;
  for (int i = 0; i < 4; ++i) k.mass[i] = 0;
  k.w0 = rambo_w0(I.n_final, par->sqrt_s);
  if (par->process == MG_EEMUMU) {
    const double sw2 = 1 - (par->mW * par->mW) / (par->mZ * par->mZ), cw2 = 1 - sw2;   // R14
    k.ee = sqrt(4 * pi / par->alpha_em_inv);                                           // R15
    const double gz = k.ee / sqrt(sw2 * cw2);
    k.gzl = gz * (-0.5 + sw2); k.gzr = gz * sw2;
    k.mZ = par->mZ; k.mZ2 = par->mZ * par->mZ; k.mZgZ = par->mZ * par->gammaZ;
    k.me_norm = 1.0 / I.denom;
  } else {
    k.mass[0] = k.mass[1] = par->mt; k.mt = par->mt;
    k.gs = sqrt(4 * pi * par->alpha_s);                                                // R15
    const int ng = I.n_ext - 2;                                                        // = number of g_s vertices of every diagram
    k.me_norm = pow(4 * pi * par->alpha_s, ng) / I.denom;                              // g_s^(2 n_g) / denominator
  }
  p->sm_count = prop.multiProcessorCount;
  p->rescue_kappa = kDefaultRescueKappa;
  DeviceGuard g(par->device);
  bool ok = g.ok && cudaStreamCreateWithFlags(&p->own_stream, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&p->own_stream2, cudaStreamNonBlocking) == cudaSuccess &&
            cudaEventCreate(&p->ev0) == cudaSuccess && cudaEventCreate(&p->ev1) == cudaSuccess &&
            scratch_init(p->sc_host) && scratch_init(p->sc_xsec) && scratch_init(p->sc_rescue[0]) && scratch_init(p->sc_rescue[1]) && scratch_init(p->sc_split) &&
            cudaEventCreateWithFlags(&p->split_fork, cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&p->split_join, cudaEventDisableTiming) == cudaSuccess;
  for (int i = 0; ok && i < 16; ++i) ok = cudaEventCreate(&p->kev[i]) == cudaSuccess;
  if (!ok) { cudaGetLastError(); mg_free_process(p); return MG_ECUDA; }
  *out = p;
  return MG_OK;
}

int mg_free_process(mg_process* p) {
  if (!p) return MG_OK;
  DeviceGuard g(p->par.device);
  scratch_free(p->sc_host); scratch_free(p->sc_xsec); scratch_free(p->sc_rescue[0]); scratch_free(p->sc_rescue[1]);
  scratch_free(p->sc_split);                      // waits for the last graph launch
  if (p->split_exec) cudaGraphExecDestroy(p->split_exec);
  if (p->split_fork) cudaEventDestroy(p->split_fork);
  if (p->split_join) cudaEventDestroy(p->split_join);
  for (int i = 0; i < 16; ++i) if (p->kev[i]) cudaEventDestroy(p->kev[i]);
  if (p->ev0) cudaEventDestroy(p->ev0);
  if (p->ev1) cudaEventDestroy(p->ev1);
  if (p->own_stream) cudaStreamDestroy(p->own_stream);
  if (p->own_stream2) cudaStreamDestroy(p->own_stream2);
  delete p;
  return MG_OK;
}

int mg_n_external(const mg_process* p) { return p ? p->n_ext : MG_EINVAL; }
int mg_n_final(const mg_process* p) { return p ? p->n_final : MG_EINVAL; }
int mg_n_helicities(const mg_process* p) { return p ? p->n_hel : MG_EINVAL; }
int mg_n_colour_flows(const mg_process* p) { return p ? p->n_flows : MG_EINVAL; }
int mg_n_diagrams(const mg_process* p) { return p ? p->n_diag : MG_EINVAL; }
int mg_n_amplitudes(const mg_process* p) { return p ? p->n_amp : MG_EINVAL; }
int mg_me_denominator(const mg_process* p) { return p ? p->denom : MG_EINVAL; }
int64_t mg_padded_stride(int64_t n) { return n <= 0 ? 0 : (n + 31) / 32 * 32; }

int mg_colour_matrix(const mg_process* p, double* h_out) {
  if (!p || !h_out) return MG_EINVAL;
  if (p->par.process == MG_EEMUMU) { h_out[0] = 1.0; return MG_OK; }
  int den = 1;
  const int* num = me_colour_numerators(p->par.process, &den);
  if (!num) return MG_EINVAL;
  for (int i = 0; i < p->n_flows * p->n_flows; ++i) h_out[i] = (double)num[i] / den;
  return MG_OK;
}

int mg_rng_words(mg_process* p, uint64_t seed, uint64_t first_event, int64_t n, int64_t ld, uint32_t* d_words, void* stream) {
  if (!valid_handle(p) || n < 0) return MG_EINVAL;
  if (n == 0) return MG_OK;
  if (!d_words || ld < n || !aligned(d_words, 4)) return MG_EINVAL;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  return cuda_rc(launch_rng_words(p, seed, first_event, n, ld, d_words, (cudaStream_t)stream));
}

int mg_rng(mg_process* p, uint64_t seed, uint64_t first_event, int64_t n, int64_t ld, void* d_rnd, void* stream) {
  int rc = check_soa(p, d_rnd, n, ld); if (rc != MG_OK || n == 0) return rc;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  return cuda_rc(launch_rng(p, seed, first_event, n, ld, d_rnd, (cudaStream_t)stream));
}

int mg_rambo(mg_process* p, const void* d_rnd, int64_t n, int64_t ld, void* d_momenta, void* d_ps_weight, void* stream) {
  int rc = check_soa(p, d_rnd, n, ld); if (rc != MG_OK || n == 0) return rc;
  rc = check_soa(p, d_momenta, n, ld); if (rc != MG_OK) return rc;
  if (d_ps_weight && !aligned(d_ps_weight, elem(p))) return MG_EINVAL;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  return cuda_rc(launch_rambo(p, d_rnd, n, ld, d_momenta, d_ps_weight, (cudaStream_t)stream));
}

int mg_generate(mg_process* p, uint64_t seed, uint64_t first_event, int64_t n, int64_t ld, void* d_momenta, void* d_ps_weight, void* stream) {
  int rc = check_soa(p, d_momenta, n, ld); if (rc != MG_OK || n == 0) return rc;
  if (d_ps_weight && !aligned(d_ps_weight, elem(p))) return MG_EINVAL;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  return cuda_rc(launch_generate(p, seed, first_event, n, ld, d_momenta, d_ps_weight, (cudaStream_t)stream));
}

int mg_sigmakin(mg_process* p, const void* d_momenta, int64_t n, int64_t ld, void* d_me, const void* d_ps_weight, void* d_event_weight, void* stream) {
  int rc = check_soa(p, d_momenta, n, ld); if (rc != MG_OK || n == 0) return rc;
  if (!d_me || !aligned(d_me, elem(p))) return MG_EINVAL;
  MeArgs a{d_momenta, n, ld, d_me, nullptr, nullptr, nullptr, p->hel_mask};
  if (d_ps_weight && d_event_weight) { a.psw = d_ps_weight; a.evw = d_event_weight; }
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  p->rescue_last_mask = 0;
  return run_me(p, a, (cudaStream_t)stream, 0);
}

// mg_sigmakin_split: see include/mg.h and csrc/split.cuh
int mg_sigmakin_split(mg_process* p, const void* d_momenta, int64_t n, int64_t ld, void* d_me, const void* d_ps_weight, void* d_event_weight,
                      int64_t chunk_events, void* stream) {
  int rc = check_soa(p, d_momenta, n, ld); if (rc != MG_OK) return rc;
  if (!shared_memory_kernel(p) || chunk_events < 0 || chunk_events % 8 != 0) return MG_EINVAL;
  if (n == 0) return MG_OK;
  if (!d_me || !aligned(d_me, elem(p))) return MG_EINVAL;
  const bool gg = p->par.process == MG_GGTTGG;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  cudaStream_t s = (cudaStream_t)stream;
  if (cuda_rc(gg ? prepare_split_ggttgg(p) : prepare_split_ggttg(p)) != MG_OK) { cudaGetLastError(); return MG_ECUDA; }
  // default chunk: measured on B200 (chunks of 1 184 .. 262 144 events): chunks whose J_f stay in the L2
  // (6 / 12 KB per event in FP64) lose more to the tails of their short launches than they save in HBM traffic
  int64_t chunk = chunk_events ? chunk_events : 16384;
  if (chunk > n) chunk = (n + 7) / 8 * 8;
  const size_t per_branch = ((gg ? split_scratch_bytes_ggttgg(p, chunk) : split_scratch_bytes_ggttg(p, chunk)) + 255) / 256 * 256;
  const void* psw = (d_ps_weight && d_event_weight) ? d_ps_weight : nullptr;
  void* evw = psw ? d_event_weight : nullptr;
  rc = acquire(p->sc_split, 2 * per_branch, s); if (rc != MG_OK) return rc;
  auto& key = p->split_key;
  const bool same = p->split_exec && key.mom == d_momenta && key.n == n && key.ld == ld && key.me == d_me && key.psw == psw && key.evw == evw &&
                    key.chunk == chunk && key.mask == p->hel_mask && key.scratch == p->sc_split.d;
  if (!same) {
    if (p->split_exec) {
      if (p->sc_split.used) cudaEventSynchronize(p->sc_split.done);       // the old graph may still be running
      cudaGraphExecDestroy(p->split_exec); p->split_exec = nullptr;
    }
    // capture: fork own_stream -> own_stream2, chunk c on branch c % 2 (kernel A, kernel B, its own half of the scratch), join
    cudaStream_t br[2] = {p->own_stream, p->own_stream2};
    const size_t es = elem(p);
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamBeginCapture(br[0], cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) e = cudaEventRecord(p->split_fork, br[0]);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(br[1], p->split_fork, 0);
    int64_t c = 0;
    for (int64_t c0 = 0; e == cudaSuccess && c0 < n; c0 += chunk, ++c) {
      const int64_t width = n - c0 < chunk ? n - c0 : chunk;
      MeArgs a{(const char*)d_momenta + (size_t)c0 * es, width, ld, (char*)d_me + (size_t)c0 * es,
               psw ? (const char*)psw + (size_t)c0 * es : nullptr, evw ? (char*)evw + (size_t)c0 * es : nullptr, nullptr, p->hel_mask};
      void* jamp = (char*)p->sc_split.d + (size_t)(c & 1) * per_branch;
      e = gg ? launch_split_chunk_ggttgg(p, a, jamp, br[c & 1]) : launch_split_chunk_ggttg(p, a, jamp, br[c & 1]);
    }
    if (e == cudaSuccess) e = cudaEventRecord(p->split_join, br[1]);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(br[0], p->split_join, 0);
    const cudaError_t e2 = cudaStreamEndCapture(br[0], &graph);           // always ends the capture, also after an error
    if (e == cudaSuccess) e = e2;
    if (e == cudaSuccess) e = cudaGraphInstantiate(&p->split_exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (e != cudaSuccess) { cudaGetLastError(); p->split_exec = nullptr; return cuda_rc(e); }
    key.mom = d_momenta; key.n = n; key.ld = ld; key.me = d_me; key.psw = psw; key.evw = evw; key.chunk = chunk; key.mask = p->hel_mask;
    key.scratch = p->sc_split.d;
  }
  const cudaError_t e = cudaGraphLaunch(p->split_exec, s);
  rc = release(p->sc_split, s);
  return e != cudaSuccess ? cuda_rc(e) : rc;
}

int mg_sigmakin_fused(mg_process* p, uint64_t seed, uint64_t first_event, int64_t n, void* d_me, void* d_ps_weight, void* d_event_weight, void* stream) {
  if (!valid_handle(p) || n < 0) return MG_EINVAL;
  if (n == 0) return MG_OK;
  const size_t es = elem(p);
  if (!d_me || !aligned(d_me, es) || (d_ps_weight && !aligned(d_ps_weight, es)) || (d_event_weight && !aligned(d_event_weight, es))) return MG_EINVAL;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  cudaStream_t s = (cudaStream_t)stream;
  if (p->par.process == MG_EEMUMU) return cuda_rc(launch_fused_eemumu(p, seed, first_event, n, d_me, d_ps_weight, d_event_weight, s));
  if (p->par.process == MG_GGTT) return cuda_rc(launch_fused_ggtt(p, seed, first_event, n, d_me, d_ps_weight, d_event_weight, s));
  if (p->par.process == MG_QQTT) return cuda_rc(launch_fused_qqtt(p, seed, first_event, n, d_me, d_ps_weight, d_event_weight, s));
  if (p->par.process == MG_QQTTG) return cuda_rc(launch_fused_qqttg(p, seed, first_event, n, d_me, d_ps_weight, d_event_weight, s));
  // shared-memory kernels: the CTA generates the momenta of its events into shared memory (recycle.cuh, M_GEN)
  MeArgs a{nullptr, n, n, d_me, nullptr, d_event_weight, nullptr, p->hel_mask};
  a.gen = true; a.seed = seed; a.first = first_event; a.psw_out = d_ps_weight;
  p->rescue_last_mask = 0;
  return run_me(p, a, s, 0);
}

int mg_weight_sums_async(mg_process* p, const void* d_weights, int64_t n, double* d_sums_out, void* stream) {
  if (!valid_handle(p) || n < 0 || !d_sums_out || !aligned(d_sums_out, sizeof(double))) return MG_EINVAL;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  cudaStream_t s = (cudaStream_t)stream;
  if (n == 0) return cuda_rc(cudaMemsetAsync(d_sums_out, 0, 3 * sizeof(double), s));
  if (!d_weights || !aligned(d_weights, elem(p))) return MG_EINVAL;
  const int64_t nb = weight_sums_blocks(n);
  int rc = acquire(p->sc_xsec, (size_t)nb * 3 * sizeof(double), s); if (rc != MG_OK) return rc;
  const cudaError_t e = launch_weight_sums(p, d_weights, n, (double*)p->sc_xsec.d, d_sums_out, s);
  rc = release(p->sc_xsec, s);
  return e != cudaSuccess ? cuda_rc(e) : rc;
}

int mg_weight_sums(mg_process* p, const void* d_weights, int64_t n, double* h_sums_out, void* stream) {
  if (!valid_handle(p) || n < 0 || !h_sums_out) return MG_EINVAL;
  h_sums_out[0] = h_sums_out[1] = h_sums_out[2] = 0.0;
  if (n == 0) return MG_OK;
  if (!d_weights || !aligned(d_weights, elem(p))) return MG_EINVAL;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  cudaStream_t s = (cudaStream_t)stream;
  const int64_t nb = weight_sums_blocks(n);
  int rc = acquire(p->sc_xsec, (size_t)(nb + 1) * 3 * sizeof(double), s); if (rc != MG_OK) return rc;
  double* d_part = (double*)p->sc_xsec.d;
  double* d_out = d_part + 3 * nb;
  cudaError_t e = launch_weight_sums(p, d_weights, n, d_part, d_out, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(h_sums_out, d_out, 3 * sizeof(double), cudaMemcpyDeviceToHost, s);
  rc = release(p->sc_xsec, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  return e != cudaSuccess ? cuda_rc(e) : rc;
}

int mg_unweight_async(mg_process* p, uint64_t seed, uint64_t first_event, const void* d_weights, int64_t n, double w_max,
                      int64_t* d_kept_out, int64_t* d_count_out, void* stream) {
  if (!valid_handle(p) || n < 0 || !d_count_out || !aligned(d_count_out, sizeof(int64_t))) return MG_EINVAL;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  cudaStream_t s = (cudaStream_t)stream;
  if (n == 0) return cuda_rc(cudaMemsetAsync(d_count_out, 0, sizeof(int64_t), s));
  if (!d_weights || !aligned(d_weights, elem(p)) || !d_kept_out || !aligned(d_kept_out, sizeof(int64_t)) || !(w_max > 0.0)) return MG_EINVAL;
  const int64_t nt = unweight_tiles(n);
  int rc = acquire(p->sc_xsec, (size_t)(nt + 1) * sizeof(unsigned long long), s); if (rc != MG_OK) return rc;
  const cudaError_t e = launch_unweight(p, seed, first_event, d_weights, n, w_max, (unsigned long long*)p->sc_xsec.d, d_kept_out, d_count_out, s);
  rc = release(p->sc_xsec, s);
  return e != cudaSuccess ? cuda_rc(e) : rc;
}

int mg_unweight(mg_process* p, uint64_t seed, uint64_t first_event, const void* d_weights, int64_t n, double w_max,
                int64_t* d_kept_out, int64_t* h_count_out, void* stream) {
  if (!valid_handle(p) || n < 0 || !h_count_out) return MG_EINVAL;
  *h_count_out = 0;
  if (n == 0) return MG_OK;
  if (!d_weights || !aligned(d_weights, elem(p)) || !d_kept_out || !aligned(d_kept_out, sizeof(int64_t)) || !(w_max > 0.0)) return MG_EINVAL;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  cudaStream_t s = (cudaStream_t)stream;
  const int64_t nt = unweight_tiles(n);
  const size_t state_b = ((size_t)(nt + 1) * sizeof(unsigned long long) + 255) / 256 * 256;
  int rc = acquire(p->sc_xsec, state_b + sizeof(int64_t), s); if (rc != MG_OK) return rc;
  int64_t* d_count = (int64_t*)((char*)p->sc_xsec.d + state_b);
  cudaError_t e = launch_unweight(p, seed, first_event, d_weights, n, w_max, (unsigned long long*)p->sc_xsec.d, d_kept_out, d_count, s);
  int64_t total = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&total, d_count, sizeof(int64_t), cudaMemcpyDeviceToHost, s);
  rc = release(p->sc_xsec, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return cuda_rc(e);
  *h_count_out = total;
  return rc;
}

int mg_sigmakin_per_helicity(mg_process* p, const void* d_momenta, int64_t n, int64_t ld, void* d_me_hel, void* stream) {
  int rc = check_soa(p, d_momenta, n, ld); if (rc != MG_OK || n == 0) return rc;
  rc = check_soa(p, d_me_hel, n, ld); if (rc != MG_OK) return rc;
  MeArgs a{d_momenta, n, ld, nullptr, nullptr, nullptr, d_me_hel, 0};
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  return cuda_rc(launch_me(p, a, (cudaStream_t)stream));
}

int mg_set_helicity_mask(mg_process* p, uint64_t mask) {
  if (!p) return MG_EINVAL;
  const uint64_t all = p->n_hel == 64 ? ~0ull : ((1ull << p->n_hel) - 1);
  p->hel_mask = mask & all;
  return MG_OK;
}
int mg_get_helicity_mask(const mg_process* p, uint64_t* out) {
  if (!p || !out) return MG_EINVAL;
  *out = p->hel_mask;
  return MG_OK;
}

int mg_filter_helicities(mg_process* p, const void* d_momenta, int64_t probe_n, int64_t ld, uint64_t* h_out_mask, void* stream) {
  if (!valid_handle(p) || probe_n <= 0 || probe_n > (1 << 20)) return MG_EINVAL;
  int rc = check_soa(p, d_momenta, probe_n, ld); if (rc != MG_OK) return rc;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  const size_t es = elem(p);
  const int64_t pld = mg_padded_stride(probe_n);
  void* d_hel = nullptr;
  if (cudaMalloc(&d_hel, (size_t)pld * p->n_hel * es) != cudaSuccess) { cudaGetLastError(); return MG_ENOMEM; }
  // the probe kernel indexes momenta with the caller's ld and the output with the same ld: use a
  // compact copy of the probe momenta so that both strides are pld
  void* d_mom = nullptr;
  const int rows = 4 * p->n_ext;
  if (cudaMalloc(&d_mom, (size_t)pld * rows * es) != cudaSuccess) { cudaGetLastError(); cudaFree(d_hel); return MG_ENOMEM; }
  cudaStream_t s = (cudaStream_t)stream;
  cudaError_t e = cudaMemcpy2DAsync(d_mom, (size_t)pld * es, d_momenta, (size_t)ld * es, (size_t)probe_n * es, rows, cudaMemcpyDeviceToDevice, s);
  MeArgs a{d_mom, probe_n, pld, nullptr, nullptr, nullptr, d_hel, 0};
  if (e == cudaSuccess) e = launch_me(p, a, s);
  const size_t hb = (size_t)pld * p->n_hel * es;
  void* h = malloc(hb);
  if (!h) { cudaFree(d_hel); cudaFree(d_mom); return MG_ENOMEM; }
  if (e == cudaSuccess) e = cudaMemcpyAsync(h, d_hel, hb, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  cudaFree(d_hel); cudaFree(d_mom);
  if (e != cudaSuccess) { cudaGetLastError(); free(h); return MG_ECUDA; }
  // R16: h is good iff max over probe events of |M|^2_h / sum_h' |M|^2_h' > 1e-10.  (Selection on
  // kernel outputs; the arithmetic of the path is all in the kernel.)
  uint64_t mask = 0;
  for (int64_t ev = 0; ev < probe_n; ++ev) {
    double tot = 0;
    for (int hh = 0; hh < p->n_hel; ++hh) tot += es == 8 ? ((double*)h)[hh * pld + ev] : (double)((float*)h)[hh * pld + ev];
    if (!(tot > 0) || !isfinite(tot)) continue;
    for (int hh = 0; hh < p->n_hel; ++hh) {
      const double v = es == 8 ? ((double*)h)[hh * pld + ev] : (double)((float*)h)[hh * pld + ev];
      if (v / tot > 1e-10) mask |= 1ull << hh;
    }
  }
  free(h);
  if (mask == 0) return MG_EPARAM;
  p->hel_mask = mask;
  if (h_out_mask) *h_out_mask = mask;
  return MG_OK;
}

int mg_sigmakin_host(mg_process* p, const void* h_momenta, int64_t n, int64_t ld, void* h_me) {
  if (!valid_handle(p) || n < 0) return MG_EINVAL;
  if (n == 0) return MG_OK;
  if (!h_momenta || !h_me || ld < n) return MG_EINVAL;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  const size_t es = elem(p);
  const int rows = 4 * p->n_ext;
  const size_t mom_b = (size_t)ld * rows * es, me_b = (size_t)n * es;
  const size_t me_off = (mom_b + 255) / 256 * 256;
  cudaStream_t st[2] = {p->own_stream, p->own_stream2};
  int rc = acquire(p->sc_host, me_off + me_b, st[0]); if (rc != MG_OK) return rc;
  char* d = (char*)p->sc_host.d;
  // The batch goes through in chunks of events that alternate between two streams, so that the H2D copy of one chunk
  // and the D2H copy of another overlap the kernel of a third (PAPER.md:112 copy:compute balance; the momenta are
  // structure-of-arrays, so a chunk is a 2-D copy: `rows` rows of `width` events with row pitch ld).
  const int64_t min_chunk = 1 << 16;
  int nchunk = (int)(n / min_chunk); if (nchunk < 1) nchunk = 1; if (nchunk > 8) nchunk = 8;
  const int64_t per = ((n + nchunk - 1) / nchunk + 31) / 32 * 32;
  p->rescue_last_mask = 0;
  cudaError_t e = cudaEventRecord(p->ev0, st[0]);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(st[1], p->ev0, 0);      // stream 2 starts after the region is ours
  int c = 0;
  for (int64_t c0 = 0; c0 < n && e == cudaSuccess && rc == MG_OK; c0 += per, ++c) {
    const int64_t width = (n - c0) < per ? (n - c0) : per;
    cudaStream_t s = st[c & 1];
    e = cudaMemcpy2DAsync(d + (size_t)c0 * es, (size_t)ld * es, (const char*)h_momenta + (size_t)c0 * es, (size_t)ld * es,
                          (size_t)width * es, rows, cudaMemcpyHostToDevice, s);
    MeArgs a{d + (size_t)c0 * es, width, ld, d + me_off + (size_t)c0 * es, nullptr, nullptr, nullptr, p->hel_mask};
    if (e == cudaSuccess) e = cudaEventRecord(p->kev[2 * c], s);
    if (e == cudaSuccess) rc = run_me(p, a, s, c & 1);
    if (e == cudaSuccess) e = cudaEventRecord(p->kev[2 * c + 1], s);
    if (e == cudaSuccess) e = cudaMemcpyAsync((char*)h_me + (size_t)c0 * es, d + me_off + (size_t)c0 * es, (size_t)width * es, cudaMemcpyDeviceToHost, s);
  }
  if (e == cudaSuccess) e = cudaEventRecord(p->ev1, st[1]);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(st[0], p->ev1, 0);      // the region is free when BOTH streams are done
  if (e == cudaSuccess && rc == MG_OK) rc = release(p->sc_host, st[0]);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st[0]);
  if (e != cudaSuccess) { cudaGetLastError(); return MG_ECUDA; }
  if (rc != MG_OK) return rc;
  double total = 0;
  for (int i = 0; i < c; ++i) { float ms = 0; cudaEventElapsedTime(&ms, p->kev[2 * i], p->kev[2 * i + 1]); total += ms; }
  p->last_kernel_ms = total;
  return MG_OK;
}

int mg_run_host(mg_process* p, uint64_t seed, uint64_t first_event, int64_t n, int64_t ld, void* h_momenta, void* h_ps_weight, void* h_me) {
  if (!valid_handle(p) || n < 0) return MG_EINVAL;
  if (n == 0) return MG_OK;
  if (!h_me || ld < n) return MG_EINVAL;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  const size_t es = elem(p);
  const int rows = 4 * p->n_ext;
  const size_t mom_b = (size_t)ld * rows * es, vec_b = ((size_t)n * es + 255) / 256 * 256;
  const size_t mom_off = 0, w_off = (mom_b + 255) / 256 * 256, me_off = w_off + vec_b;
  cudaStream_t s = p->own_stream;
  int rc = acquire(p->sc_host, me_off + vec_b, s); if (rc != MG_OK) return rc;
  char* d = (char*)p->sc_host.d;
  p->rescue_last_mask = 0;
  cudaError_t e = launch_generate(p, seed, first_event, n, ld, d + mom_off, d + w_off, s);
  if (e == cudaSuccess) e = cudaEventRecord(p->kev[0], s);
  MeArgs a{d + mom_off, n, ld, d + me_off, nullptr, nullptr, nullptr, p->hel_mask};
  if (e == cudaSuccess) rc = run_me(p, a, s, 0);
  if (e == cudaSuccess) e = cudaEventRecord(p->kev[1], s);
  if (e == cudaSuccess && h_momenta) e = cudaMemcpyAsync(h_momenta, d + mom_off, mom_b, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess && h_ps_weight) e = cudaMemcpyAsync(h_ps_weight, d + w_off, (size_t)n * es, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(h_me, d + me_off, (size_t)n * es, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess && rc == MG_OK) rc = release(p->sc_host, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) { cudaGetLastError(); return MG_ECUDA; }
  if (rc != MG_OK) return rc;
  float ms = 0; cudaEventElapsedTime(&ms, p->kev[0], p->kev[1]); p->last_kernel_ms = ms;
  return MG_OK;
}

int mg_set_fp32_rescue(mg_process* p, double kappa_max) {
  if (!p || !(kappa_max >= 0.0)) return MG_EINVAL;
  p->rescue_kappa = kappa_max;
  return MG_OK;
}
double mg_get_fp32_rescue(const mg_process* p) { return p ? p->rescue_kappa : 0.0; }

int mg_last_rescued(mg_process* p, int64_t* h_count_out) {
  if (!p || !h_count_out) return MG_EINVAL;
  *h_count_out = 0;
  DeviceGuard g(p->par.device); if (!g.ok) return MG_ECUDA;
  for (int i = 0; i < 2; ++i) {
    mg_scratch& sc = p->sc_rescue[i];
    if (!sc.used || !((p->rescue_last_mask >> i) & 1)) continue;
    unsigned long long c = 0;
    if (cudaEventSynchronize(sc.done) != cudaSuccess || cudaMemcpy(&c, sc.d, sizeof(c), cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return MG_ECUDA; }
    *h_count_out += (int64_t)c;
  }
  return MG_OK;
}

int64_t mg_flops_per_event(const mg_process* p, int stage) {
  if (!p) return MG_EINVAL;
  if (stage == MG_STAGE_SIGMAKIN) {
    const int64_t rc = me_flops_per_event_recycle(p->par.process, p->par.precision == MG_FP64);
    if (rc >= 0) return rc;
    // helicity combinations the kernel evaluates: the good ones; one of each (h, complement) pair for the QCD processes
    // (helicity-flip symmetry, me_common.cuh flip_half)
    int good = __builtin_popcountll(p->hel_mask);
    if (p->par.process != MG_EEMUMU) {
      uint64_t half = 0;
      for (int h = 0; h < p->n_hel / 2; ++h) half |= (((p->hel_mask >> h) | (p->hel_mask >> (p->n_hel - 1 - h))) & 1ull) << h;
      good = __builtin_popcountll(half);
    }
    const bool f64 = p->par.precision == MG_FP64;
    return me_flops_per_event_fixed(p->par.process, f64) + (int64_t)good * me_flops_per_helicity(p->par.process, f64);
  }
  return 0;  // the RNG and RAMBO stages are HBM-bound; their roofline is bytes (mg_bytes_per_event)
}

int64_t mg_bytes_per_event(const mg_process* p, int stage) {
  if (!p) return MG_EINVAL;
  const int64_t es = (int64_t)elem(p);
  switch (stage) {
    case MG_STAGE_RNG: return es * 4 * p->n_final;                                         // write uniforms
    case MG_STAGE_RAMBO: return es * (4 * p->n_final + 4 * p->n_ext + 1);                  // read uniforms, write momenta + weight
    case MG_STAGE_SIGMAKIN: return es * (4 * p->n_ext + 1);                                // read momenta, write ME
    case MG_STAGE_GENERATE: return es * (4 * p->n_ext + 1);                                // write momenta + weight
  }
  return MG_EINVAL;
}

double mg_last_kernel_ms(const mg_process* p) { return p ? p->last_kernel_ms : 0.0; }

const char* mg_strerror(int code) {
  switch (code) {
    case MG_OK: return "ok";
    case MG_EINVAL: return "invalid argument (null/misaligned pointer, bad size, stride or id)";
    case MG_EPARAM: return "unphysical parameters";
    case MG_ECUDA: return "CUDA error or no sm_100 device";
    case MG_ENOMEM: return "out of memory";
    case MG_ELIMIT: return "size above the fixed maximum of a no-allocation entry point (mg_weight_sums_static_max_events)";
  }
  return "unknown error";
}
const char* mg_version(void) { return "mg-b200 0.2 (sm_100a)"; }

}  // extern "C"
