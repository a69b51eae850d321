/* mg.h — C ABI of the B200 (sm_100a) tree-level matrix-element library.
 *
 * The library implements the data-parallel hot path of arXiv 2106.12631:
 *   random numbers -> RAMBO momenta -> helicity amplitudes -> colour-summed |M|^2 ("sigmaKin"),
 * PAPER.md:78 (§3, the three components), PAPER.md:92 (§4, data flow), PAPER.md:33/:35 (§2, the
 * ME algorithm).  Stateless functions over a basket of events reading/writing fixed-size C arrays
 * (PAPER.md:94, :98); memory is allocated by the caller before the first and freed after the last
 * iteration.  Readings of the paper's silences are numbered R1.. in DESIGN.md.
 *
 * Conventions common to every call
 *  - Return value: 0 (MG_OK) or a negative MG_E* code; no exceptions, no abort().  n == 0 is a no-op.
 *  - d_* pointers are DEVICE memory owned by the caller; h_* pointers are HOST memory owned by the
 *    caller.  The library allocates nothing per call except where stated, and keeps no reference
 *    to a caller buffer after the work it enqueued has finished.
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls taking only d_*
 *    buffers are asynchronous on that stream unless stated otherwise.
 *  - Element type of every floating-point buffer = the precision of the handle (double for
 *    MG_FP64, float for MG_FP32).
 *  - Layout: structure of arrays, EVENT INDEX FASTEST, row stride `ld` elements (ld >= n):
 *        rnd     [(i_final*4 + k ) * ld + e]    k  = 0..3  (rho_1..rho_4 of final particle i_final)
 *        momenta [(i_par  *4 + mu) * ld + e]    mu = 0..3  (E, px, py, pz), GeV
 *        me, ps_weight, event_weight [e]
 *    Particle order (R9): beams first, then the final state as the process is written:
 *        MG_EEMUMU: e+ e- mu+ mu-      MG_GGTT..: g g t t~ [g [g]]      MG_QQTT, MG_QQTTG: u u~ t t~ [g]  (massless u;
 *        the quark-initiated channel of SURVEY.md 8(f) N4; its colour basis are the diagrams themselves)
 *    Beams (R5): particle 0 = (sqrt_s/2,0,0,+sqrt_s/2), particle 1 = (sqrt_s/2,0,0,-sqrt_s/2).
 *  - Helicity-combination index: bit k of the index = helicity of particle k (0 <-> -1, 1 <-> +1).
 *  - Determinism: the result for event e depends only on (seed, first_event + e, params), never on
 *    n, ld, the launch shape or the stream.
 *  - There is no CPU fallback: every entry point that computes needs a CUDA device of compute
 *    capability 10.x and fails with MG_ECUDA otherwise.
 *  - Streams and threads: a handle may be used with any stream, and with different streams in successive calls.
 *    Calls that need device scratch (the host-buffer forms, mg_weight_sums*, mg_unweight*, and mg_sigmakin /
 *    mg_sigmakin_fused of the FP32 handles of g g -> t t~ g (g)) take it from regions owned by the handle; each
 *    region remembers the end of its last use with an event, the next user's stream waits for it, and a region is
 *    only reallocated after its last user has finished.  Two calls on different streams that need the same region
 *    are therefore serialised on the device, never corrupted.  A handle must not be used by two HOST threads at the
 *    same time (no locking); use one handle per thread.
 */
#ifndef MG_B200_H
#define MG_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mg_process mg_process; /* opaque; owns constant tables, two streams and device scratch regions */

enum { MG_EEMUMU = 0, MG_GGTT = 1, MG_GGTTG = 2, MG_GGTTGG = 3, MG_QQTT = 4, MG_QQTTG = 5 };
enum { MG_FP64 = 0, MG_FP32 = 1 };
enum { MG_OK = 0, MG_EINVAL = -1, MG_EPARAM = -2, MG_ECUDA = -3, MG_ENOMEM = -4, MG_ELIMIT = -5 };
/* stages for mg_flops_per_event / mg_bytes_per_event */
enum { MG_STAGE_RNG = 0, MG_STAGE_RAMBO = 1, MG_STAGE_SIGMAKIN = 2, MG_STAGE_GENERATE = 3 };

/* Physics and run parameters (BASELINE.json configs; readings R12-R15). */
typedef struct {
  int32_t process;     /* MG_EEMUMU .. MG_QQTTG */
  int32_t precision;   /* MG_FP64 | MG_FP32 */
  int32_t device;      /* CUDA device ordinal */
  int32_t reserved;    /* must be 0 */
  double sqrt_s;       /* GeV; 1500 */
  double alpha_em_inv; /* 132.507            (MG_EEMUMU) */
  double mZ, gammaZ;   /* 91.188, 2.441 GeV  (MG_EEMUMU) */
  double mW;           /* 80.419 GeV: sin^2(theta_W) = 1 - mW^2/mZ^2 (R14) */
  double mt;           /* 173 GeV            (MG_GGTT.., MG_QQTT..); the top width is 0 (R12) */
  double alpha_s;      /* 0.118              (MG_GGTT.., MG_QQTT..) */
} mg_params;

/* Fills *out with the BASELINE.json parameter set for (process, precision), device 0. */
int mg_default_params(int process, int precision, mg_params* out);

/* Creates a process handle: validates params (MG_EPARAM if sum of final masses >= sqrt_s or a
 * parameter is not finite/positive), selects the device, allocates a few KB of device scratch.
 * The helicity mask starts as "all helicities" (no filtering).  PAPER.md:136 (constants),
 * PAPER.md:112 (allocation outside the event loop). */
int mg_init_process(const mg_params* params, mg_process** out);
int mg_free_process(mg_process* p);

/* Static facts of the process (Fig. 3: 4/4/5/6 external particles; BASELINE configs). */
int mg_n_external(const mg_process* p);     /* 4,4,5,6 */
int mg_n_final(const mg_process* p);        /* 2,2,3,4 */
int mg_n_helicities(const mg_process* p);   /* 16,16,32,64 */
int mg_n_colour_flows(const mg_process* p); /* 1,2,6,24 */
int mg_n_diagrams(const mg_process* p);     /* 2,3,16,123 */
int mg_n_amplitudes(const mg_process* p);   /* 2,3,18,159 (a 4-gluon vertex carries 3 structures) */
int mg_me_denominator(const mg_process* p); /* 4,256,256,512 (R11) */
/* Colour matrix C (n_flows x n_flows, row-major, doubles) copied to host memory `out`. */
int mg_colour_matrix(const mg_process* p, double* h_out);
/* Smallest row stride the library recommends for n events (n rounded up to a multiple of 32). */
int64_t mg_padded_stride(int64_t n);

/* A1: Philox4x32-10 words (R1, R2).  d_words[(i_final*4+k)*ld + e] = word k of
 * Philox(counter = (event_lo, event_hi, i_final, 0), key = (seed_lo, seed_hi)), event =
 * first_event + e.  uint32 regardless of precision. */
int mg_rng_words(mg_process* p, uint64_t seed, uint64_t first_event, int64_t n, int64_t ld,
                 uint32_t* d_words, void* stream);
/* A1+A2: the same words mapped to uniforms in (0,1) (R3): FP64 (x+0.5)*2^-32, FP32 ((x>>9)+0.5)*2^-23. */
int mg_rng(mg_process* p, uint64_t seed, uint64_t first_event, int64_t n, int64_t ld,
           void* d_rnd, void* stream);

/* A3+A4: RAMBO (Kleiss-Stirling-Ellis; R5-R8).  Reads rnd[4*n_final][ld], writes
 * momenta[4*n_external][ld] (beams included) and the phase-space weight ps_weight[n] (nullable).
 * sqrt_s and masses come from the handle. */
int mg_rambo(mg_process* p, const void* d_rnd, int64_t n, int64_t ld,
             void* d_momenta, void* d_ps_weight, void* stream);

/* A1-A4 fused: uniforms never touch HBM.  Same results as mg_rng + mg_rambo. */
int mg_generate(mg_process* p, uint64_t seed, uint64_t first_event, int64_t n, int64_t ld,
                void* d_momenta, void* d_ps_weight, void* stream);

/* A1-A13 fused (PAPER.md:112-118 copy:compute balance): random numbers, momenta and matrix
 * element of events first_event .. first_event+n-1 without the momenta ever being stored: ONE launch for every
 * process.  Writes me[n] and, if non-NULL, ps_weight[n] and event_weight[n] = ps_weight * me (R18); uses the
 * installed helicity mask.  e+e- -> mu+mu- and g g -> t t~ keep everything in registers; in the shared-memory kernels
 * of g g -> t t~ g(g) four lanes per event of the CTA generate the momenta into shared memory before the first step.
 * Asynchronous on `stream`.  Same values as mg_generate + mg_sigmakin up to rounding of contracted multiply-adds (the
 * shared-memory kernels: the same bits).
 * Errors: MG_EINVAL (NULL/misaligned d_me, bad handle, n < 0), MG_ENOMEM, MG_ECUDA. */
int mg_sigmakin_fused(mg_process* p, uint64_t seed, uint64_t first_event, int64_t n,
                      void* d_me, void* d_ps_weight, void* d_event_weight, void* stream);

/* A5-A13 as TWO kernels per chunk of events under a CUDA graph (§5, the third remedy
 * for the register pressure of sigmaKin: "splitting the SIGMAKIN kernel into many smaller kernels ... orchestrated by
 * CUDA graphs").  Same arguments and the same values, bit for bit, as mg_sigmakin of the same handle; only
 * MG_GGTTG and MG_GGTTGG (the shared-memory kernels), MG_EINVAL otherwise.  Kernel A of a chunk evaluates the
 * amplitudes and writes the colour-flow sums J_f of every evaluated helicity combination to device scratch of the
 * handle; kernel B reads them back and does the colour sum, the helicity sum and the averaging.  The n events are cut
 * into chunks of chunk_events (a positive multiple of 8; 0 = the library's choice, 16 384); chunk c runs on branch
 * c % 2 of the graph with its own scratch, so that B of one chunk overlaps A of the next.  The graph is built on the first call and kept in the handle; it is rebuilt when
 * any argument other than `stream`, or the helicity mask, changes.  FP32 handles: the double-precision pass over the
 * ill-conditioned events (mg_set_fp32_rescue) is NOT part of this path; the values are those of mg_sigmakin with the
 * pass switched off.  This is the measured alternative, not the default: DESIGN.md §7.2 has the numbers.
 * Scratch: 2 * chunk_events * 2^(n_external-1) * n_colour_flows complex numbers.  Asynchronous on `stream`.
 * Errors: MG_EINVAL, MG_ENOMEM, MG_ECUDA. */
int mg_sigmakin_split(mg_process* p, const void* d_momenta, int64_t n, int64_t ld, void* d_me,
                      const void* d_ps_weight, void* d_event_weight, int64_t chunk_events, void* stream);

/* After the hot path ("a fiducial cross section ... and a sample of N_unw unweighted
 * events", "event unweighting, where data stream compaction should in principle be straight-forward").
 *
 * mg_weight_sums: h_sums_out[0..2] = (sum w, sum w^2, max w) over the n non-negative event weights d_weights[n]
 * (element type = the handle's precision), accumulated in double in a fixed order (bit-reproducible for a given n).
 * The cross-section estimate of reading R27 is sum/n / (2 s) * 0.3893793721e9 pb, its MC error
 * sqrt((sum2/n - (sum/n)^2)/n) times the same factor.  Synchronous on `stream` (returns host values).
 *
 * mg_unweight: hit-or-miss against w_max (R29): event e of the batch is kept iff u * w_max < w[e] in the weights'
 * precision, u = word 0 of Philox4x32-10 with key = seed and counter (first_event + e, 0xFFFFFFFF, 0) mapped to (0,1)
 * as in mg_rng (R28): the decision depends on the global event index only.  Writes the batch-relative indices of
 * the kept events in increasing order to d_kept_out[0 .. *h_count_out) (caller allocates n int64) — a stable stream
 * compaction, unique result.  Synchronous.  MG_EINVAL for w_max <= 0, NULL or misaligned pointers.
 * Both use a device scratch region owned by the handle (grown on first use).
 *
 * The *_async forms do the same work and leave the results ON THE DEVICE: d_sums_out[3] doubles, d_count_out one
 * int64 (caller-owned device memory, 8-byte aligned); no allocation once the scratch has its size, no host
 * synchronisation: they can be chained behind mg_sigmakin on one stream or captured in a CUDA graph. */
int mg_weight_sums(mg_process* p, const void* d_weights, int64_t n, double* h_sums_out, void* stream);
int mg_unweight(mg_process* p, uint64_t seed, uint64_t first_event, const void* d_weights, int64_t n, double w_max,
                int64_t* d_kept_out, int64_t* h_count_out, void* stream);
int mg_weight_sums_async(mg_process* p, const void* d_weights, int64_t n, double* d_sums_out, void* stream);
int mg_unweight_async(mg_process* p, uint64_t seed, uint64_t first_event, const void* d_weights, int64_t n, double w_max,
                      int64_t* d_kept_out, int64_t* d_count_out, void* stream);

/* mg_weight_sums_async WITHOUT any allocation, for callers that may not call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it): d_sums_out[0..2] = (sum w, sum w^2, max w) over the n event
 * weights d_weights[n], the same kernels, the same order of additions and therefore the same bits as
 * mg_weight_sums_async.  The per-CTA partial sums between its two kernels live in a
 * fixed 48 KB array in the library's device image (csrc/xsec.cu) instead of the handle's scratch region, which
 * cudaMalloc grows on demand; every GPU that loads the library holds that array until the process exits.
 *  - Limit: n <= mg_weight_sums_static_max_events() = 2^24 (the largest batch of BASELINE.json); MG_ELIMIT beyond it.
 *  - Allocates nothing and frees nothing, on the host or the device.  The first call on a device asks the runtime for
 *    the array's device address (a lookup, not an allocation); make that first call outside a stream capture.
 *  - All calls on a device share the array (all handles, all streams) and there is NO ordering between them: calls
 *    that overlap on the GPU — different streams, or graphs launched concurrently — race on it; keep them on one
 *    stream or order them with events.  Nothing in the array has to start at zero (the second kernel reads only the
 *    partials the first kernel of the same call has written); what a call leaves behind is never read.
 * Asynchronous on `stream`; results stay on the device.  n == 0 writes three zeros.
 * Errors: MG_EINVAL (NULL or misaligned pointer, n < 0, bad handle), MG_ELIMIT, MG_ECUDA. */
int mg_weight_sums_static(mg_process* p, const void* d_weights, int64_t n, double* d_sums_out, void* stream);
int64_t mg_weight_sums_static_max_events(void);

/* A12: good-helicity filter (R16).  Evaluates every helicity combination on the
 * first probe_n events of d_momenta (1 <= probe_n <= n... the caller guarantees probe_n events are
 * present), marks h good iff max_e |M|^2_h / sum_h' |M|^2_h' > 1e-10, returns the mask in
 * *h_out_mask (nullable) AND installs it in the handle.  Synchronises the stream.  Allocates and
 * frees probe_n * n_helicities elements of device scratch. */
int mg_filter_helicities(mg_process* p, const void* d_momenta, int64_t probe_n, int64_t ld,
                         uint64_t* h_out_mask, void* stream);
int mg_set_helicity_mask(mg_process* p, uint64_t mask); /* bits above n_helicities are ignored */
int mg_get_helicity_mask(const mg_process* p, uint64_t* h_out_mask);

/* A5-A11 (+A13): sigmaKin.  me[e] = (1/denominator) * sum over the
 * helicities in the handle's mask of J^dagger C J.  If both d_ps_weight and d_event_weight are
 * non-NULL also writes event_weight[e] = ps_weight[e] * me[e] (R18). */
int mg_sigmakin(mg_process* p, const void* d_momenta, int64_t n, int64_t ld, void* d_me,
                const void* d_ps_weight, void* d_event_weight, void* stream);

/* Mixed precision of the FP32 handles of g g -> t t~ g and g g -> t t~ g g (§6: single
 * precision "would require ... a better control of numeric instabilities").  The FP32 kernel evaluates
 * every propagator denominator in double and lists the events whose largest |s / denominator| exceeds kappa_max (soft
 * or collinear gluons: the gauge cancellations between diagrams then amplify FP32 rounding by ~sqrt(kappa)); a second
 * launch recomputes the listed events in double from the SAME FP32 momenta and overwrites their me / event_weight.
 * The decision depends on the event's momenta only, so results stay independent of batch shape and stream.
 * kappa_max = 0 switches the second pass off (pure FP32).  Default 1000 (2 % of flat RAMBO g g -> t t~ g g events,
 * 0.5 % of g g -> t t~ g).  No effect on FP64 handles and on the other processes.  mg_last_rescued returns the number of events the
 * most recent mg_sigmakin / mg_sigmakin_fused / host call sent through the double pass (synchronises with it). */
int mg_set_fp32_rescue(mg_process* p, double kappa_max);
double mg_get_fp32_rescue(const mg_process* p);
int mg_last_rescued(mg_process* p, int64_t* h_count_out);

/* Diagnostic form of A5-A10: |M|^2 of EVERY helicity combination (mask ignored, no 1/denominator):
 * d_me_hel[h*ld + e].  Used by the filter and by the parity tests (per-helicity |M|^2 is
 * convention independent, R22). */
int mg_sigmakin_per_helicity(mg_process* p, const void* d_momenta, int64_t n, int64_t ld,
                             void* d_me_hel, void* stream);

/* Host-buffer forms (the end-to-end path; "copy ... to the host").  Synchronous.
 * mg_sigmakin_host: copies h_momenta [4*n_external][ld] to the device, runs sigmaKin, copies
 * h_me[n] back; batches of 2^17 events or more go through in up to 8 chunks on two streams of the handle so that
 * the copies overlap the kernels (pinned host buffers are needed for that overlap).  mg_run_host: runs A1-A13 for events [first_event, first_event+n) on the device and
 * copies momenta (nullable), ps_weight (nullable) and me to the host.  Device scratch is grown
 * inside the handle on first use and reused. */
int mg_sigmakin_host(mg_process* p, const void* h_momenta, int64_t n, int64_t ld, void* h_me);
int mg_run_host(mg_process* p, uint64_t seed, uint64_t first_event, int64_t n, int64_t ld,
                void* h_momenta, void* h_ps_weight, void* h_me);

/* Algorithmic work per event of one stage: explicit
 * tallies emitted with the kernels (FMA = 2).  MG_STAGE_SIGMAKIN: e+e- -> mu+mu- and g g -> t t~ (one thread per
 * event, helicity loop over the good helicities) count the CURRENT helicity mask; the shared-memory kernels of
 * g g -> t t~ g (g) evaluate every helicity combination and only drop the masked ones from the sum, so their count
 * does not depend on the mask. */
int64_t mg_flops_per_event(const mg_process* p, int stage);
int64_t mg_bytes_per_event(const mg_process* p, int stage);
/* GPU time in ms of the sigmaKin launches of the last mg_*_host call: CUDA events around the sigmaKin launch(es) of
 * every chunk on its stream, summed over the chunks (copies and the event generation excluded; 0 if none). */
double mg_last_kernel_ms(const mg_process* p);

const char* mg_strerror(int code);
const char* mg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MG_B200_H */
