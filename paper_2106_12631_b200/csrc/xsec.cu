// xsec.cu — the two steps after the hot path: batch sums of the event weights
// (cross-section estimate) and hit-or-miss unweighting with stream compaction.  Both are HBM-bound passes over
// 8 (4) bytes per event; readings R27-R29 in DESIGN.md.
//
//   weight sums   pass 1: every CTA reduces 1024 x ITEMS weights in double (fixed tree: thread-sequential, warp
//                 butterfly, warps in order) and writes one partial (sum, sum of squares, max); pass 2: one CTA adds
//                 the partials in a fixed tree and leaves the three results ON THE DEVICE -> deterministic for a
//                 given n, no host round trip.
//   unweighting   ONE pass with a decoupled look-back: a tile of 2048 events takes its decisions (one Philox call per
//                 event), counts them, publishes its count, looks back over the tiles before it until it meets an
//                 inclusive prefix, publishes its own inclusive prefix and scatters the kept event indices (ballot
//                 ranks inside a warp, warp offsets inside the tile, tile offset from the look-back).  Tiles are
//                 handed out by an atomic ticket in launch order, so a tile only ever waits for tiles that already
//                 run; the compaction is stable, so the result is unique.  The weights are read once.
#include "mg_internal.h"
#include "philox.cuh"

namespace mg {
namespace {

constexpr int kTile = 1024;
constexpr int kItems = 8;          // weights per thread in the reduction

template <class T>
__global__ void __launch_bounds__(kTile) weight_sums_kernel(const T* __restrict__ w, int64_t n, double* __restrict__ part) {
  __shared__ double sh[3][kTile / 32];
  const int64_t base = (int64_t)blockIdx.x * kTile * kItems;
  double s1 = 0, s2 = 0, mx = 0;
#pragma unroll
  for (int i = 0; i < kItems; ++i) {
    const int64_t e = base + (int64_t)i * kTile + threadIdx.x;
    if (e < n) {
      const double x = (double)__ldcs(w + e);
      s1 += x; s2 = fma(x, x, s2); mx = fmax(mx, x);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  }
  if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = s1; sh[1][threadIdx.x >> 5] = s2; sh[2][threadIdx.x >> 5] = mx; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0, b = 0, c = 0;
    for (int k = 0; k < kTile / 32; ++k) { a += sh[0][k]; b += sh[1][k]; c = fmax(c, sh[2][k]); }
    part[3 * blockIdx.x + 0] = a; part[3 * blockIdx.x + 1] = b; part[3 * blockIdx.x + 2] = c;
  }
}

// R28 + R29: is event e (global index first + e) kept?  u in (0,1) as in R3, decision in the weights' precision
template <class T>
__device__ __forceinline__ bool keep_event(uint64_t seed, uint64_t event, T w, T wmax) {
  const u32x4 r = philox_event_particle(seed, event, 0xFFFFFFFFu);
  return u32_to_uniform<T>(r.x) * wmax < w;
}

// pass 2 of the weight sums: one CTA, partial b of thread (b mod 256) in increasing b, then a fixed tree
__global__ void __launch_bounds__(256) weight_sums_final_kernel(const double* __restrict__ part, int64_t nb, double* __restrict__ out) {
  __shared__ double sh[3][256];
  double a = 0, b = 0, c = 0;
  for (int64_t i = threadIdx.x; i < nb; i += 256) { a += part[3 * i]; b += part[3 * i + 1]; c = fmax(c, part[3 * i + 2]); }
  sh[0][threadIdx.x] = a; sh[1][threadIdx.x] = b; sh[2][threadIdx.x] = c;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sh[0][threadIdx.x] += sh[0][threadIdx.x + o];
      sh[1][threadIdx.x] += sh[1][threadIdx.x + o];
      sh[2][threadIdx.x] = fmax(sh[2][threadIdx.x], sh[2][threadIdx.x + o]);
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[0] = sh[0][0]; out[1] = sh[1][0]; out[2] = sh[2][0]; }
}

constexpr int kUwThreads = 512, kUwItems = 4, kUwTile = kUwThreads * kUwItems;   // events per tile
constexpr unsigned long long kAggregate = 1ull << 62, kInclusive = 2ull << 62, kValueMask = (1ull << 62) - 1;

// state[t]: status (2 bits) | count (62 bits) of tile t;  state[ntile]: the tile ticket
template <class T>
__global__ void __launch_bounds__(kUwThreads) unweight_kernel(uint64_t seed, uint64_t first, const T* __restrict__ w, int64_t n, T wmax,
                                                              int64_t ntile, unsigned long long* __restrict__ state,
                                                              int64_t* __restrict__ out, int64_t* __restrict__ count_out) {
  __shared__ int cnt[kUwItems * kUwThreads / 32];      // kept events of every (round, warp), then their exclusive prefix
  __shared__ long long tile_sh, base_sh;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (threadIdx.x == 0) tile_sh = (long long)atomicAdd(state + ntile, 1ull);
  __syncthreads();
  const int64_t tile = tile_sh;
  const int64_t e0 = tile * kUwTile;
  unsigned ballots[kUwItems];
#pragma unroll
  for (int i = 0; i < kUwItems; ++i) {
    const int64_t e = e0 + (int64_t)i * kUwThreads + threadIdx.x;
    const bool k = e < n && keep_event<T>(seed, first + (uint64_t)e, __ldcs(w + e), wmax);
    ballots[i] = __ballot_sync(0xffffffffu, k);
    if (lane == 0) cnt[i * (kUwThreads / 32) + wid] = __popc(ballots[i]);
  }
  __syncthreads();
  if (wid == 0) {
    // exclusive scan of the 64 (round, warp) counts: two per lane
    const int a = cnt[2 * lane], b = cnt[2 * lane + 1];
    int incl = a + b;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    cnt[2 * lane] = incl - a - b; cnt[2 * lane + 1] = incl - b;
    if (lane == 0) {
      unsigned long long prefix = 0;
      if (tile > 0) {
        atomicExch(state + tile, kAggregate | (unsigned long long)total);
        for (int64_t j = tile - 1; j >= 0; --j) {
          unsigned long long v;
          do { v = atomicAdd(state + j, 0ull); } while ((v >> 62) == 0);
          prefix += v & kValueMask;
          if ((v >> 62) == 2) break;
        }
      }
      atomicExch(state + tile, kInclusive | (prefix + (unsigned long long)total));
      base_sh = (long long)prefix;
      if (tile == ntile - 1) *count_out = (int64_t)(prefix + (unsigned long long)total);
    }
  }
  __syncthreads();
  const int64_t base = base_sh;
#pragma unroll
  for (int i = 0; i < kUwItems; ++i)
    if ((ballots[i] >> lane) & 1u)
      out[base + cnt[i * (kUwThreads / 32) + wid] + __popc(ballots[i] & ((1u << lane) - 1u))] = e0 + (int64_t)i * kUwThreads + threadIdx.x;
}

}  // namespace

// partials: 3 doubles per CTA in d_part (caller sizes it with weight_sums_blocks)
int64_t weight_sums_blocks(int64_t n) { return (n + (int64_t)kTile * kItems - 1) / ((int64_t)kTile * kItems); }

cudaError_t launch_weight_sums(const mg_process* p, const void* d_w, int64_t n, double* d_part, double* d_out, cudaStream_t s) {
  const unsigned g = (unsigned)weight_sums_blocks(n);
  if (p->par.precision == MG_FP64) weight_sums_kernel<double><<<g, kTile, 0, s>>>((const double*)d_w, n, d_part);
  else weight_sums_kernel<float><<<g, kTile, 0, s>>>((const float*)d_w, n, d_part);
  weight_sums_final_kernel<<<1, 256, 0, s>>>(d_part, (int64_t)g, d_out);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------
// mg_weight_sums_static: the weight sums WITHOUT any allocation (include/mg.h).  The per-CTA partials of pass 1 live in a
// file-scope device array instead of the handle's scratch region (which cudaMalloc grows on demand): for callers that
// may not allocate — code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
// Limit: kStaticMaxEvents events per call (the largest batch of BASELINE.json); the array is 48 KB and every GPU that
// loads the library holds it until the process exits.  All calls on a device share it; pass 2 reads only partials
// that pass 1 of the SAME call has written, so nothing in it has to start at zero and the contents the previous call
// left behind are never read — but two calls that overlap on the GPU (different streams) race on it.
// ---------------------------------------------------------------------------------------------------
constexpr int64_t kStaticMaxEvents = (int64_t)1 << 24;
constexpr int64_t kStaticMaxBlocks = kStaticMaxEvents / ((int64_t)kTile * kItems);      // 2048 CTAs
static __device__ __align__(256) double g_ws_static_partials[3 * kStaticMaxBlocks];     // 49 152 bytes

// In host code the array's name is only a stand-in: its device address is asked for once per device, with that
// device current (not an allocation: the array is part of the loaded module)
static cudaError_t static_partials(int device, double** out) {
  static double* addr[64];
  if (device < 0 || device >= 64) return cudaErrorInvalidDevice;
  if (addr[device] == nullptr) {
    double* q = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&q, g_ws_static_partials);
    if (e != cudaSuccess) return e;
    if (q == nullptr) return cudaErrorInvalidSymbol;
    addr[device] = q;
  }
  *out = addr[device];
  return cudaSuccess;
}

int64_t unweight_tiles(int64_t n) { return (n + kUwTile - 1) / kUwTile; }

cudaError_t launch_unweight(const mg_process* p, uint64_t seed, uint64_t first, const void* d_w, int64_t n, double wmax,
                            unsigned long long* d_state, int64_t* d_out, int64_t* d_count, cudaStream_t s) {
  const int64_t nt = unweight_tiles(n);
  cudaError_t e = cudaMemsetAsync(d_state, 0, (size_t)(nt + 1) * sizeof(unsigned long long), s);
  if (e != cudaSuccess) return e;
  if (p->par.precision == MG_FP64)
    unweight_kernel<double><<<(unsigned)nt, kUwThreads, 0, s>>>(seed, first, (const double*)d_w, n, wmax, nt, d_state, d_out, d_count);
  else
    unweight_kernel<float><<<(unsigned)nt, kUwThreads, 0, s>>>(seed, first, (const float*)d_w, n, (float)wmax, nt, d_state, d_out, d_count);
  return cudaGetLastError();
}

}  // namespace mg

extern "C" {

int64_t mg_weight_sums_static_max_events(void) { return mg::kStaticMaxEvents; }

int mg_weight_sums_static(mg_process* p, const void* d_weights, int64_t n, double* d_sums_out, void* stream) {
  if (p == nullptr || n < 0 || d_sums_out == nullptr || ((uintptr_t)d_sums_out % sizeof(double)) != 0) return MG_EINVAL;
  if (n > mg::kStaticMaxEvents) return MG_ELIMIT;
  const size_t es = p->par.precision == MG_FP64 ? 8 : 4;
  if (n > 0 && (d_weights == nullptr || ((uintptr_t)d_weights % es) != 0)) return MG_EINVAL;
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); return MG_ECUDA; }
  if (prev != p->par.device && cudaSetDevice(p->par.device) != cudaSuccess) { cudaGetLastError(); return MG_ECUDA; }
  cudaStream_t s = (cudaStream_t)stream;
  cudaError_t e;
  if (n == 0) {
    e = cudaMemsetAsync(d_sums_out, 0, 3 * sizeof(double), s);
  } else {
    double* d_part = nullptr;
    e = mg::static_partials(p->par.device, &d_part);
    if (e == cudaSuccess) e = mg::launch_weight_sums(p, d_weights, n, d_part, d_sums_out, s);
  }
  if (e != cudaSuccess) cudaGetLastError();
  if (prev != p->par.device) cudaSetDevice(prev);
  return e == cudaSuccess ? MG_OK : MG_ECUDA;
}

}  // extern "C"
