// xsec.cu — the two steps after the hot path: batch sums of the event weights
// (cross-section estimate) and hit-or-miss unweighting with stream compaction.  Both are HBM-bound passes over
// 8 (4) bytes per event; readings R27-R29 in DESIGN.md.
//
//   weight sums   one pass, every CTA reduces 1024 x ITEMS weights in double (fixed tree: thread-sequential, warp
//                 butterfly, warps in order) and writes one partial (sum, sum of squares, max); the partials are
//                 added on the host in block order -> deterministic for a given n.
//   unweighting   pass 1 takes the decisions (one Philox call per event: this pass is bound by integer issue, not by
//                 HBM), stores them as one ballot word per warp and counts the kept events of every 1024-event
//                 tile; pass 2 is an exclusive scan of the tile counts by one CTA; pass 3 reads the ballots and
//                 scatters the kept event indices in increasing order (ballot ranks inside a warp, warp offsets
//                 inside the tile, tile offset from pass 2): a stable compaction, so the result is unique.
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

template <class T>
__global__ void __launch_bounds__(kTile) unweight_count_kernel(uint64_t seed, uint64_t first, const T* __restrict__ w, int64_t n,
                                                               T wmax, int* __restrict__ counts, unsigned* __restrict__ ballots) {
  const int64_t e = (int64_t)blockIdx.x * kTile + threadIdx.x;
  const bool k = e < n && keep_event<T>(seed, first + (uint64_t)e, __ldcs(w + e), wmax);
  const unsigned b = __ballot_sync(0xffffffffu, k);
  if ((threadIdx.x & 31) == 0) ballots[e >> 5] = b;
  const int c = __syncthreads_count(k);
  if (threadIdx.x == 0) counts[blockIdx.x] = c;
}

// exclusive scan of the tile counts by ONE CTA (2^24 events = 16384 tiles): every thread owns a contiguous chunk,
// the 1024 chunk sums are scanned with warp shuffles (two levels); total -> offsets[ntile]
__global__ void __launch_bounds__(kTile) scan_counts_kernel(const int* __restrict__ counts, int64_t ntile, int64_t* __restrict__ offsets) {
  __shared__ int64_t warp_sum[kTile / 32];
  const int64_t chunk = (ntile + kTile - 1) / kTile;
  const int64_t lo = (int64_t)threadIdx.x * chunk, hi = lo + chunk < ntile ? lo + chunk : ntile;
  int64_t mine = 0;
  for (int64_t i = lo; i < hi; ++i) mine += counts[i];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int64_t incl = mine;                                    // inclusive scan inside the warp
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int64_t t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) warp_sum[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    int64_t v = warp_sum[lane], sc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int64_t t = __shfl_up_sync(0xffffffffu, sc, o);
      if (lane >= o) sc += t;
    }
    warp_sum[lane] = sc - v;                              // exclusive prefix of the warps
  }
  __syncthreads();
  int64_t run = warp_sum[wid] + incl - mine;              // exclusive prefix of this thread's chunk
  for (int64_t i = lo; i < hi; ++i) { offsets[i] = run; run += counts[i]; }
  if (threadIdx.x == kTile - 1) offsets[ntile] = warp_sum[wid] + incl;
}

__global__ void __launch_bounds__(kTile) unweight_scatter_kernel(const unsigned* __restrict__ ballots, const int64_t* __restrict__ offsets,
                                                                 int64_t* __restrict__ out) {
  __shared__ int warp_base[kTile / 32];
  const int64_t e = (int64_t)blockIdx.x * kTile + threadIdx.x;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const unsigned b = __ldg(ballots + (e >> 5));          // one word per warp (events beyond n have a zero bit)
  const bool k = (b >> lane) & 1u;
  if (lane == 0) warp_base[wid] = __popc(b);
  __syncthreads();
  if (threadIdx.x == 0) {
    int acc = 0;
    for (int i = 0; i < kTile / 32; ++i) { const int c = warp_base[i]; warp_base[i] = acc; acc += c; }
  }
  __syncthreads();
  if (k) out[offsets[blockIdx.x] + warp_base[wid] + __popc(b & ((1u << lane) - 1u))] = e;
}

}  // namespace

// partials: 3 doubles per CTA in d_part (caller sizes it with weight_sums_blocks)
int64_t weight_sums_blocks(int64_t n) { return (n + (int64_t)kTile * kItems - 1) / ((int64_t)kTile * kItems); }

cudaError_t launch_weight_sums(const mg_process* p, const void* d_w, int64_t n, double* d_part, cudaStream_t s) {
  const unsigned g = (unsigned)weight_sums_blocks(n);
  if (p->par.precision == MG_FP64) weight_sums_kernel<double><<<g, kTile, 0, s>>>((const double*)d_w, n, d_part);
  else weight_sums_kernel<float><<<g, kTile, 0, s>>>((const float*)d_w, n, d_part);
  return cudaGetLastError();
}

int64_t unweight_tiles(int64_t n) { return (n + kTile - 1) / kTile; }

// d_counts: int[ntile], d_ballots: unsigned[32 * ntile], d_offsets: int64[ntile + 1]; d_out: int64[n] (kept event indices, increasing)
cudaError_t launch_unweight(const mg_process* p, uint64_t seed, uint64_t first, const void* d_w, int64_t n, double wmax,
                            int* d_counts, unsigned* d_ballots, int64_t* d_offsets, int64_t* d_out, cudaStream_t s) {
  const int64_t nt = unweight_tiles(n);
  if (p->par.precision == MG_FP64) {
    unweight_count_kernel<double><<<(unsigned)nt, kTile, 0, s>>>(seed, first, (const double*)d_w, n, wmax, d_counts, d_ballots);
  } else {
    unweight_count_kernel<float><<<(unsigned)nt, kTile, 0, s>>>(seed, first, (const float*)d_w, n, (float)wmax, d_counts, d_ballots);
  }
  scan_counts_kernel<<<1, kTile, 0, s>>>(d_counts, nt, d_offsets);
  unweight_scatter_kernel<<<(unsigned)nt, kTile, 0, s>>>(d_ballots, d_offsets, d_out);
  return cudaGetLastError();
}

}  // namespace mg
