// split.cuh — sigmaKin of the shared-memory processes SPLIT INTO TWO KERNELS under a CUDA graph: the third remedy of
// PAPER.md:136 (§5: "splitting the SIGMAKIN kernel into many smaller kernels ... orchestrated by CUDA graphs"),
// SURVEY.md §8(f) N1.  Built to be measured against the single kernel of recycle.cuh, which stays the default
// (DESIGN.md §7.2 has the numbers).
//
// The cut is where the live state is smallest and the two halves differ most in what they need:
//   kernel A  (sigmakin_recycle_kernel<.., M_SPLIT>)  steps A5-A9: wavefunctions, amplitudes, colour-flow sums J_f of
//             every evaluated helicity combination; writes the J_f (NFLOW complex numbers per thread) to a scratch array;
//   kernel B  (colour_sum_kernel, below)             steps A10-A13: colour quadratic form, helicity sum, averaging,
//             event weight; no shared memory, no barriers, 64 registers.
// The events of a call are cut into chunks of `chunk` events; chunk c runs A then B on branch c % 2 of the graph, each
// branch with its own scratch buffer, so that B of one chunk overlaps A of the next and — for chunks whose J_f fit the
// L2 — the J_f never reach HBM.  Scratch layout: J[f][t], t = index of the thread within the chunk's grid (the same in
// A and B: t = CTA * NT + thread), one 16-byte (FP64) / 8-byte (FP32) word each: consecutive threads, consecutive words.
#pragma once
#include "recycle.cuh"

namespace mg {
namespace rc {

template <class P, class T>
__global__ void __launch_bounds__(P::NT) colour_sum_kernel(const __grid_constant__ Consts k, const __grid_constant__ RcArgs<T> a) {
  static_assert(P::NHEL <= 32, "one event per warp or less");
  typedef typename V2<T>::type W;
  const int tid = threadIdx.x;
  const int el = tid / P::NHEL, hl = tid - el * P::NHEL;
  int h = 0;
#pragma unroll
  for (int i = 0; i < P::NBITS; ++i) h |= ((hl >> i) & 1) << ((P::HPERM >> (4 * i)) & 15);
  const int64_t stride = (int64_t)gridDim.x * P::NT;
  const W* j = reinterpret_cast<const W*>(a.jamp) + (int64_t)blockIdx.x * P::NT + tid;
  cx<T> jamp[P::NFLOW];
#pragma unroll
  for (int f = 0; f < P::NFLOW; ++f) { const W w = j[f * stride]; jamp[f] = cx<T>(w.x, w.y); }
  T me_h = P::template colour<T>(jamp);
  if (P::FLIP) me_h *= (T)((int)((a.mask >> h) & 1) + (int)((a.mask >> (P::NHEL_FULL - 1 - h)) & 1));
  else if (!((a.mask >> h) & 1)) me_h = (T)0;
#pragma unroll
  for (int o = P::NHEL / 2; o > 0; o >>= 1) me_h += __shfl_xor_sync(0xffffffffu, me_h, o);
  const int64_t ge = (int64_t)blockIdx.x * P::E + el;
  if (h == 0 && ge < a.n) {
    const T r = me_h * (T)k.me_norm;
    a.me[ge] = r;
    if (a.evw != nullptr) a.evw[ge] = a.psw[ge] * r;
  }
}

// function attributes of kernel A: to be set before the graph is captured
template <class P> cudaError_t prepare_split(const mg_process* p) {
  return p->par.precision == MG_FP64 ? prepare_rc<P, double, double, M_SPLIT>(p) : prepare_rc<P, float, float, M_SPLIT>(p);
}

// bytes of J scratch one chunk of `chunk` events needs
template <class P> size_t split_scratch_bytes(const mg_process* p, int64_t chunk) {
  const size_t word = p->par.precision == MG_FP64 ? 16 : 8;
  return (size_t)((chunk + P::E - 1) / P::E) * P::NT * P::NFLOW * word;
}

// kernels A and B of one chunk on stream s: m describes the chunk's slice of the caller's arrays
template <class P, class T> cudaError_t launch_split_chunk_t(const mg_process* p, const MeArgs& m, void* jamp, cudaStream_t s) {
  const unsigned g = (unsigned)((m.n + P::E - 1) / P::E);
  RcArgs<T> a{(const T*)m.mom, m.n, m.ld, (T*)m.me, (const T*)m.psw, nullptr, (T*)m.evw, nullptr, m.mask, 0, 0, nullptr, nullptr, 0.f, jamp};
  const cudaError_t e = launch_rc<P, T, T, M_SPLIT>(p, a, g, s);
  if (e != cudaSuccess) return e;
  colour_sum_kernel<P, T><<<g, P::NT, 0, s>>>(p->k, a);
  return cudaGetLastError();
}
template <class P> cudaError_t launch_split_chunk(const mg_process* p, const MeArgs& m, void* jamp, cudaStream_t s) {
  return p->par.precision == MG_FP64 ? launch_split_chunk_t<P, double>(p, m, jamp, s) : launch_split_chunk_t<P, float>(p, m, jamp, s);
}

}  // namespace rc
}  // namespace mg
