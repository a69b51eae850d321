// recycle.cuh — sigmaKin with HELICITY RECYCLING in shared memory: the sm_100a mapping
// of steps A5-A11 for the processes whose live set does not fit one thread's registers.
//
// PAPER.md:136-138 names the register pressure of the one-thread-per-event sigmaKin kernel and lists the
// remedies: shared memory for the wavefunctions, smaller kernels, or "different threads process different
// helicities of the same event".  This kernel combines the first and the last:
//   * a CTA works on E events; thread (e, h) owns helicity combination h of event e;
//   * a wavefunction depends only on the helicities of the external legs it contains.  Each distinct
//     (wavefunction, helicity variant) is a TASK computed once per event by one thread and stored in
//     shared memory (wavefunctions shared between diagrams -> also shared between helicities);
//   * a diagram psibar.Vslash.psi is closed as an inner product of a stored row spinor with a stored
//     column spinor (the half product Vslash.psi or psibar.Vslash is itself a task); diagrams made of gluon
//     trees only are closed as  J(all gluons) . G(t t~ current);
//   * what stays per helicity: the inner products, the +-1 colour-flow sums (jamps in registers), the colour
//     quadratic form, and the reduction over the helicity lanes.
// The task tables (which node, which operands, which momentum, which propagator) and the unrolled
// per-helicity code are written by gen/recycle.py; this header holds the generic task routines and the kernel.
//
// Shared-memory entry layout: entry i of event e holds 4 complex numbers (a Vec4 or a Spinor l0,l1,r0,r1),
// stored component-major  ent[e][k][i], k = 0..3, one 16-byte (FP64) / 8-byte (FP32) word each.  A node with
// nbits helicity bits owns 2^nbits consecutive entries (variant index = its helicity bits, compacted in
// particle order).  Lanes of a warp are helicities of one event, so one request touches <= 2^nbits
// consecutive words: broadcast, conflict-free.
#pragma once
#include "me_common.cuh"
#include "philox.cuh"
#include "rambo.cuh"

namespace mg {
namespace rc {

enum Kind { K_POLVEC = 0, K_UBAR = 1, K_VSP = 2, K_VCUR = 3, K_ROWPROP = 4, K_COLPROP = 5, K_FFCUR = 6, K_SLASHCOL = 7, K_SLASHROW = 8, K_EXT = 9,
            // the same four operations on a signed SUM of slash products (terms in the term table; gen/recycle.py _presum)
            K_ROWPROPN = 10, K_COLPROPN = 11, K_SLASHCOLN = 12, K_SLASHROWN = 13 };

// operand word: low 16 bits = first entry of the operand node, high 16 bits = 4 * mask, where mask says which of
// the consumer's variant bits select the operand's variant (pext through the per-variant table, see pext4)
typedef unsigned int Op;
struct NodeDesc {
  short out;        // first entry of the result
  short prop;       // index into the inverse-propagator table, -1: none
  short mom;        // momentum-table index (line momentum of a propagator; particle index of an external)
  short aux;        // K_EXT: 0/1 = incoming/outgoing polarisation vector, 2 = ubar, 3 = v;  K_VCUR: first term
  int nterm;        // K_VCUR: number of terms
  Op op[2];
};
struct TermDesc {   // one term of a gluon current: type 0: V3(A,kA,B,kB);  1..3: four-gluon structure `type`(A,B,C);
                    // one term of a sum of slash products (K_*N nodes): op[0] = spinor, op[1] = vector, signbit
  short type;
  short momA, momB, pad;
  unsigned int signbit;   // 0 or 0x80000000: the term enters with sign -1
  Op op[3];
};
struct __align__(8) MomDef { signed char c[6]; signed char propkind; signed char pad; };   // momentum = sum_i c[i] p_i ; 0 none, 1: 1/q^2, 2: 1/(q^2-mt^2)

template <class T> struct V2;
template <> struct V2<double> { typedef double2 type; };
template <> struct V2<float> { typedef float2 type; };

// compaction of the bits of v selected by mask (order preserved)
__device__ __forceinline__ int pext(int v, int mask) {
  int r = 0, j = 0;
#pragma unroll
  for (int b = 0; b < 6; ++b)
    if ((mask >> b) & 1) { r |= ((v >> b) & 1) << j; ++j; }
  return r;
}
// pext of a variant index v < 16 with any mask < 16 from ONE 64-bit word per v: nibble `mask` of kPext4[v] is
// pext(v, mask).  A thread's v is fixed within a group (v = low bits of the thread index), so the word is
// fetched once per task and every operand costs a shift and an AND.
__device__ __forceinline__ int entry_of(Op op, unsigned long long pt) {
  return (int)(op & 0xffffu) + (int)((pt >> (op >> 16)) & 15ull);
}
template <int MASK> __device__ __forceinline__ int pextc(int v) {
  int r = 0, j = 0;
#pragma unroll
  for (int b = 0; b < 6; ++b)
    if ((MASK >> b) & 1) { r |= ((v >> b) & 1) << j; ++j; }
  return r;
}

// kernel modes (template parameter MODE, bit set)
//   M_PERHEL  write |M|^2 of every helicity combination instead of the sum (good-helicity filter, parity tests)
//   M_GATHER  the CTA's events are taken from a list of event indices written by an earlier launch (the double-
//             precision pass over the ill-conditioned events of an FP32 batch); persistent grid
//   M_GEN     the momenta are not read but GENERATED by the CTA (Philox -> RAMBO, four lanes per event) into shared
//             memory: mg_sigmakin_fused, A1-A13 in one launch, momenta never in HBM
//   M_SPLIT   kernel A of the two-kernel form (split.cuh, "many smaller kernels ... CUDA graphs"): stop after
//             the colour-flow sums J_f and write them to a.jamp; colour and helicity sums are kernel B's
enum { M_PERHEL = 1, M_GATHER = 2, M_GEN = 4, M_SPLIT = 8 };

// kernel arguments; TI = element type of the caller's arrays (the handle's precision), the arithmetic type T of the
// kernel may be wider (T = double over TI = float in the M_GATHER pass)
template <class TI> struct RcArgs {
  const TI* mom; int64_t n, ld;            // momenta (unused with M_GEN), events, row stride
  TI* me; const TI* psw; TI* psw_out; TI* evw; TI* hel_out;
  uint64_t mask;
  uint64_t seed, first;                    // M_GEN: Philox key and global index of event 0
  int64_t* rlist; unsigned long long* rcount; float kappa;   // ill-conditioned events: list, its length, threshold
  void* jamp;                              // M_SPLIT / colour_sum_kernel: J[f][thread of the grid], one complex word each
};

// view of one event's shared memory.  STAGED: the external momenta sit in shared memory (M_GATHER, M_GEN), else they
// are read from the caller's array by the tasks of step 0
template <class T, class TI, int NSLOT, bool STAGED> struct View {
  typedef typename V2<T>::type W;
  const TI* gm;    // the event's column of the caller's momenta array (row stride gld): externals are read once, by step 0
  int64_t gld;
  const T* pext;   // STAGED: [NPAR][4] external momenta
  const T* mom;    // [NMOM][4]  line momenta
  const T* ip;     // [NMOM]     inverse propagator denominators
  W* ent;          // [4][NSLOT]
  __device__ __forceinline__ cx<T> ld(int k, int i) const { const W w = ent[k * NSLOT + i]; return cx<T>(w.x, w.y); }
  __device__ __forceinline__ void st(int k, int i, cx<T> c) const { W w; w.x = c.re; w.y = c.im; ent[k * NSLOT + i] = w; }
  __device__ __forceinline__ Vec4<T> ldv(int i) const { Vec4<T> v; v.v[0] = ld(0, i); v.v[1] = ld(1, i); v.v[2] = ld(2, i); v.v[3] = ld(3, i); return v; }
  __device__ __forceinline__ Spinor<T> lds(int i) const { Spinor<T> s; s.l[0] = ld(0, i); s.l[1] = ld(1, i); s.r[0] = ld(2, i); s.r[1] = ld(3, i); return s; }
  __device__ __forceinline__ void stv(int i, const Vec4<T>& v) const { st(0, i, v.v[0]); st(1, i, v.v[1]); st(2, i, v.v[2]); st(3, i, v.v[3]); }
  __device__ __forceinline__ void sts(int i, const Spinor<T>& s) const { st(0, i, s.l[0]); st(1, i, s.l[1]); st(2, i, s.r[0]); st(3, i, s.r[1]); }
  __device__ __forceinline__ Mom<T> ldm(int m) const { return ld4(mom + 4 * m); }
  __device__ __forceinline__ T ext(int i, int mu) const {
    if (STAGED) return pext[4 * i + mu];
    return (T)__ldg(gm + (int64_t)(4 * i + mu) * gld);
  }
  __device__ __forceinline__ Mom<T> ldx(int i) const {
    if (STAGED) return ld4(pext + 4 * i);
    Mom<T> p;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) p.v[mu] = (T)__ldg(gm + (int64_t)(4 * i + mu) * gld);
    return p;
  }
  static __device__ __forceinline__ Mom<T> ld4(const T* q) {
    const W a = reinterpret_cast<const W*>(q)[0], b = reinterpret_cast<const W*>(q)[1];
    Mom<T> p; p.v[0] = a.x; p.v[1] = a.y; p.v[2] = b.x; p.v[3] = b.y; return p;
  }
};

// ---------------------------------------------------------------------------------------------------
// one task = one (node, helicity variant v) of one event.  pt = kPext4 word of v (see entry_of).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ double flip(double x, unsigned int signbit) {
  return __hiloint2double(__double2hiint(x) ^ (int)signbit, __double2loint(x));
}
__device__ __forceinline__ float flip(float x, unsigned int signbit) { return __int_as_float(__float_as_int(x) ^ (int)signbit); }
template <class T> __device__ __forceinline__ cx<T> flip(cx<T> a, unsigned int signbit) { return cx<T>(flip(a.re, signbit), flip(a.im, signbit)); }

// acc += (+-) V3(J1,k1,J2,k2): helas.cuh vvv_cur with the sign applied as a sign-bit flip of the three scalars
template <class T> __device__ __forceinline__ void vvv_acc(Vec4<T>& acc, unsigned int signbit, const Vec4<T>& J1, Mom<T> k1, const Vec4<T>& J2, Mom<T> k2) {
  Mom<T> d, e, f;
#pragma unroll
  for (int i = 0; i < 4; ++i) { d.v[i] = k1.v[i] - k2.v[i]; e.v[i] = fma_<T>((T)2, k2.v[i], k1.v[i]); f.v[i] = -fma_<T>((T)2, k1.v[i], k2.v[i]); }
  const cx<T> j12 = flip(mdot(J1, J2), signbit);
  const cx<T> a = flip(mdot(J1, e), signbit);
  const cx<T> b = flip(mdot(J2, f), signbit);
#pragma unroll
  for (int i = 0; i < 4; ++i) acc.v[i] = cfma(b, J1.v[i], cfma(a, J2.v[i], rfma(d.v[i], j12, acc.v[i])));
}
// acc += (+-) [ (A.B) C - (C.B) A ]: every four-gluon structure of helas.cuh vvvv_cur is this form after a
// permutation of its operands, done by the generator (s1: (A,C,B), s2: (A,B,C), s3: (B,A,C))
template <class T> __device__ __forceinline__ void vvvv_acc(Vec4<T>& acc, unsigned int signbit, const Vec4<T>& A, const Vec4<T>& B, const Vec4<T>& C) {
  const cx<T> p = flip(mdot(A, B), signbit), q = flip(mdot(C, B), signbit);
#pragma unroll
  for (int i = 0; i < 4; ++i) acc.v[i] = cfms(q, A.v[i], cfma(p, C.v[i], acc.v[i]));
}

template <class P, class T, int KIND> struct Task;
#define MG_RC_TASK(K) template <class P, class T> struct Task<P, T, K> { \
  template <class VW> static __device__ __forceinline__ void run(const NodeDesc& d, int v, unsigned long long pt, const VW& ev, T mt)

MG_RC_TASK(K_POLVEC) { ev.stv(d.out + v, polvec<T>(ev.ldx(d.mom), v ? 1 : -1, d.aux != 0)); } };
MG_RC_TASK(K_UBAR) { ev.sts(d.out + v, bar(spinor_u<T>(ev.ldx(d.mom), mt, v ? 1 : -1))); } };
MG_RC_TASK(K_VSP) { ev.sts(d.out + v, spinor_v<T>(ev.ldx(d.mom), mt, v ? 1 : -1)); } };
MG_RC_TASK(K_EXT) {      // external wavefunctions of one warp: polarisation vectors and the two spinors
  const Mom<T> p = ev.ldx(d.mom);
  if (d.aux < 2) ev.stv(d.out + v, polvec<T>(p, v ? 1 : -1, d.aux != 0));
  else if (d.aux == 2) ev.sts(d.out + v, bar(spinor_u<T>(p, mt, v ? 1 : -1)));
  else ev.sts(d.out + v, spinor_v<T>(p, mt, v ? 1 : -1));
} };
MG_RC_TASK(K_VCUR) {
  Vec4<T> acc;
#pragma unroll
  for (int i = 0; i < 4; ++i) acc.v[i] = cx<T>((T)0, (T)0);
  for (int it = 0; it < d.nterm; ++it) {
    const TermDesc& t = P::term(d.aux + it);
    const Vec4<T> A = ev.ldv(entry_of(t.op[0], pt));
    const Vec4<T> B = ev.ldv(entry_of(t.op[1], pt));
    if (t.type == 0) {
      vvv_acc<T>(acc, t.signbit, A, ev.ldm(t.momA), B, ev.ldm(t.momB));
    } else {
      const Vec4<T> C = ev.ldv(entry_of(t.op[2], pt));
      vvvv_acc<T>(acc, t.signbit, A, B, C);
    }
  }
  if (d.prop >= 0) acc = scale(ev.ip[d.prop], acc);
  ev.stv(d.out + v, acc);
} };
MG_RC_TASK(K_ROWPROP) {   // psibar' = psibar Vslash (qslash+m) / (q^2-m^2)
  const Spinor<T> s = ev.lds(entry_of(d.op[0], pt));
  const Vec4<T> V = ev.ldv(entry_of(d.op[1], pt));
  ev.sts(d.out + v, ffv_row_prop(s, V, ev.ldm(d.mom), mt, ev.ip[d.prop]));
} };
MG_RC_TASK(K_COLPROP) {   // psi' = (qslash+m) Vslash psi / (q^2-m^2)
  const Spinor<T> s = ev.lds(entry_of(d.op[0], pt));
  const Vec4<T> V = ev.ldv(entry_of(d.op[1], pt));
  ev.sts(d.out + v, ffv_col_prop(s, V, ev.ldm(d.mom), mt, ev.ip[d.prop]));
} };
MG_RC_TASK(K_FFCUR) {     // G = (psibar gamma^mu psi) / K^2
  const Spinor<T> a = ev.lds(entry_of(d.op[0], pt));
  const Spinor<T> b = ev.lds(entry_of(d.op[1], pt));
  ev.stv(d.out + v, scale(ev.ip[d.prop], ff_current(a, b)));
} };
MG_RC_TASK(K_SLASHCOL) {  // half product Vslash psi (op0 = psi, op1 = V)
  const Spinor<T> s = ev.lds(entry_of(d.op[0], pt));
  const Vec4<T> V = ev.ldv(entry_of(d.op[1], pt));
  ev.sts(d.out + v, slash_col(slash_parts(V), s));
} };
MG_RC_TASK(K_SLASHROW) {  // half product psibar Vslash (op0 = psibar, op1 = V)
  const Spinor<T> s = ev.lds(entry_of(d.op[0], pt));
  const Vec4<T> V = ev.ldv(entry_of(d.op[1], pt));
  ev.sts(d.out + v, slash_row(slash_parts(V), s));
} };
// sum_i (+-) psibar_i Vslash_i (ROW) or sum_i (+-) Vslash_i psi_i: wavefunctions that enter the same colour-flow sums with the
// same partner are added up before the propagator / before the inner product (linearity; gen/recycle.py _presum)
template <class P, class T, bool ROW, class VW> __device__ __forceinline__ Spinor<T> slash_sum(const NodeDesc& d, unsigned long long pt, const VW& ev) {
  Spinor<T> acc;
  for (int it = 0; it < d.nterm; ++it) {
    const TermDesc& t = P::term(d.aux + it);
    const Spinor<T> s = ev.lds(entry_of(t.op[0], pt));
    const Vec4<T> V = ev.ldv(entry_of(t.op[1], pt));
    const Spinor<T> x = ROW ? slash_row(slash_parts(V), s) : slash_col(slash_parts(V), s);
    if (it == 0) {
      acc.l[0] = flip(x.l[0], t.signbit); acc.l[1] = flip(x.l[1], t.signbit); acc.r[0] = flip(x.r[0], t.signbit); acc.r[1] = flip(x.r[1], t.signbit);
    } else {
      acc.l[0] = acc.l[0] + flip(x.l[0], t.signbit); acc.l[1] = acc.l[1] + flip(x.l[1], t.signbit);
      acc.r[0] = acc.r[0] + flip(x.r[0], t.signbit); acc.r[1] = acc.r[1] + flip(x.r[1], t.signbit);
    }
  }
  return acc;
}
MG_RC_TASK(K_ROWPROPN) { ev.sts(d.out + v, scale(ev.ip[d.prop], qslash_m_row(ev.ldm(d.mom), mt, slash_sum<P, T, true>(d, pt, ev)))); } };
MG_RC_TASK(K_COLPROPN) { ev.sts(d.out + v, scale(ev.ip[d.prop], qslash_m_col(ev.ldm(d.mom), mt, slash_sum<P, T, false>(d, pt, ev)))); } };
MG_RC_TASK(K_SLASHCOLN) { ev.sts(d.out + v, slash_sum<P, T, false>(d, pt, ev)); } };
MG_RC_TASK(K_SLASHROWN) { ev.sts(d.out + v, slash_sum<P, T, true>(d, pt, ev)); } };
#undef MG_RC_TASK

// shared memory of one CTA
template <class P, class T_, class TI_, int MODE> struct Smem {
  typedef T_ T;
  typedef TI_ TI;
  typedef typename V2<T>::type W;
  static constexpr bool STAGED = (MODE & (M_GATHER | M_GEN)) != 0;
  typedef View<T, TI, P::NSLOT, STAGED> VW;
  unsigned long long* pext4;   // [16]  nibble m of word v = pext(v, m)
  const TI* gmom;  // caller's momenta, column of the CTA's first event; ld, nev: row stride, events of this CTA that exist
  int64_t ld;
  int nev;
  T* mom;   // [E][NMOM][4]
  T* ip;    // [E][NMOM]
  T* pext;  // STAGED: [E][NPAR][4]
  W* ent;   // [E][4][NSLOT]
  T* red;   // [NT/32]
  static constexpr size_t kScalars = (size_t)P::E * (P::NMOM * 5 + (STAGED ? P::NPAR * 4 : 0));
  static constexpr size_t kEntOff = 128 + (kScalars * sizeof(T) + 15) / 16 * 16;
  // STAGED modes keep, after `red`, E event indices (int64) and E phase-space weights (TI)
  // entry table of one event: [4][NSLOT] words + padding.  FP32 words are 8 bytes: a producer warp that spans several
  // events (8 variants x 4 events) would hit the same 16 banks from every event when the event stride is a multiple of
  // 128 bytes (4-way conflict: 33 % of the FP32 kernel's shared-memory wavefronts, profiles/r02_d_*_fp32.md); 64 bytes of
  // padding per event alternate the bank halves.  FP64 words fill a bank row per 8 variants: no padding.
  static constexpr int kEvStride = 4 * P::NSLOT + 64 / (int)sizeof(W);
  static constexpr size_t kRedOff = kEntOff + (size_t)P::E * kEvStride * sizeof(W);
  static constexpr size_t kIdxOff = (kRedOff + (P::NT / 32) * sizeof(T) + 15) / 16 * 16;
  // M_GEN: a CTA generates the momenta of NB batches of E events up front (one or two warps per batch, side by side) and
  // then runs the batches one after the other: the wait for the RAMBO chain is paid once per NB batches (P::GENB / GENB32,
  // gen/recycle.py: 2 for g g -> t t~ g in FP64, else 1).  Batch 0 uses the regions above; batch b > 0 has its own [pext T[E][NPAR][4]] [event indices int64[E]] [weights TI[E]] after them.
  static constexpr int NB = (MODE == M_GEN) ? (sizeof(T) == 8 ? P::GENB : P::GENB32) : 1;
  static constexpr size_t kSlotOff = kIdxOff + (STAGED ? (size_t)P::E * 16 : 0) + 16;
  static constexpr size_t kSlotPext = ((size_t)P::E * P::NPAR * 4 * sizeof(T) + 15) / 16 * 16;
  static constexpr size_t kSlotBytes = kSlotPext + (size_t)P::E * 16;
  static constexpr size_t bytes() { return kSlotOff + (size_t)(NB - 1) * kSlotBytes; }
  __device__ __forceinline__ void bind(unsigned char* raw) {
    pext4 = reinterpret_cast<unsigned long long*>(raw);
    mom = reinterpret_cast<T*>(raw + 128);
    ip = mom + P::E * P::NMOM * 4;
    pext = ip + P::E * P::NMOM;
    ent = reinterpret_cast<W*>(raw + kEntOff);
    red = reinterpret_cast<T*>(raw + kRedOff);
  }
  static __device__ __forceinline__ unsigned char* slot_base(unsigned char* raw, int slot) { return raw + kSlotOff + (size_t)(slot - 1) * kSlotBytes; }
  static __device__ __forceinline__ int64_t* evidx(unsigned char* raw, int slot = 0) {
    return reinterpret_cast<int64_t*>(slot ? slot_base(raw, slot) + kSlotPext : raw + kIdxOff);
  }
  static __device__ __forceinline__ TI* wps(unsigned char* raw, int slot = 0) {
    return reinterpret_cast<TI*>((slot ? slot_base(raw, slot) + kSlotPext : raw + kIdxOff) + (size_t)P::E * 8);
  }
  __device__ __forceinline__ void use_slot(unsigned char* raw, int slot) { if (slot) pext = reinterpret_cast<T*>(slot_base(raw, slot)); }
  __device__ __forceinline__ VW view(int e) const {
    VW v;
    v.gm = gmom + (e < nev ? e : nev - 1); v.gld = ld;     // tail events re-read the last event and are not stored
    v.pext = pext + e * P::NPAR * 4;
    v.mom = mom + e * P::NMOM * 4; v.ip = ip + e * P::NMOM; v.ent = ent + e * kEvStride;
    return v;
  }
};

// task t of a group of `nfam` nodes that all have NB helicity bits: t -> (node, event, variant), variant fastest
// A CTA holds E events in E / EG GROUPS of EG events; a group's threads share its tasks and its barrier, groups never
// exchange data (ebase = first event of the thread's group).
template <class P, class SM, int KIND, int NB> __device__ __forceinline__ void run_group(const SM& s, int first_node, int nfam, int t, typename SM::T mt, int ebase) {
  constexpr int PER = P::EG << NB;
  const int fam = t / PER;
  if (fam >= nfam) return;
  const int r = t - fam * PER, v = r & ((1 << NB) - 1);
  Task<P, typename SM::T, KIND>::run(P::node(first_node + fam), v, s.pext4[v], s.view(ebase + (r >> NB)), mt);
}
// barrier over the threads of one group
template <class P> __device__ __forceinline__ void sync_group(int grp) {
  if (P::EG == P::E || (P::EG * P::NHEL) % 32 != 0) __syncthreads();
  else asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "n"(P::EG * P::NHEL) : "memory");
}
// line momenta (signed sums of external momenta) and inverse propagator denominators, in double also for
// T = float (once per event; k_i.k_j cancels like theta^2 for collinear pairs, R19).  Task t = (event, entry).
template <class P, class SM> __device__ __forceinline__ void run_momtab(const SM& s, int t, typename SM::T mt, int ebase) {
  typedef typename SM::T T;
  if (t >= P::EG * P::NMOM) return;
  const int e = ebase + t / P::NMOM, m = t - (t / P::NMOM) * P::NMOM;
  const MomDef d = P::momdef(m);
  const typename SM::VW ev = s.view(e);
  // the six coefficients (+1 / -1 / 0) arrive as ONE 8-byte constant load and become doubles by bit assembly: no
  // per-coefficient constant load and integer-to-double conversion on the critical path of the first phase
  const unsigned long long dw = *reinterpret_cast<const unsigned long long*>(&d);
  const int propkind = (int)((dw >> 48) & 0xffull);
  double q[4] = {0, 0, 0, 0}, ql[4] = {0, 0, 0, 0};
#pragma unroll
  for (int j = 0; j < P::NPAR; ++j) {
    const int cj = (int)(signed char)((dw >> (8 * j)) & 0xffull);
    const double c = __hiloint2double(cj == 0 ? 0 : (cj > 0 ? 0x3ff00000 : (int)0xbff00000), 0);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      if (sizeof(T) == 8) {
        // FP64: the sum is carried as an unevaluated pair (Knuth's two-sum), see below
        const double x = c * (double)ev.ext(j, mu), a = q[mu];
        const double sm = a + x, bb = sm - a;
        ql[mu] += (a - (sm - bb)) + (x - bb);
        q[mu] = sm;
      } else {
        q[mu] = fma(c, (double)ev.ext(j, mu), q[mu]);      // sums of floats: exact in double up to 2^-29 of the largest
      }
    }
  }
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) s.mom[(e * P::NMOM + m) * 4 + mu] = (T)q[mu];
  double den;
  if (sizeof(T) == 8) {
    // q^2 of a collinear pair cancels like theta^2: in plain double the denominator of such a propagator keeps
    // only eps / theta^2 (3e-10 seen in 2^20 uncut events, R30).  Evaluated here as the exact function of
    // the given momenta to ~2^-100: q = (hi, lo) per component, squares by error-free products (fma), the four terms
    // added in a double-double accumulator.  Once per line momentum and event: < 1 % of the event's flops.
    double sh = 0.0, sl = 0.0;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      const double h = q[mu], l = ql[mu];
      double p = h * h;
      double pe = fma(h, h, -p) + 2.0 * h * l;             // (h + l)^2 = p + pe + O(l^2)
      if (mu) { p = -p; pe = -pe; }
      const double t = sh + p, bb = t - sh;
      sl += ((sh - (t - bb)) + (p - bb)) + pe;
      sh = t;
    }
    if (propkind == 2) {
      const double p = -(double)mt * (double)mt, pe = -fma((double)mt, (double)mt, p);
      const double t = sh + p, bb = t - sh;
      sl += ((sh - (t - bb)) + (p - bb)) + pe;
      sh = t;
    }
    den = sh + sl;
  } else {
    den = fma(q[0], q[0], fma(-q[1], q[1], fma(-q[2], q[2], -q[3] * q[3])));
    if (propkind == 2) den = fma(-(double)mt, (double)mt, den);
  }
  s.ip[e * P::NMOM + m] = propkind ? (T)(1.0 / den) : (T)0;
}

// ---------------------------------------------------------------------------------------------------
// the kernel: grid = ceil(n / E) CTAs of NT = E * NHEL threads (M_GATHER: a persistent grid over the list)
// ---------------------------------------------------------------------------------------------------
// A1-A4 on four lanes per event (M_GEN): lane i < NF of event e draws the four Philox uniforms of final particle i and
// evaluates its direction and energy (the transcendental part of RAMBO, rambo.cuh), then the lanes of an event finish RAMBO
// together (rambo_finish_lanes: every sum in the order of rambo_core, so the momenta are those of mg_generate bit for bit).
// The CTA waits for this chain, which is why it is spread over the particles.  ltid = 4 e + i for e < E: whole warps.
template <class P, class T, class TI>
__device__ __forceinline__ void gen_momenta(int ltid, int64_t event, T* pext, TI* wps, const Consts& k, const RcArgs<TI>& a) {
  constexpr int NF = P::NPAR - 2;
  static_assert((P::E * 4) % 32 == 0 && P::E * 4 <= P::NT, "whole warps generate the momenta");
  const int e = ltid >> 2, i = ltid & 3;
  const u32x4 r = philox_event_particle(a.seed, a.first + (uint64_t)event, (uint32_t)(i < NF ? i : 0));
  TI q0, nx, ny, nz;
  rambo_direction<TI>(u32_to_uniform<TI>(r.x), u32_to_uniform<TI>(r.y), u32_to_uniform<TI>(r.z), u32_to_uniform<TI>(r.w), q0, nx, ny, nz);
  TI pf[4];
  const TI w = rambo_finish_lanes<TI, NF>(i, q0, nx, ny, nz, k, pf);
  T* o = pext + e * P::NPAR * 4;
  if (i < NF) {
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) o[8 + 4 * i + mu] = (T)pf[mu];
  }
  if (i == 0) {
    wps[e] = w;
    const T hs = (T)((TI)0.5 * (TI)k.sqrt_s);          // beams (R5), as rambo_event writes them
    o[0] = hs; o[1] = (T)0; o[2] = (T)0; o[3] = hs;
    o[4] = hs; o[5] = (T)0; o[6] = (T)0; o[7] = -hs;
  }
}

// one batch of E events: events ev0 .. ev0 + E - 1 of `total` (of the caller's arrays, or of the list with M_GATHER)
template <class P, class T, class TI, int MODE>
__device__ __forceinline__ void rc_batch(unsigned char* smem_raw, const Consts& k, const RcArgs<TI>& a, int64_t ev0, int64_t total,
                                         int slot = 0, bool pregen = false) {
  typedef Smem<P, T, TI, MODE> SM;
  constexpr bool PER_HEL = (MODE & M_PERHEL) != 0, GATHER = (MODE & M_GATHER) != 0, GEN = (MODE & M_GEN) != 0;
  // FP32 batches: events whose propagators are close to a pole are listed for the double-precision pass
  constexpr bool FLAG = sizeof(T) == 4 && !PER_HEL && !GATHER;
  SM s;
  s.bind(smem_raw);
  const int tid = threadIdx.x;
  const int el = tid / P::NHEL, hl = tid - el * P::NHEL;
  // helicity combination of this lane: bit i of the lane index is the helicity of particle HPERM[i] (a permutation
  // chosen so that the lanes of a quarter warp share as many shared-memory operands as possible)
  int h = 0;
#pragma unroll
  for (int i = 0; i < P::NBITS; ++i) h |= ((hl >> i) & 1) << ((P::HPERM >> (4 * i)) & 15);
  s.nev = (int)((total - ev0) < (int64_t)P::E ? (total - ev0) : (int64_t)P::E);
  if (SM::STAGED) {
    // A5 (M_GATHER) or A1-A4 (M_GEN): the external momenta of the CTA's events go to shared memory first
    int64_t* evidx = SM::evidx(smem_raw, slot);
    TI* wps = SM::wps(smem_raw, slot);
    s.use_slot(smem_raw, slot);
    if (!pregen) {
    if (tid < P::E) {
      const int e = tid < s.nev ? tid : s.nev - 1;
      evidx[tid] = GATHER ? a.rlist[ev0 + e] : ev0 + e;
    }
    __syncthreads();
    if (GEN) {
      if (tid < P::E * 4) gen_momenta<P, T, TI>(tid, evidx[tid >> 2], s.pext, wps, k, a);
    } else {
      for (int t = tid; t < P::E * P::NPAR * 4; t += P::NT) {
        const int e = t / (P::NPAR * 4), r = t - e * (P::NPAR * 4);
        s.pext[t] = (T)__ldg(a.mom + (int64_t)r * a.ld + evidx[e]);
      }
    }
    __syncthreads();
    }
  } else {
    // A5: the momenta are read straight from the caller's array by the tasks of step 0 (line momenta, external
    // wavefunctions): no staging copy and no barrier in front of the first step
    s.gmom = a.mom + ev0; s.ld = a.ld;
  }
  if (MODE & M_SPLIT) {
    cx<T> jamp[P::NFLOW];
    P::template amplitudes<T>(s, tid, el, h, (T)k.mt, jamp);
    typedef typename V2<T>::type W;
    const int64_t stride = (int64_t)gridDim.x * P::NT;
    W* j = reinterpret_cast<W*>(a.jamp) + (int64_t)blockIdx.x * P::NT + tid;
#pragma unroll
    for (int f = 0; f < P::NFLOW; ++f) { W w; w.x = jamp[f].re; w.y = jamp[f].im; j[f * stride] = w; }
    return;
  }
  T me_h = P::template run<T>(s, tid, el, h, (T)k.mt);     // generated: producer steps + inner products + colour sum
  // index of this thread's event in the caller's arrays
  const int64_t ge = SM::STAGED ? SM::evidx(smem_raw, slot)[el] : ev0 + el;
  const bool live = el < s.nev;

  // helicity-flip symmetry (P::FLIP, R35): the thread's combination h has the last particle at helicity -1; its
  // |M|^2 is also that of the complement NHEL_FULL-1-h (all helicities flipped)
  if (PER_HEL) {
    if (live) {
      a.hel_out[(int64_t)h * a.ld + ge] = (TI)me_h;
      if (P::FLIP) a.hel_out[(int64_t)(P::NHEL_FULL - 1 - h) * a.ld + ge] = (TI)me_h;
    }
    return;
  }
  if (P::FLIP) me_h *= (T)((int)((a.mask >> h) & 1) + (int)((a.mask >> (P::NHEL_FULL - 1 - h)) & 1));
  else if (!((a.mask >> h) & 1)) me_h = (T)0;
  // A11: sum over the helicity lanes of the event (fixed order: butterfly inside the warp, then warps in order)
  constexpr int LANES = P::NHEL < 32 ? P::NHEL : 32;
#pragma unroll
  for (int o = LANES / 2; o > 0; o >>= 1) me_h += __shfl_xor_sync(0xffffffffu, me_h, o);
  if (P::NHEL > 32) {
    if ((tid & 31) == 0) s.red[tid >> 5] = me_h;
    sync_group<P>(tid / (P::EG * P::NHEL));
    if (h == 0) {
      me_h = (T)0;
#pragma unroll
      for (int w = 0; w < P::NHEL / 32; ++w) me_h += s.red[el * (P::NHEL / 32) + w];
    }
  }
  if (FLAG) {
    // conditioning of the event: the largest |s / propagator denominator| (denominators were evaluated in double)
    if (a.rlist != nullptr && hl < LANES) {
      float c = 0.f;
      for (int m = hl; m < P::NMOM; m += LANES) c = fmaxf(c, fabsf((float)s.ip[el * P::NMOM + m]));
#pragma unroll
      for (int o = LANES / 2; o > 0; o >>= 1) c = fmaxf(c, __shfl_xor_sync(0xffffffffu, c, o));
      if (hl == 0 && live && c * (float)(k.sqrt_s * k.sqrt_s) > a.kappa) a.rlist[atomicAdd(a.rcount, 1ull)] = ge;
    }
  }
  if (h == 0 && live) {
    const TI r = (TI)(me_h * (T)k.me_norm);
    a.me[ge] = r;
    if (GEN) {
      const TI w = SM::wps(smem_raw, slot)[el];
      if (a.psw_out != nullptr) a.psw_out[ge] = w;
      if (a.evw != nullptr) a.evw[ge] = w * r;
    } else if (a.evw != nullptr) {
      a.evw[ge] = a.psw[ge] * r;
    }
  }
}

template <class P, class T, class TI, int MODE>
__global__ void __launch_bounds__(P::NT, sizeof(T) == 8 ? P::MINB : P::MINB32) sigmakin_recycle_kernel(const __grid_constant__ Consts k, const __grid_constant__ RcArgs<TI> a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  if (threadIdx.x < 16) {
    unsigned long long w = 0;
#pragma unroll
    for (int m = 0; m < 16; ++m) w |= (unsigned long long)pext(threadIdx.x, m) << (4 * m);
    reinterpret_cast<unsigned long long*>(smem_raw)[threadIdx.x] = w;   // Smem::pext4: first read by the tasks of step 1, after the barrier that ends step 0
  }
  if (MODE & M_GATHER) {
    const int64_t total = (int64_t)*a.rcount;
    for (int64_t ev0 = (int64_t)blockIdx.x * P::E; ev0 < total; ev0 += (int64_t)gridDim.x * P::E) {
      rc_batch<P, T, TI, MODE>(smem_raw, k, a, ev0, total);
      __syncthreads();      // the next batch of the persistent grid overwrites the shared memory
    }
  } else if (MODE == M_GEN && Smem<P, T, TI, MODE>::NB > 1) {
    // the momenta of NB batches first, each on its own warp(s), then the batches one after the other (Smem::NB)
    typedef Smem<P, T, TI, MODE> SM;
    const int64_t b0 = (int64_t)blockIdx.x * SM::NB;
    const int slot = (int)threadIdx.x / (P::E * 4), ltid = (int)threadIdx.x - slot * (P::E * 4);
    const int64_t gev0 = (b0 + slot) * P::E;
    if (slot < SM::NB && gev0 < a.n) {
      SM s;
      s.bind(smem_raw);
      s.use_slot(smem_raw, slot);
      const int64_t left = a.n - gev0;
      const int e = ltid >> 2;
      const int64_t event = gev0 + ((int64_t)e < left ? e : (int)left - 1);     // tail events repeat the last one and are not stored
      if ((ltid & 3) == 0) SM::evidx(smem_raw, slot)[e] = event;
      gen_momenta<P, T, TI>(ltid, event, s.pext, SM::wps(smem_raw, slot), k, a);
    }
    __syncthreads();
#pragma unroll 1
    for (int sl = 0; sl < SM::NB; ++sl) {
      const int64_t ev0 = (b0 + sl) * P::E;
      if (ev0 >= a.n) break;
      if (sl > 0) {
        // the batch body works on the regions of batch 0 (fixed offsets: no pointer that depends on the batch is alive in
        // its steps): momenta, event indices and weights of batch sl are copied there first (1.7 KB)
        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(SM::slot_base(smem_raw, sl));
        SM s0;
        s0.bind(smem_raw);
        unsigned long long* dp = reinterpret_cast<unsigned long long*>(s0.pext);
        unsigned long long* di = reinterpret_cast<unsigned long long*>(SM::evidx(smem_raw));
        constexpr int NP = (int)(SM::kSlotPext / 8), NI = P::E * 2;
        for (int t = threadIdx.x; t < NP + NI; t += P::NT) {
          if (t < NP) { if (t < (int)((size_t)P::E * P::NPAR * 4 * sizeof(T) / 8)) dp[t] = src[t]; }
          else di[t - NP] = src[t];
        }
        __syncthreads();
      }
      rc_batch<P, T, TI, MODE>(smem_raw, k, a, ev0, a.n, 0, true);
      __syncthreads();      // the next batch overwrites the shared memory
    }
  } else {
    rc_batch<P, T, TI, MODE>(smem_raw, k, a, (int64_t)blockIdx.x * P::E, a.n);
  }
}

// Shared-memory carve-out that just holds the `ctas` CTAs the register file admits, `bytes` dynamic shared memory (+1 KB reserved) each:
// the smallest configuration of sm_100 that fits, so that what is left of the 256 KB stays L1 for the register spills
// (asking for 100 % costs 0.8 % on g g -> t t~ g g FP64, profiles/r01_c_*).  The driver rounds the hint UP to a
// supported size, hence the floor.
inline int carveout_percent(size_t bytes, int ctas) {
  static const int kb[] = {0, 8, 16, 32, 64, 100, 132, 164, 196, 228};
  const size_t need = (size_t)ctas * (bytes + 1024);
  for (int c : kb)
    if ((size_t)c * 1024 >= need) return c * 100 / 228;
  return 100;
}

// function attributes are per device: set once per kernel and device (not a stream operation: call it outside a capture).
// *ctas_out (optional): resident CTAs per SM of this kernel (sizes the persistent grid of the M_GATHER pass)
template <class P, class T, class TI, int MODE>
cudaError_t prepare_rc(const mg_process* p, int* ctas_out = nullptr) {
  auto kern = sigmakin_recycle_kernel<P, T, TI, MODE>;
  const size_t sm = Smem<P, T, TI, MODE>::bytes();
  static int done[64], ctas_of[64];
  const int dev = p->par.device & 63;
  cudaError_t e = cudaSuccess;
  if (!done[dev]) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    int ctas = 0;
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, kern, P::NT, sm);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, carveout_percent(sm, ctas));
    if (e != cudaSuccess) return e;
    ctas_of[dev] = ctas > 0 ? ctas : 1;
    done[dev] = 1;
  }
  if (ctas_out) *ctas_out = ctas_of[dev];
  return cudaSuccess;
}

// one launch of one instantiation
template <class P, class T, class TI, int MODE>
cudaError_t launch_rc(const mg_process* p, const RcArgs<TI>& a, unsigned grid, cudaStream_t s, int* ctas_out = nullptr) {
  int ctas = 1;
  const cudaError_t e = prepare_rc<P, T, TI, MODE>(p, &ctas);
  if (e != cudaSuccess) return e;
  if (ctas_out) *ctas_out = ctas;
  if (grid == 0) grid = (unsigned)(ctas * p->sm_count);      // persistent grid
  sigmakin_recycle_kernel<P, T, TI, MODE><<<grid, P::NT, Smem<P, T, TI, MODE>::bytes(), s>>>(p->k, a);
  return cudaGetLastError();
}

// A5-A13 (gen = false) or A1-A13 (gen = true: momenta generated in the kernel, a.seed / a.first) for one batch.
// FP32 handles with a rescue list (a.rlist): the FP32 launch lists the ill-conditioned events, a second launch
// recomputes them in double from the same FP32 momenta.
template <class P>
cudaError_t launch_sigmakin_recycle(const mg_process* p, const MeArgs& m, cudaStream_t s) {
  const unsigned g = (unsigned)((m.n + P::E - 1) / P::E);
  const bool f64 = p->par.precision == MG_FP64;
  cudaError_t e;
  if (f64) {
    RcArgs<double> a{(const double*)m.mom, m.n, m.ld, (double*)m.me, (const double*)m.psw, (double*)m.psw_out, (double*)m.evw,
                     (double*)m.hel_out, m.mask, m.seed, m.first, nullptr, nullptr, 0.f, nullptr};
    if (m.hel_out) return launch_rc<P, double, double, M_PERHEL>(p, a, g, s);
    return m.gen ? launch_rc<P, double, double, M_GEN>(p, a, (g + P::GENB - 1) / P::GENB, s) : launch_rc<P, double, double, 0>(p, a, g, s);
  }
  RcArgs<float> a{(const float*)m.mom, m.n, m.ld, (float*)m.me, (const float*)m.psw, (float*)m.psw_out, (float*)m.evw,
                  (float*)m.hel_out, m.mask, m.seed, m.first, m.rescue_list, m.rescue_count, (float)m.rescue_kappa, nullptr};
  if (m.hel_out) { a.rlist = nullptr; return launch_rc<P, float, float, M_PERHEL>(p, a, g, s); }
  if (a.rlist != nullptr) {
    e = cudaMemsetAsync(a.rcount, 0, sizeof(unsigned long long), s);
    if (e != cudaSuccess) return e;
  }
  e = m.gen ? launch_rc<P, float, float, M_GEN>(p, a, (g + P::GENB32 - 1) / P::GENB32, s) : launch_rc<P, float, float, 0>(p, a, g, s);
  if (e != cudaSuccess || a.rlist == nullptr) return e;
  return m.gen ? launch_rc<P, double, float, M_GATHER | M_GEN>(p, a, 0, s) : launch_rc<P, double, float, M_GATHER>(p, a, 0, s);
}

}  // namespace rc
}  // namespace mg
