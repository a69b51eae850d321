"""Offline generator of the gg -> t t~ (+ g, + g g) sigmaKin kernels (replaces the paper's
MG5aMC/ALOHA code generation, for exactly these processes).

What it does:
  1. enumerates the tree-level Feynman diagrams: one quark line from t to t~ with an ordered
     sequence of gluon trees attached; gluon trees built recursively from 3- and 4-gluon vertices
     (SURVEY.md §8(c) C6 recurrence: 3 / 16 / 123 diagrams, 3 / 18 / 159 amplitudes);
  2. decomposes every colour factor onto the colour-flow basis (strings T^{a_s1}...T^{a_sn},
     permutations in lexicographic order) with f^{abc} T^c = -i [T^a, T^b]; with the REDUCED Feynman
     rules of csrc/helas.cuh all coefficients are +-1;
  3. merges sub-diagrams with the same colour structure into one off-shell current (a 4-gluon
     structure has the colour of a chain of two 3-gluon vertices), shares every wavefunction between
     all diagrams that contain it, chooses for each diagram the vertex at which the
     amplitude is closed so that the number of distinct wavefunctions is small;
  4. emits the CUDA source (a `Proc` struct for csrc/me_common.cuh), the colour matrix, and an
     explicit flop tally.

Run:  python -m paper_2106_12631_b200.gen.qcdgen          (rewrites csrc/gen_*.cuh)
"""
import itertools
import os
from collections import OrderedDict

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(os.path.dirname(HERE), "csrc")

# ----------------------------------------------------------------------------------------------
# flop costs of the helas.cuh routines (FMA = 2, complex mul = 6, complex add = 2, cfma = 8, rfma = 4)
# ----------------------------------------------------------------------------------------------
F_MDOT_VV = 30
F_MDOT_VK = 14
F_SLASH_PARTS = 8
F_SLASH = 56
F_QSLASH = 58
F_SCALE = 8
F_FFV_PROP = F_SLASH_PARTS + F_SLASH + F_QSLASH + F_SCALE      # 130
F_ROW_COL = 30
F_FFV_AMP = F_SLASH_PARTS + F_SLASH + F_ROW_COL                 # 94
F_FF_CUR = 72
F_VVV_K = 20
F_VVV_CUR = F_VVV_K + F_MDOT_VV + 2 * F_MDOT_VK + 80            # 158
F_VVV_AMP = F_VVV_K + 3 * F_MDOT_VV + 3 * F_MDOT_VK + 6 + 16    # 174
F_VVVV_CUR = 2 * F_MDOT_VV + 64                                 # 124
F_VVVV_AMP = 4 * F_MDOT_VV + 14                                 # 134
F_POLVEC = 24        # 2 rsqrt-type ops, ~10 mul, per helicity (pT != 0 branch)
F_SPINOR = 30        # 2 sqrt, 2 div, ~12 mul


# ----------------------------------------------------------------------------------------------
# colour algebra on words (tuples of gluon ids)
# ----------------------------------------------------------------------------------------------
def pmul(a, b):
    r = {}
    for wa, ca in a.items():
        for wb, cb in b.items():
            w = wa + wb
            r[w] = r.get(w, 0) + ca * cb
    return {w: c for w, c in r.items() if c != 0}


def padd(a, b, sb=1):
    r = dict(a)
    for w, c in b.items():
        r[w] = r.get(w, 0) + sb * c
    return {w: c for w, c in r.items() if c != 0}


def comm(a, b):
    return padd(pmul(a, b), pmul(b, a), -1)


def canon(p):
    """(sign, canonical poly as sorted tuple) with the coefficient of the smallest word made positive."""
    items = sorted(p.items())
    s = 1 if items[0][1] > 0 else -1
    return s, tuple((w, c * s) for w, c in items)


# ----------------------------------------------------------------------------------------------
# wavefunction / operation records
# ----------------------------------------------------------------------------------------------
class Struct:
    """One off-shell gluon current of a gluon subset with a definite colour structure."""

    def __init__(self, subset, colour, name):
        self.subset = subset          # frozenset of gluon ids
        self.colour = colour          # canonical poly (tuple)
        self.name = name
        self.terms = []               # (sign, 'V3', a, b) | (sign, 'S4', which, a, b, c)
        self.namp = 0                 # raw (MG-style) sub-amplitudes merged here
        self.namp4 = 0                # of which contain a 4-gluon vertex


def set_partitions_2(S):
    S = sorted(S)
    lo, rest = S[0], S[1:]
    for r in range(0, len(rest)):
        for extra in itertools.combinations(rest, r):
            A = frozenset((lo,) + extra)
            B = frozenset(S) - A
            if B:
                yield A, B


def set_partitions_3(S):
    for A, R in set_partitions_2(S):
        if len(R) < 2:
            continue
        for B, C in set_partitions_2(R):
            yield A, B, C


def ordered_set_partitions(items):
    """All ordered partitions of a list of distinct items into non-empty blocks (as frozensets)."""
    items = list(items)
    if not items:
        yield ()
        return
    n = len(items)
    for r in range(1, n + 1):
        for first in itertools.combinations(items, r):
            rest = [x for x in items if x not in first]
            for tail in ordered_set_partitions(rest):
                yield (frozenset(first),) + tail


class Generator:
    def __init__(self, ng):
        self.ng = ng
        self.gl_particle = [0, 1, 4, 5][:ng]
        self.flows = list(itertools.permutations(range(ng)))
        self.flow_index = {w: i for i, w in enumerate(self.flows)}
        self.cur = {}                     # subset -> list of Struct
        self.struct_order = []            # creation order of composite structs
        self.quark_wfs = OrderedDict()    # name -> ('L'|'R', prev_name, struct, absorbed subset)
        self.closures = []                # (colour poly dict, [(sign, kind, args...)])
        self.n_amp = 0
        self.n_amp4 = 0
        self._build_currents()
        self._build_diagrams()

    # ------------------------------------------------------------------ gluon trees
    def _sname(self, S):
        return "".join(str(g) for g in sorted(S))

    def _build_currents(self):
        ng = self.ng
        for g in range(ng):
            s = Struct(frozenset([g]), canon({(g,): 1})[1], "eps%d" % g)
            s.namp = 1
            self.cur[frozenset([g])] = [s]
        for size in range(2, ng):          # proper subsets only; the full set is closed with the t t~ current
            for S in map(frozenset, itertools.combinations(range(ng), size)):
                self.cur[S] = self._combine(S, as_current=True)

    def _combine(self, S, as_current):
        """All colour structures of the gluon trees over subset S (root vertex 3g or 4g)."""
        groups = OrderedDict()

        def add(col, term, namp, namp4):
            sg, key = canon(col)
            if key not in groups:
                groups[key] = Struct(S, key, None)
            st = groups[key]
            st.terms.append((sg * term[0],) + term[1:])
            st.namp += namp
            st.namp4 += namp4

        for A, B in set_partitions_2(S):
            for a in self.cur[A]:
                for b in self.cur[B]:
                    add(comm(dict(a.colour), dict(b.colour)), (1, "V3", a, b), a.namp * b.namp,
                        a.namp4 * b.namp + a.namp * b.namp4)
        for A, B, C in set_partitions_3(S):
            for a in self.cur[A]:
                for b in self.cur[B]:
                    for c in self.cur[C]:
                        ca, cb, cc = dict(a.colour), dict(b.colour), dict(c.colour)
                        n = a.namp * b.namp * c.namp
                        add(comm(comm(ca, cb), cc), (1, "S4", 1, a, b, c), n, n)
                        add(comm(comm(ca, cc), cb), (1, "S4", 2, a, b, c), n, n)
                        add(comm(comm(cb, cc), ca), (1, "S4", 3, a, b, c), n, n)
        out = list(groups.values())
        if as_current:
            for i, st in enumerate(out):
                st.name = "J%s_%d" % (self._sname(S), i) if len(out) > 1 else "J%s" % self._sname(S)
                self.struct_order.append(st)
        return out

    # ------------------------------------------------------------------ quark line
    def _L(self, seq):
        """psibar after absorbing the structs in seq from the t end; registers all prefixes."""
        name = "ubar"
        absorbed = frozenset()
        for i, st in enumerate(seq):
            absorbed = absorbed | st.subset
            new = "L_" + "_".join(s.name for s in seq[: i + 1])
            if new not in self.quark_wfs:
                self.quark_wfs[new] = ("L", name, st, absorbed)
            name = new
        return name

    def _R(self, seq):
        """psi after absorbing the structs in seq (given in quark-line order) from the t~ end."""
        name = "v"
        absorbed = frozenset()
        for i in range(len(seq) - 1, -1, -1):
            st = seq[i]
            absorbed = absorbed | st.subset
            new = "R_" + "_".join(s.name for s in seq[i:])
            if new not in self.quark_wfs:
                self.quark_wfs[new] = ("R", name, st, absorbed)
            name = new
        return name

    def _needed(self, seq, c):
        names = []
        for i in range(1, c + 1):
            names.append("L_" + "_".join(s.name for s in seq[:i]))
        for i in range(c + 1, len(seq)):
            names.append("R_" + "_".join(s.name for s in seq[i:]))
        return names

    def _build_diagrams(self):
        ng = self.ng
        diagrams = []   # (seq of structs) for k >= 2
        for blocks in ordered_set_partitions(range(ng)):
            if len(blocks) == 1:
                continue
            for seq in itertools.product(*[self.cur[b] for b in blocks]):
                diagrams.append(seq)
        # closure choice: local search on the number of distinct quark-line wavefunctions.
        # Start from "close at the largest block" and move one diagram's closure at a time while the
        # total strictly decreases (reference counts per wavefunction).
        diagrams.sort(key=lambda s: -len(s))
        choice = {}
        ref = {}
        for d, seq in enumerate(diagrams):
            c = max(range(len(seq)), key=lambda i: (len(seq[i].subset), -abs(i - (len(seq) - 1) / 2.0 - 0.5)))
            choice[d] = c
            for x in self._needed(seq, c):
                ref[x] = ref.get(x, 0) + 1
        improved = True
        while improved:
            improved = False
            for d, seq in enumerate(diagrams):
                cur_need = self._needed(seq, choice[d])
                freed = sum(1 for x in cur_need if ref[x] == 1)
                best = None
                for c in range(len(seq)):
                    if c == choice[d]:
                        continue
                    need = self._needed(seq, c)
                    added = sum(1 for x in need if ref.get(x, 0) == 0 or (ref.get(x, 0) == 1 and x in cur_need and False))
                    # wavefunctions shared between the old and the new closure stay alive
                    added = sum(1 for x in need if (ref.get(x, 0) - (1 if x in cur_need else 0)) == 0)
                    gain = freed - sum(1 for x in cur_need if ref[x] == 1 and x in need) - added
                    # chain lengths also matter: prefer absorbing small blocks
                    if gain > 0 and (best is None or gain > best[0]):
                        best = (gain, c)
                if best:
                    for x in cur_need:
                        ref[x] -= 1
                    choice[d] = best[1]
                    for x in self._needed(seq, best[1]):
                        ref[x] = ref.get(x, 0) + 1
                    improved = True
        for d, seq in enumerate(diagrams):
            c = choice[d]
            Lname = self._L(seq[:c])
            Rname = self._R(seq[c + 1:])
            col = {(): 1}
            namp, namp4 = 1, 0
            for st in seq:
                col = pmul(col, dict(st.colour))
                namp4 = namp4 * st.namp + namp * st.namp4
                namp = namp * st.namp
            self.closures.append((col, [(1, "FFV", Lname, seq[c], Rname)]))
            self.n_amp += namp
            self.n_amp4 += namp4
        # k = 1: all gluons in one tree, closed with the t t~ current G
        full = self._combine(frozenset(range(ng)), as_current=False)
        for st in full:
            terms = []
            for t in st.terms:
                if t[1] == "V3":
                    terms.append((t[0], "V3G", t[2], t[3]))
                else:
                    terms.append((t[0], "S4G", t[2], t[3], t[4], t[5]))
            self.closures.append((dict(st.colour), terms))
            self.n_amp += st.namp
            self.n_amp4 += st.namp4
        assert self.n_amp4 % 3 == 0
        self.n_diag = self.n_amp - self.n_amp4 + self.n_amp4 // 3

    # ------------------------------------------------------------------ colour matrix
    def colour_matrix(self):
        """C_{st} = sum_{a,i,j} (T^s)_{ij} conj((T^t)_{ij}) with T = lambda/2; returns (numerators, denominator)."""
        lam = np.zeros((8, 3, 3), dtype=complex)
        lam[0][0, 1] = lam[0][1, 0] = 1
        lam[1][0, 1] = -1j; lam[1][1, 0] = 1j
        lam[2][0, 0] = 1; lam[2][1, 1] = -1
        lam[3][0, 2] = lam[3][2, 0] = 1
        lam[4][0, 2] = -1j; lam[4][2, 0] = 1j
        lam[5][1, 2] = lam[5][2, 1] = 1
        lam[6][1, 2] = -1j; lam[6][2, 1] = 1j
        lam[7] = np.diag([1, 1, -2]) / np.sqrt(3)
        T = lam / 2
        ng = self.ng
        nf = len(self.flows)
        strings = np.zeros((nf,) + (8,) * ng + (3, 3), dtype=complex)
        letters = "abcd"
        for f, perm in enumerate(self.flows):
            # (T^{a_perm[0]} T^{a_perm[1]} ...)_{ij} for all colour assignments at once
            spec = ",".join(letters[perm[pos]] + "ijklm"[pos] + "ijklm"[pos + 1] for pos in range(ng))
            spec += "->" + letters[:ng] + "i" + "ijklm"[ng]
            strings[f] = np.einsum(spec, *([T] * ng))
        flat = strings.reshape(nf, -1)
        C = (flat @ flat.conj().T).real
        den = {2: 3, 3: 9, 4: 54}[ng]
        num = np.rint(C * den).astype(int)
        assert np.abs(C * den - num).max() < 1e-9
        return num, den


# ----------------------------------------------------------------------------------------------
# emission (variant "reg": every wavefunction is a local variable; ptxas allocates registers)
# ----------------------------------------------------------------------------------------------
PROC_NAME = {2: "Ggtt", 3: "Ggttg", 4: "Ggttgg"}
FILE_NAME = {2: "gen_ggtt.cuh", 3: "gen_ggttg.cuh", 4: "gen_ggttgg.cuh"}


class Emitter:
    def __init__(self, gen):
        self.g = gen
        self.lines = []
        self.flops_hel = 0
        self.flops_fixed = 0
        # index tables for inverse propagators
        ng = gen.ng
        self.gsets = [S for size in range(2, ng) for S in map(frozenset, itertools.combinations(range(ng), size))]
        self.ik_index = {S: i for i, S in enumerate(self.gsets)}
        self.ik_full = len(self.gsets)
        self.qkeys = []      # ('L'|'R', subset)
        for name, (side, prev, st, absorbed) in gen.quark_wfs.items():
            key = (side, absorbed)
            if key not in self.qkeys:
                self.qkeys.append(key)
        self.iq_index = {k: i for i, k in enumerate(self.qkeys)}

    def w(self, s=""):
        self.lines.append(s)

    def kname(self, S):
        return "K" + "".join(str(g) for g in sorted(S))

    def qname(self, key):
        return "q%s%s" % (key[0], "".join(str(g) for g in sorted(key[1])))

    def emit(self):
        g, w = self.g, self.w
        ng = g.ng
        npar = ng + 2
        name = PROC_NAME[ng]
        num, den = g.colour_matrix()
        nf = len(g.flows)
        w("// GENERATED by paper_2106_12631_b200/gen/qcdgen.py — do not edit.")
        w("// g g -> t t~%s : %d diagrams, %d amplitudes (MG counting), %d colour flows." % (" g" * (ng - 2), g.n_diag, g.n_amp, nf))
        w("// Wavefunctions: %d external, %d off-shell gluon currents, %d off-shell quark lines, 1 t t~ current;" %
          (npar, len(g.struct_order), len(g.quark_wfs)))
        w("// %d closing contractions feeding %d colour-flow updates." %
          (sum(len(c[1]) for c in g.closures), sum(len(c[0]) for c in g.closures)))
        w("// Steps A6-A11 of SURVEY.md §8(a); PAPER.md:33-35.  Gluon ids 0..%d = particles %s." % (ng - 1, g.gl_particle))
        w("#pragma once")
        w('#include "helas.cuh"')
        w("namespace mg {")
        w("struct %s {" % name)
        w("  static constexpr int NHEL = %d;" % (1 << npar))
        w("  static constexpr bool FLIP = true;    // QCD: |M(h)|^2 = |M(-h)|^2 at fixed momenta (me_common.cuh)")
        w("  static constexpr int MINB = %d;   // resident CTAs of 128 threads the register allocation aims at" % {2: 3}.get(ng, 1))
        w("  static constexpr int NPAR = %d;" % npar)
        w("  static constexpr int NFLOW = %d;" % nf)
        w("  static constexpr int NIK = %d;" % (len(self.gsets) + 1))
        w("  static constexpr int NIQ = %d;" % len(self.qkeys))
        w("  template <class T> struct Event { Mom<T> p[NPAR]; T ik[NIK]; T iq[NIQ]; };")
        w("")
        self._emit_momenta_fn()
        self._emit_finish()
        self._emit_helicity(num, den)
        w("};")
        w("}  // namespace mg")
        return "\n".join(self.lines) + "\n", num, den

    def _mom_lines(self, ev="ev.p", T="T"):
        """local momentum definitions used by both finish() and helicity()"""
        g = self.g
        out = []
        for gi in range(g.ng):
            ip = g.gl_particle[gi]
            out.append("    const Mom<T> K%d = %s%s[%d];" % (gi, "" if gi < 2 else "-", ev, ip))
        for S in self.gsets:
            parts = sorted(S)
            # build from the largest already-defined subset
            if len(parts) == 2:
                out.append("    const Mom<T> %s = K%d + K%d;" % (self.kname(S), parts[0], parts[1]))
            else:
                sub = frozenset(parts[:-1])
                out.append("    const Mom<T> %s = %s + K%d;" % (self.kname(S), self.kname(sub), parts[-1]))
        out.append("    const Mom<T> pt = %s[2], ptb = %s[3];" % (ev, ev))
        for key in self.qkeys:
            # quark-line momenta counted from the t end (q = p_t - gluons absorbed on the way to t~), as in the plain
            # definition: the same function of the inputs also when they conserve momentum only to
            # FP32 rounding
            side, S = key
            S = S if side == "L" else frozenset(range(g.ng)) - S
            kn = self.kname(S) if len(S) > 1 else "K%d" % sorted(S)[0]
            out.append("    const Mom<T> %s = pt - %s;" % (self.qname(key), kn))
        return [l.replace("Mom<T>", "Mom<%s>" % T) for l in out]

    def _emit_momenta_fn(self):
        pass

    def _emit_finish(self):
        w = self.w
        w("  // helicity-independent part: inverse propagator denominators.  Always evaluated in double")
        w("  // (also for T = float): k_i.k_j cancels like 1/theta^2 for collinear pairs, and this is once per")
        w("  // event, not once per helicity (DESIGN.md R19 / mixed precision).")
        w("  template <class T> static MG_HD void finish(Event<T>& ev, const Consts& k) {")
        w("    Mom<double> pd[NPAR];")
        w("    for (int i = 0; i < NPAR; ++i) for (int mu = 0; mu < 4; ++mu) pd[i].v[mu] = (double)ev.p[i].v[mu];")
        for l in self._mom_lines(ev="pd", T="double"):
            w(l)
        w("    const double mt2 = k.mt * k.mt;")
        for S in self.gsets:
            w("    ev.ik[%d] = (T)(1.0 / mdot(%s, %s));" % (self.ik_index[S], self.kname(S), self.kname(S)))
            self.flops_fixed += 8 + 4 * (len(S) - 1)
        w("    { const Mom<double> Kf = %s; ev.ik[%d] = (T)(1.0 / mdot(Kf, Kf)); }   // t t~ current: all gluon momenta" % (" + ".join("K%d" % gi for gi in range(self.g.ng)), self.ik_full))
        for key in self.qkeys:
            w("    ev.iq[%d] = (T)(1.0 / (mdot(%s, %s) - mt2));" % (self.iq_index[key], self.qname(key), self.qname(key)))
            self.flops_fixed += 13
        w("  }")
        w("")

    def _cur_term(self, t, first):
        init = "true" if first else "false"
        sg = "(T)%d" % t[0]
        if t[1] == "V3":
            a, b = t[2], t[3]
            self.flops_hel += F_VVV_CUR - (4 if first else 0)
            return "vvv_cur<T, %s>(acc, %s, %s, %s, %s, %s);" % (init, sg, a.name, self._k(a), b.name, self._k(b))
        which, a, b, c = t[2], t[3], t[4], t[5]
        self.flops_hel += F_VVVV_CUR - (8 if first else 0)
        return "vvvv_cur<T, %s>(acc, %s, %d, %s, %s, %s);" % (init, sg, which, a.name, b.name, c.name)

    def _k(self, st):
        return self.kname(st.subset) if len(st.subset) > 1 else "K%d" % sorted(st.subset)[0]

    def _emit_helicity(self, num, den):
        g, w = self.g, self.w
        ng = g.ng
        nf = len(g.flows)
        w("  // |M|^2 of ONE helicity combination, colour summed, without g_s^(2 n_g)/denominator")
        w("  template <class T> static MG_HD T helicity(const Event<T>& ev, int ihel, const Consts& k) {")
        for l in self._mom_lines():
            w(l)
        w("    const T mt = (T)k.mt;")
        w("    // A6: external wavefunctions")
        for gi in range(ng):
            ip = g.gl_particle[gi]
            w("    const Vec4<T> eps%d = polvec<T>(ev.p[%d], (ihel >> %d) & 1 ? 1 : -1, %s);" % (gi, ip, ip, "false" if gi < 2 else "true"))
            self.flops_hel += F_POLVEC
        w("    const Spinor<T> ubar = bar(spinor_u<T>(ev.p[2], mt, (ihel >> 2) & 1 ? 1 : -1));")
        w("    const Spinor<T> v = spinor_v<T>(ev.p[3], mt, (ihel >> 3) & 1 ? 1 : -1);")
        self.flops_hel += 2 * F_SPINOR
        w("    // A7: off-shell gluon currents (merged by colour structure)")
        for st in g.struct_order:
            w("    Vec4<T> %s;" % st.name)
            w("    { Vec4<T> acc;")
            for i, t in enumerate(st.terms):
                w("      " + self._cur_term(t, i == 0))
            w("      %s = scale(ev.ik[%d], acc); }" % (st.name, self.ik_index[st.subset]))
            self.flops_hel += F_SCALE
        w("    // A7: off-shell quark lines")
        for name, (side, prev, st, absorbed) in g.quark_wfs.items():
            key = (side, absorbed)
            fn = "ffv_row_prop" if side == "L" else "ffv_col_prop"
            w("    const Spinor<T> %s = %s(%s, %s, %s, mt, ev.iq[%d]);" % (name, fn, prev, st.name, self.qname(key), self.iq_index[key]))
            self.flops_hel += F_FFV_PROP
        need_g = any(t[1] in ("V3G", "S4G") for c in g.closures for t in c[1])
        if need_g:
            w("    const Vec4<T> G = scale(ev.ik[%d], ff_current(ubar, v));" % self.ik_full)
            self.flops_hel += F_FF_CUR + F_SCALE
        w("    // A8 + A9: amplitudes and colour-flow sums (coefficients +-1)")
        w("    cx<T> jamp[NFLOW];")
        seen = set()
        for col, terms in g.closures:
            exprs = []
            for t in terms:
                sg = "" if t[0] > 0 else "-"
                if t[1] == "FFV":
                    e = "ffv_amp(%s, %s, %s)" % (t[2], t[3].name, t[4])
                    self.flops_hel += F_FFV_AMP
                elif t[1] == "V3G":
                    a, b = t[2], t[3]
                    e = "vvv_amp(%s, %s, %s, %s, G)" % (a.name, self._k(a), b.name, self._k(b))
                    self.flops_hel += F_VVV_AMP
                else:
                    e = "vvvv_amp(%d, %s, %s, %s, G)" % (t[2], t[3].name, t[4].name, t[5].name)
                    self.flops_hel += F_VVVV_AMP
                exprs.append((sg, e))
            w("    { cx<T> a = %s%s;" % (exprs[0][0], exprs[0][1]))
            for sg, e in exprs[1:]:
                w("      a = a %s %s;" % ("-" if sg else "+", e))
                self.flops_hel += 2
            for word, c in sorted(col.items()):
                f = g.flow_index[word]
                assert c in (1, -1)
                if f not in seen:
                    seen.add(f)
                    w("      jamp[%d] = %sa;" % (f, "" if c > 0 else "-"))
                else:
                    w("      jamp[%d] = jamp[%d] %s a;" % (f, f, "+" if c > 0 else "-"))
                    self.flops_hel += 2
            w("    }")
        assert len(seen) == nf
        w("    // A10: colour sum  sum_f C_ff |J_f|^2 + 2 sum_{f<g} C_fg Re(J_f^* J_g),  C = numerators / %d" % den)
        w("    T me = (T)0;")
        for f in range(nf):
            terms_re, terms_im = [], []
            w("    { T zr = (T)%d * jamp[%d].re, zi = (T)%d * jamp[%d].im;" % (num[f][f], f, num[f][f], f))
            self.flops_hel += 2
            for h in range(f + 1, nf):
                if num[f][h] == 0:
                    continue
                w("      zr = fma_<T>((T)%d, jamp[%d].re, zr); zi = fma_<T>((T)%d, jamp[%d].im, zi);" % (2 * num[f][h], h, 2 * num[f][h], h))
                self.flops_hel += 4
            w("      me = fma_<T>(jamp[%d].re, zr, fma_<T>(jamp[%d].im, zi, me)); }" % (f, f))
            self.flops_hel += 4
        w("    return me * (T)%s;" % repr(1.0 / den))
        self.flops_hel += 1
        w("  }")


def generate(ng):
    gen = Generator(ng)
    em = Emitter(gen)
    src, num, den = em.emit()
    return gen, em, src, num, den


EMITTED = (2,)        # one thread per event only for g g -> t t~; g g -> t t~ g (g) use gen/recycle.py


def main():
    table = []
    for ng in (2, 3, 4):
        gen, em, src, num, den = generate(ng)
        if ng in EMITTED:
            with open(os.path.join(CSRC, FILE_NAME[ng]), "w") as f:
                f.write(src)
        table.append((ng, gen, em, num, den))
        print("ng=%d: %d diagrams, %d amplitudes, flops/helicity %d, fixed %d" % (ng, gen.n_diag, gen.n_amp, em.flops_hel, em.flops_fixed))
    # tables: flop tallies and colour matrices
    with open(os.path.join(CSRC, "gen_tables.cuh"), "w") as f:
        f.write("// GENERATED by paper_2106_12631_b200/gen/qcdgen.py — do not edit.\n#pragma once\nnamespace mg {\n")
        for ng, gen, em, num, den in table:
            nf = len(gen.flows)
            f.write("static const int kFlopsPerHelicity_%d = %d;\nstatic const int kFlopsFixed_%d = %d;\n" % (ng, em.flops_hel, ng, em.flops_fixed))
            f.write("static const int kColourDen_%d = %d;\nstatic const int kColourNum_%d[%d] = {%s};\n" %
                    (ng, den, ng, nf * nf, ", ".join(str(int(x)) for x in num.reshape(-1))))
            f.write("static const int kNDiagrams_%d = %d;\nstatic const int kNAmplitudes_%d = %d;\n" % (ng, gen.n_diag, ng, gen.n_amp))
        f.write("}  // namespace mg\n")


if __name__ == "__main__":
    main()
