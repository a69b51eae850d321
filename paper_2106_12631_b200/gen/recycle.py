"""Helicity-recycling back-end of the gg -> t t~ (+ g, + g g) generator (csrc/recycle.cuh).

Input: the diagram list of qcdgen.Generator (wavefunctions shared between diagrams; colour-flow
decomposition).  Output: a PROGRAM for the kernel `sigmakin_recycle_kernel`:

  nodes     every wavefunction as a node with the set of external legs whose helicity it depends on (`dep`);
            a node with b legs has 2^b helicity variants, each computed once per event (a task);
            besides the wavefunctions of the diagram list there are HALF PRODUCTS  Vslash.psi / psibar.Vslash
            (so that a diagram closes as  row spinor . column spinor) and the all-gluon currents (closed with
            the t t~ current G);
  steps     producer steps (groups of nodes of the same kind and the same number of helicity bits, separated by
            __syncthreads()) interleaved with per-helicity chunks of closures (inner products added into the
            colour-flow sums); chunks bound the number of half products alive at once;
  slots     shared-memory entries assigned by liveness (a node's entries are reused after its last reader);
  tally     the explicit flop count of everything the kernel executes per event.

The same program object is interpreted in numpy by tests/rc_interp.py (CPU check of tables, slots and signs
against the oracle) and written out as CUDA by `emit()`.
"""
import itertools
import os
from collections import OrderedDict

from . import qcdgen
from .qcdgen import (F_FF_CUR, F_FFV_PROP, F_MDOT_VV, F_POLVEC, F_QSLASH, F_ROW_COL, F_SCALE, F_SLASH, F_SLASH_PARTS,
                     F_SPINOR, F_VVV_CUR, F_VVVV_CUR)

CSRC = qcdgen.CSRC
PROC_NAME = {2: "RcGgtt", 3: "RcGgttg", 4: "RcGgttgg"}
FILE_NAME = {2: "gen_rc_ggtt.cuh", 3: "gen_rc_ggttg.cuh", 4: "gen_rc_ggttgg.cuh"}
KINDS = ["POLVEC", "UBAR", "VSP", "VCUR", "ROWPROP", "COLPROP", "FFCUR", "SLASHCOL", "SLASHROW"]
KIND_ID = {k: i for i, k in enumerate(KINDS)}
T_PART, TB_PART = 2, 3
F_SETUP_MOM = 6 * 4 * 2 + 8 + 2      # one line momentum (6 fma x 4) + Minkowski square + mass shift + reciprocal
# the same in the FP64 kernels, where the sum is carried as an unevaluated pair and squared exactly (recycle.cuh
# run_momtab, R30): per component npar x (1 mul + 6 add) two-sums, 6 for the square, 7 for the accumulation;
# mass shift 10; final sum and reciprocal 2 (npar particles in the sum)
def f_setup_mom_dd(npar):
    return 4 * (npar * 7 + 6 + 7) + 10 + 2


class RNode:
    def __init__(self, name, kind, dep, ops=(), **params):
        self.name, self.kind = name, kind
        self.dep = tuple(sorted(dep))
        self.ops = list(ops)            # operand nodes (VCUR: see terms)
        self.params = params            # mom, prop, outgoing, terms
        self.level = 0
        self.born = None                # step that writes it
        self.last = None                # last step that reads it
        self.slot = None                # first shared-memory entry

    @property
    def nbits(self):
        return len(self.dep)

    @property
    def nvar(self):
        return 1 << len(self.dep)

    def operands(self):
        if "terms" in self.params:
            out = []
            for t in self.params["terms"]:
                out.extend(t["ops"])
            return out
        return self.ops

    def local_mask(self, op):
        """which of this node's variant bits select the operand's variant"""
        assert set(op.dep) <= set(self.dep), (self.name, op.name)
        return sum(1 << j for j, p in enumerate(self.dep) if p in op.dep)

    def flops(self):
        k = self.kind
        if k == "POLVEC":
            return F_POLVEC
        if k in ("UBAR", "VSP"):
            return F_SPINOR
        if k == "VCUR":
            f = sum(F_VVV_CUR if t["type"] == 0 else F_VVVV_CUR for t in self.params["terms"])
            return f + (F_SCALE if self.params.get("prop") is not None else 0)
        if k in ("ROWPROP", "COLPROP"):
            return F_FFV_PROP
        if k == "FFCUR":
            return F_FF_CUR + F_SCALE
        if k in ("ROWPROPN", "COLPROPN", "SLASHCOLN", "SLASHROWN"):      # sum of slash products, then at most one propagator
            nt = len(self.params["terms"])
            return nt * (F_SLASH_PARTS + F_SLASH) + 8 * (nt - 1) + (F_QSLASH + F_SCALE if k.endswith("PROPN") else 0)
        return F_SLASH_PARTS + F_SLASH


class Closure:
    def __init__(self, kind, a, b, flows):
        self.kind, self.a, self.b, self.flows = kind, a, b, flows   # kind: 'DOTS' row.col | 'DOTV' vector.vector


def _closure_key(c):
    """order of the closures inside a step: those sharing the second operand adjacent (it is loaded once)"""
    return (c.b.name, c.a.name)


# Launch shape and schedule parameters per number of gluons, tuned on B200 (profiles/r01_c_*):
#   E, MINB, MINB32   events per CTA, resident CTAs per SM in FP64 / FP32
#   EG                events per synchronisation group inside a CTA (divides E)
#   RELAXED           closure steps NOT followed by a barrier: 'auto' = every one whose inputs can be held through the
#                     next producer step without more shared memory; 'all', '0' (none) or a comma list of step indices
#   SLOTS             shared-memory entries per event that still let E x MINB events share an SM (0: schedule minimum)
#   BUDGET            entries of new half products per closure chunk
#   HOIST             producer steps ride with an earlier producer step when that costs no shared memory
#   HPERM             lane bit i of a thread's index within its event carries the helicity of particle HPERM[i]
#   FLIP              helicity-flip symmetry (R35): the last particle's helicity is fixed at -1, one thread per
#                     combination of the OTHER helicities; |M|^2 counts for the combination and its complement
#   PRESUM            wavefunctions that enter the same colour-flow sums with the same partner are added up BEFORE the
#                     inner product: sum_i s_i (R_i . C) = (sum_i s_i R_i) . C, rows first, then columns (_presum)
#   GENB, GENB32      fused path (momenta generated in the kernel): batches of E events whose momenta a CTA generates up front,
#                     side by side on different warps, before it runs them one after the other (FP64, FP32): the wait for
#                     the RAMBO chain is paid once per GENB batches.  g g -> t t~ g FP64: 4.59 -> 4.01 ms per 2^21 events with
#                     2; slower for FP32 (2.51 -> 2.62) and for g g -> t t~ g g (17.8 -> 21.2: the loop over batches costs
#                     1.9 KB of spills there)
#   ORDER             order of the closure classes (indices into the classes sorted by (helicity bits, kind) of their
#                     half product); None = sorted
DEFAULTS = {
    2: dict(E=8, MINB=3, MINB32=3, EG=None, RELAXED='auto', SLOTS=0, BUDGET=240, HOIST=True, HPERM="2301", ORDER=None, FLIP=False, PRESUM=False, GENB=1, GENB32=1),
    # FLIP (round 2): one warp (g g -> t t~ g g) / half a warp (g g -> t t~ g) per event, 16 / 32 events per SM.  Without it the
    # tuned shapes were E=4, MINB=4/5, HPERM="23104" and E=4, MINB=2/3, SLOTS=424, HPERM="320145", ORDER=(0, 3, 1, 2)
    # (27.2 ms per 2^20 g g -> t t~ g g events against 17.1 ms; shapes and all 120 / 24 lane orders timed:
    # profiles/r02_h_shapes_and_lane_orders.md)
    # g g -> t t~ g: 96 entries in 6 steps instead of 112 in 4 (BUDGET) so that 32 instead of 24 events fit an SM in FP64, as 2 CTAs
    # of 16 events: 4.39 -> 3.71 ms per 2^21 events (FP32, 4 CTAs: 2.59 -> 2.35); profiles/r02_h_shapes_and_lane_orders.md
    3: dict(E=16, MINB=2, MINB32=4, EG=None, RELAXED='auto', SLOTS=0, BUDGET=64, HOIST=True, HPERM="2310", ORDER=None, FLIP=True, PRESUM=False, GENB=2, GENB32=1),
    4: dict(E=8, MINB=2, MINB32=3, EG=None, RELAXED='auto', SLOTS=0, BUDGET=96, HOIST=True, HPERM="32410", ORDER=None, FLIP=True, PRESUM=True, GENB=1, GENB32=1),
}


class Program:
    def __init__(self, ng, **opts):
        """opts override DEFAULTS[ng] (used by sweeps; the committed kernels are the defaults)."""
        self.ng = ng
        g = self.g = qcdgen.Generator(ng)
        self.npar = ng + 2
        o = dict(DEFAULTS[ng])
        assert set(opts) <= set(o), opts
        o.update(opts)
        self.opts = o
        self.E, self.MINB, self.MINB32 = o["E"], o["MINB"], o["MINB32"]
        self.EG = o["EG"] or self.E
        assert self.E % self.EG == 0
        self.RELAXED = o["RELAXED"]
        self.SLOT_LIMIT = o["SLOTS"]
        self.flip = bool(o["FLIP"])
        self.fixed = self.npar - 1 if self.flip else None       # particle whose helicity is not a thread index bit
        self.nhel = 1 << (self.npar - (1 if self.flip else 0))    # threads per event
        self.NT = self.E * self.nhel
        self.gp = g.gl_particle
        self._build_momenta()
        self._build_nodes()
        self._build_closures()
        if o["PRESUM"]:
            self._presum()
        self._schedule(o["BUDGET"])
        if self.RELAXED == 'auto':
            self.RELAXED = '0'
            self._allocate()
            base, chosen = self.nslot, []
            for si, (kind, _) in enumerate(self.steps[:-1]):
                if kind == "F":
                    self.RELAXED = ",".join(map(str, chosen + [si]))
                    self._allocate()
                    if self.nslot <= max(base, self.SLOT_LIMIT):
                        chosen.append(si)
            self.RELAXED = ",".join(map(str, chosen)) or '0'
        self._allocate()
        self._tally()

    # ------------------------------------------------------------------ momentum table
    def _build_momenta(self):
        g, ng, npar = self.g, self.ng, self.npar
        self.mom_names, self.mom_defs = [], []          # defs: (coefficients[npar], propkind)

        def add(name, coef, kind):
            self.mom_names.append(name)
            self.mom_defs.append((tuple(coef), kind))

        # (the external momenta themselves are not in the table: the external wavefunctions read them directly)
        def kcoef(S):
            c = [0] * npar
            for gi in S:
                c[self.gp[gi]] = 1 if gi < 2 else -1     # all gluon momenta incoming
            return c

        self.kidx = {}
        for size in range(1, ng):
            for S in map(frozenset, itertools.combinations(range(ng), size)):
                self.kidx[S] = len(self.mom_names)
                add("K" + "".join(map(str, sorted(S))), kcoef(S), 1 if size > 1 else 0)
        self.qidx = {}
        for name, (side, prev, st, absorbed) in g.quark_wfs.items():
            key = (side, absorbed)
            if key in self.qidx:
                continue
            # every quark-line momentum is counted from the t end, q = p_t - (gluon momenta absorbed so far on the way to
            # t~), as the plain definition states it (q_m = p_t - sum k): for momenta that conserve
            # 4-momentum only to FP32 rounding, K - p_tbar would be a DIFFERENT function of the inputs, and the difference
            # is amplified by the gauge cancellations of soft and collinear events
            towards_t = absorbed if side == "L" else frozenset(range(ng)) - absorbed
            c = [-x for x in kcoef(towards_t)]
            c[T_PART] += 1
            self.qidx[key] = len(self.mom_names)
            add("q%s%s" % (side, "".join(map(str, sorted(absorbed)))), c, 2)
        self.kf = len(self.mom_names)                    # momentum of the t t~ current = all gluon momenta (same remark)
        add("Kf", kcoef(frozenset(range(ng))), 1)

    # ------------------------------------------------------------------ nodes of the diagram list
    def _build_nodes(self):
        g = self.g
        self.nodes = OrderedDict()

        def add(n):
            assert n.name not in self.nodes
            self.nodes[n.name] = n
            return n

        for gi in range(self.ng):
            add(RNode("eps%d" % gi, "POLVEC", [p for p in [self.gp[gi]] if p != self.fixed], mom=self.gp[gi], outgoing=gi >= 2))
        add(RNode("ubar", "UBAR", [T_PART], mom=T_PART))
        add(RNode("v", "VSP", [TB_PART], mom=TB_PART))
        for st in g.struct_order:
            add(self._vcur(st.name, st, st.terms, prop=self.kidx[st.subset]))
        for name, (side, prev, st, absorbed) in g.quark_wfs.items():
            a, b = self.nodes[prev], self.nodes[st.name]
            q = self.qidx[(side, absorbed)]
            add(RNode(name, "ROWPROP" if side == "L" else "COLPROP", set(a.dep) | set(b.dep), [a, b], mom=q, prop=q))
        add(RNode("G", "FFCUR", [T_PART, TB_PART], [self.nodes["ubar"], self.nodes["v"]], prop=self.kf))

    def _vcur(self, name, st_or_subset, terms, prop):
        subset = st_or_subset.subset if hasattr(st_or_subset, "subset") else st_or_subset
        out = []
        for t in terms:
            if t[1] in ("V3", "V3G"):
                a, b = t[2], t[3]
                out.append(dict(type=0, sign=t[0], ops=[self.nodes[a.name], self.nodes[b.name]],
                                momA=self.kidx[a.subset], momB=self.kidx[b.subset]))
            else:
                which, a, b, c = t[2], t[3], t[4], t[5]
                ops = [self.nodes[a.name], self.nodes[b.name], self.nodes[c.name]]
                # every structure is (X.Y) Z - (Z.Y) X after a permutation (csrc/recycle.cuh vvvv_acc)
                cops = {1: [ops[0], ops[2], ops[1]], 2: ops, 3: [ops[1], ops[0], ops[2]]}[which]
                out.append(dict(type=which, sign=t[0], ops=ops, cops=cops, momA=0, momB=0))
        return RNode(name, "VCUR", [self.gp[gi] for gi in subset if self.gp[gi] != self.fixed], terms=out, prop=prop)

    # ------------------------------------------------------------------ closures as inner products
    def _build_closures(self):
        g = self.g
        self.closures = []
        self.half = OrderedDict()       # half-product and all-gluon nodes
        nfull = 0
        for col, terms in g.closures:
            flows = [(g.flow_index[w], c) for w, c in sorted(col.items())]
            if terms[0][1] == "FFV":
                assert len(terms) == 1 and terms[0][0] == 1
                L, V, R = self.nodes[terms[0][2]], self.nodes[terms[0][3].name], self.nodes[terms[0][4]]
                cdep, rdep = set(V.dep) | set(R.dep), set(L.dep) | set(V.dep)
                if len(cdep) <= len(rdep):
                    key = "W_%s_%s" % (V.name, R.name)
                    if key not in self.half:
                        self.half[key] = RNode(key, "SLASHCOL", cdep, [R, V])
                    self.closures.append(Closure("DOTS", L, self.half[key], flows))
                else:
                    key = "U_%s_%s" % (L.name, V.name)
                    if key not in self.half:
                        self.half[key] = RNode(key, "SLASHROW", rdep, [L, V])
                    self.closures.append(Closure("DOTS", self.half[key], R, flows))
            else:
                key = "JF%d" % nfull
                nfull += 1
                self.half[key] = self._vcur(key, frozenset(range(self.ng)), terms, prop=None)
                self.closures.append(Closure("DOTV", self.half[key], self.nodes["G"], flows))

    # ------------------------------------------------------------------ pre-summed closures
    def _presum(self):
        """The closures add x_c = a_c . b_c into the colour-flow sums, J_f += sum_c s_fc x_c.  For the closures that share
        the operand b, J_f += (sum_a s_f,a a) . b: one inner product per DISTINCT signed sum of rows among the flows instead
        of one per row, and one update per (sum, flow) instead of one per (row, flow).  Applied to the rows of every b, then
        to the columns of every (summed) row, wherever it lowers the number of inner products: for a quark line with two
        gluons on either side of the cut this turns 9 products and 16 updates into 4 and 4 — the colour-ordered sub-currents
        found from the sign tables alone.  A sum is a task like any other (kind SUM: signed sum of stored wavefunctions),
        computed once per event and helicity variant."""
        cl = [(c.a, c.b, OrderedDict(c.flows), c.kind) for c in self.closures]
        sums = OrderedDict()
        for side in (0, 1):
            groups = OrderedDict()
            for a, b, fl, kind in cl:
                key, x = (b, a) if side == 0 else (a, b)
                groups.setdefault(key.name, (key, kind, []))[2].append((x, fl))
            out = []
            for key, kind, items in groups.values():
                byname = dict((x.name, x) for x, _ in items)
                per_flow = OrderedDict()
                for x, fl in items:
                    for fidx, sg in fl.items():
                        u = per_flow.setdefault(fidx, OrderedDict())
                        u[x.name] = u.get(x.name, 0) + sg
                distinct = OrderedDict()
                for fidx in sorted(per_flow):
                    u = dict((n, sg) for n, sg in per_flow[fidx].items() if sg)
                    assert u and all(abs(sg) == 1 for sg in u.values())
                    lead = 1 if u[min(u)] > 0 else -1
                    distinct.setdefault(tuple(sorted((n, sg * lead) for n, sg in u.items())), OrderedDict())[fidx] = lead
                if kind != "DOTS" or len(distinct) >= len(items):     # all-gluon closures: their sums would need every J alive at once
                    for x, fl in items:
                        out.append((x, key, fl, kind) if side == 0 else (key, x, fl, kind))
                    continue
                for combo, fl in distinct.items():
                    if len(combo) == 1:
                        x = byname[combo[0][0]]
                        fl = OrderedDict((fidx, lead * combo[0][1]) for fidx, lead in fl.items())
                    else:
                        if combo not in sums:
                            ops = [byname[n] for n, _ in combo]
                            dep = set()
                            for o in ops:
                                dep |= set(o.dep)
                            sums[combo] = RNode("S%d_%d" % (side, len(sums)), "SUM", dep, ops, signs=[sg for _, sg in combo])
                        x = sums[combo]
                    out.append((x, key, fl, kind) if side == 0 else (key, x, fl, kind))
            cl = out
        # A sum is not stored as a sum of stored wavefunctions: the operation that made its operands is linear, so the sum
        # is ONE task of the same kind with several (spinor, vector, sign) terms — psibar' = [sum_i s_i psibar_i Vslash_i]
        # (qslash + m)/(q^2 - m^2) for rows that share their line momentum, sum_i s_i Vslash_i psi_i for half products —
        # and the operands themselves are dropped where nothing else reads them
        fused_kind = {"ROWPROP": "ROWPROPN", "COLPROP": "COLPROPN", "SLASHCOL": "SLASHCOLN", "SLASHROW": "SLASHROWN"}
        repl = {}
        for node in sums.values():
            kinds = set(o.kind for o in node.ops)
            assert len(kinds) == 1 and kinds <= set(fused_kind), (node.name, kinds)
            k0 = node.ops[0].kind
            par = dict(terms=[dict(type=0, sign=sg, ops=[o.ops[0], o.ops[1]], momA=0, momB=0) for o, sg in zip(node.ops, node.params["signs"])])
            if k0 in ("ROWPROP", "COLPROP"):
                assert len(set((o.params["mom"], o.params["prop"]) for o in node.ops)) == 1, node.name
                par.update(mom=node.ops[0].params["mom"], prop=node.ops[0].params["prop"])
            repl[node.name] = RNode(node.name + "_" + "_".join(o.name for o in node.ops), fused_kind[k0], node.dep, [], **par)
            if k0 in ("SLASHCOL", "SLASHROW"):
                self.half[repl[node.name].name] = repl[node.name]
            else:
                self.nodes[repl[node.name].name] = repl[node.name]
        cl = [(repl.get(a.name, a), repl.get(b.name, b), fl, kind) for a, b, fl, kind in cl]
        used = set()
        for a, b, fl, kind in cl:
            used.update((a.name, b.name))
        for n in list(self.nodes.values()) + list(self.half.values()):
            used.update(o.name for o in n.operands())
        for name in [x for x in self.half if x not in used]:
            del self.half[name]
        for name in [x for x in self.nodes if x not in used]:
            del self.nodes[name]
        self.closures = [Closure(kind, a, b, list(fl.items())) for a, b, fl, kind in cl]
        for c in self.closures:
            assert (c.a.name in self.half) != (c.b.name in self.half), (c.a.name, c.b.name)

    # ------------------------------------------------------------------ steps
    def _schedule(self, budget):
        """Steps = producer steps ('P', nodes) and per-helicity chunks of closures ('F', closures).
        Closures are chunked by the class (helicity bits, kind) of their half product, classes larger than
        `budget` entries are split; every node is produced as late as possible (just before the first chunk
        that needs it), which bounds the shared memory alive at once; independent producer steps are merged."""
        for n in self.nodes.values():
            n.level = 1 + max([o.level for o in n.operands()], default=-1)

        def new_node(c):
            return c.a if c.a.name in self.half else c.b

        classes = OrderedDict()
        for c in self.closures:
            nn = new_node(c)
            classes.setdefault((nn.nbits, nn.kind), OrderedDict()).setdefault(nn.name, []).append(c)
        chunks, cur, cur_n = [], [], 0
        keys = sorted(classes)
        if self.opts["ORDER"] is not None:
            assert sorted(self.opts["ORDER"]) == list(range(len(keys))), keys
            keys = [keys[i] for i in self.opts["ORDER"]]
        for key in keys:
            names = list(classes[key])
            total = sum(self.half[x].nvar for x in names)
            if total > budget:                              # split a large class into equal parts
                if cur:
                    chunks.append(cur)
                    cur, cur_n = [], 0
                parts = -(-total // budget)
                per = -(-len(names) // parts)
                for i in range(0, len(names), per):
                    chunks.append([c for x in names[i:i + per] for c in classes[key][x]])
                continue
            if cur and cur_n + total > budget:
                chunks.append(cur)
                cur, cur_n = [], 0
            cur = cur + [c for x in names for c in classes[key][x]]
            cur_n += total
        if cur:
            chunks.append(cur)
        self.steps = []
        done = set()
        for ch in chunks:
            hp = OrderedDict()
            for c in ch:
                hp[new_node(c).name] = new_node(c)
            need, stack = OrderedDict(), []
            for c in ch:
                stack += [x for x in (c.a, c.b) if x.name not in self.half]
            for n in hp.values():
                stack += n.operands()
            while stack:
                x = stack.pop()
                if x.name in done or x.name in need:
                    continue
                need[x.name] = x
                stack += x.operands()
            psteps = []
            for lv in sorted({x.level for x in need.values()}):
                psteps.append([x for x in self.nodes.values() if x.name in need and x.level == lv])
            psteps.append(list(hp.values()))
            done.update(need)
            # merge a producer step into the previous one when it reads nothing born there
            for ps in psteps:
                prev = self.steps[-1] if self.steps and self.steps[-1][0] == "P" else None
                if prev is not None and not any(o in prev[1] for x in ps for o in x.operands()):
                    prev[1].extend(ps)
                else:
                    self.steps.append(("P", list(ps)))
            # closures sharing the second operand are adjacent: it is loaded once
            self.steps.append(("F", sorted(ch, key=_closure_key)))
        self._number()
        # HOIST: a producer step whose nodes can all be computed in an earlier producer step (operands born before it)
        # rides with that step when this costs no shared memory: one barrier-separated latency chain fewer
        if self.opts["HOIST"]:
            self.RELAXED_SAVE, self.RELAXED = self.RELAXED, '0'
            self._allocate()
            limit = max(self.nslot, self.SLOT_LIMIT)
            si = 1
            while si < len(self.steps):
                kind, items = self.steps[si]
                moved = False
                if kind == "P":
                    ready = max(o.born for n in items for o in n.operands()) if any(n.operands() for n in items) else -1
                    cands = [sj for sj in range(si - 1, ready, -1) if self.steps[sj][0] == "P"]
                    for sj in cands:
                        trial = [(k, list(it)) for k, it in self.steps]
                        trial[sj][1].extend(items)
                        del trial[si]
                        # two closure steps that become adjacent merge into one
                        merged = []
                        for k, it in trial:
                            if merged and k == "F" and merged[-1][0] == "F":
                                merged[-1] = ("F", sorted(merged[-1][1] + it, key=_closure_key))
                            else:
                                merged.append((k, it))
                        keep = self.steps
                        self.steps = merged
                        self._number()
                        self._allocate()
                        if self.nslot <= limit:
                            moved = True
                            break
                        self.steps = keep
                        self._number()
                if not moved:
                    si += 1
            self.RELAXED = self.RELAXED_SAVE
            self._number()

    def _number(self):
        # birth / last use
        for n in list(self.nodes.values()) + list(self.half.values()):
            n.born = n.last = None
        for si, (kind, items) in enumerate(self.steps):
            if kind == "P":
                for n in items:
                    n.born = si
                    for o in n.operands():
                        o.last = si
            else:
                for c in items:
                    c.a.last = si
                    c.b.last = si
        self.all_nodes = [n for kind, items in self.steps if kind == "P" for n in items]
        assert len(self.all_nodes) == len(self.nodes) + len(self.half)
        for n in self.all_nodes:
            assert n.last is not None and n.last > n.born, n.name
            assert n.nbits <= 4, "the pext table of recycle.cuh covers 4 helicity bits per node"
            for o in n.operands():
                assert o.born < n.born

    def relaxed(self, si):
        if self.steps[si][0] != "F" or not self.RELAXED or self.RELAXED == '0':
            return False
        return self.RELAXED in ('all', '1') or str(si) in self.RELAXED.split(',')

    # ------------------------------------------------------------------ shared-memory entries by liveness
    def _allocate(self):
        live = []          # (slot, size, last)
        self.nslot = 0
        # RELAXED: no barrier between a closure step and the producer step after it, so that producer step must not
        # overwrite what the closure step reads: such entries are held one step longer
        def hold(n):
            return n.last + 1 if self.relaxed(n.last) else n.last
        for n in self.all_nodes:
            live = [iv for iv in live if iv[2] >= n.born]          # entries whose last reader ran in an earlier step are free
            align = min(n.nvar, 8)
            pos = 0
            for s, size, _ in sorted(live):
                if pos + n.nvar <= s:
                    break
                pos = max(pos, (s + size + align - 1) // align * align)
            n.slot = pos
            live.append((pos, n.nvar, hold(n)))
            self.nslot = max(self.nslot, pos + n.nvar)
        self.nslot = (self.nslot + 7) // 8 * 8

    # ------------------------------------------------------------------ flops per event (everything executed)
    def _tally(self):
        self.flops_nodes = sum(n.nvar * n.flops() for n in self.all_nodes)
        self.flops_setup = len(self.mom_defs) * F_SETUP_MOM
        self.flops_setup_dd = len(self.mom_defs) * f_setup_mom_dd(self.npar)
        num, den = self.g.colour_matrix()
        self.num, self.den = num, den
        nf = len(self.g.flows)
        f = 0
        seen = set()
        for c in self.closures:
            f += F_ROW_COL if c.kind == "DOTS" else F_MDOT_VV
            for fl, sg in c.flows:
                if fl in seen:
                    f += 2
                seen.add(fl)
        for a in range(nf):
            f += 2 + 4 + 4 * sum(1 for b in range(a + 1, nf) if num[a][b] != 0)
        f += 1
        self.flops_hel = f
        self.flops_event = self.flops_setup + self.flops_nodes + self.nhel * self.flops_hel + self.nhel + 1

    # ------------------------------------------------------------------ groups of a producer step
    @staticmethod
    def groups(nodes):
        gr = OrderedDict()
        for n in nodes:
            kind = "EXT" if n.kind in ("POLVEC", "UBAR", "VSP") else n.kind     # externals share one divergent warp
            gr.setdefault((kind, n.nbits), []).append(n)
        return gr


# ----------------------------------------------------------------------------------------------
# CUDA emission
# ----------------------------------------------------------------------------------------------
def emit(prog):
    g = prog.g
    ng, npar, nf = prog.ng, prog.npar, len(g.flows)
    name = PROC_NAME[ng]
    tag = name[2:].lower()
    L = []
    w = L.append
    w("// GENERATED by paper_2106_12631_b200/gen/recycle.py — do not edit.")
    w("// g g -> t t~%s with helicity recycling (csrc/recycle.cuh; DESIGN.md §5.4): %d diagrams, %d colour flows;" % (" g" * (ng - 2), g.n_diag, nf))
    w("// %d nodes / %d tasks per event (%d half products or all-gluon currents), %d inner products per helicity," %
      (len(prog.all_nodes), sum(n.nvar for n in prog.all_nodes), len(prog.half), len(prog.closures)))
    w("// %d shared-memory entries per event, %d steps.  Flops per event: %d (setup %d, tasks %d, per helicity %d x %d)." %
      (prog.nslot, len(prog.steps), prog.flops_event, prog.flops_setup, prog.flops_nodes, prog.nhel, prog.flops_hel))
    w("#pragma once")
    w('#include "recycle.cuh"')
    w("namespace mg {")
    # tables: nodes in step/group order
    order, index = [], {}
    for kind, items in prog.steps:
        if kind != "P":
            continue
        for (k, nb), ns in Program.groups(items).items():
            for n in ns:
                index[n.name] = len(order)
                order.append(n)
    terms = []
    w("__constant__ rc::MomDef kRcMom_%s[%d] = {" % (tag, len(prog.mom_defs)))
    for nm, (coef, kind) in zip(prog.mom_names, prog.mom_defs):
        c6 = list(coef) + [0] * (6 - len(coef))
        w("  {{%s}, %d, 0},   // %s" % (", ".join(str(x) for x in c6), kind, nm))
    w("};")
    node_lines = []

    def opw(consumer, x):
        return "0x%08xu" % (x.slot | (4 * consumer.local_mask(x)) << 16)

    for n in order:
        ops = ["0u", "0u"]
        aux, nterm = 0, 0
        if "terms" in n.params:            # VCUR; sums of slash products (type 0: op0 = spinor, op1 = vector)
            aux, nterm = len(terms), len(n.params["terms"])
            for t in n.params["terms"]:
                tops = t["ops"] if t["type"] == 0 else t["cops"]
                o = [opw(n, x) for x in tops] + ["0u"] * (3 - len(tops))
                terms.append("  {%d, %d, %d, 0, %s, {%s}},   // %s: %s" % (0 if t["type"] == 0 else 1, t["momA"], t["momB"],
                             "0x80000000u" if t["sign"] < 0 else "0u", ", ".join(o), n.name, " ".join(x.name for x in tops)))
        else:
            for i, x in enumerate(n.ops):
                ops[i] = opw(n, x)
            if n.kind == "POLVEC":
                aux = 1 if n.params["outgoing"] else 0
            elif n.kind in ("UBAR", "VSP"):
                aux = 2 if n.kind == "UBAR" else 3
        prop = n.params.get("prop")
        node_lines.append("  {%d, %d, %d, %d, %d, {%s}},   // %d %s %s dep %s" % (
            n.slot, -1 if prop is None else prop, n.params.get("mom", 0), aux, nterm,
            ", ".join(ops), index[n.name], n.kind, n.name, "".join(map(str, n.dep))))
    w("__constant__ rc::TermDesc kRcTerm_%s[%d] = {" % (tag, max(1, len(terms))))
    for t in terms or ["  {0, 0, 0, 0, 0u, {0u, 0u, 0u}},"]:
        w(t)
    w("};")
    w("__constant__ rc::NodeDesc kRcNode_%s[%d] = {" % (tag, len(order)))
    for l in node_lines:
        w(l)
    w("};")
    w("struct %s {" % name)
    w("  static constexpr int NPAR = %d, NHEL = %d, NFLOW = %d, E = %d, EG = %d, NT = %d, NTG = %d, MINB = %d, MINB32 = %d;" % (npar, prog.nhel, nf, prog.E, prog.EG, prog.NT, prog.EG * prog.nhel, prog.MINB, prog.MINB32))
    w("  // NHEL = threads per event.  FLIP: the helicity of the last particle is fixed at -1 and every |M|^2 counts for the")
    w("  // combination and its complement (|M(h)|^2 = |M(-h)|^2 at fixed momenta, DESIGN.md R35); NBITS = helicity bits in a thread index")
    w("  static constexpr bool FLIP = %s;" % ("true" if prog.flip else "false"))
    w("  static constexpr int NHEL_FULL = %d, NBITS = %d;" % (1 << npar, npar - (1 if prog.flip else 0)))
    w("  static constexpr int NMOM = %d, NSLOT = %d;" % (len(prog.mom_defs), prog.nslot))
    w("  static constexpr int GENB = %d, GENB32 = %d;   // batches generated up front by a CTA of the fused path (FP64, FP32)" % (prog.opts["GENB"], prog.opts["GENB32"]))
    # lane bit i of a thread's index within its event carries the helicity of particle hperm[i]: t and t~ in the two
    # lowest bits.  Every order of the free particles was built and timed on B200 (profiles/r02_h_shapes_and_lane_orders.md):
    # 17.1 .. 18.4 ms (g g -> t t~ g g), 4.39 .. 4.54 ms (g g -> t t~ g)
    hperm = prog.opts["HPERM"]
    assert sorted(hperm) == [str(i) for i in range(npar) if i != prog.fixed]
    w("  static constexpr unsigned HPERM = 0x%s;   // nibble i: particle whose helicity is bit i of the lane index" % hperm[::-1])
    w("  static __device__ __forceinline__ const rc::NodeDesc& node(int i) { return kRcNode_%s[i]; }" % tag)
    w("  static __device__ __forceinline__ const rc::TermDesc& term(int i) { return kRcTerm_%s[i]; }" % tag)
    w("  static __device__ __forceinline__ rc::MomDef momdef(int i) { return kRcMom_%s[i]; }" % tag)
    w("")
    w("  // producer steps and inner products (A6-A9): the colour-flow sums J_f of helicity h of event el")
    w("  template <class T, class SM> static __device__ __forceinline__ void amplitudes(const SM& s, int tid, int el, int h, T mt, cx<T> (&jamp)[NFLOW]) {")
    w("    const typename SM::VW ev = s.view(el);")
    w("    const int grp = tid / NTG, gt = tid - grp * NTG, eb = grp * EG;   // synchronisation group, thread in it, its first event")
    seen = set()
    for si, (kind, items) in enumerate(prog.steps):
        if kind == "P":
            gr = Program.groups(items)
            bounds, b = [], 0
            if si == 0:                                   # line momenta and propagators ride with the external wavefunctions
                cnt = prog.EG * len(prog.mom_defs)
                bounds.append(("MOMTAB", 0, 0, 0, 0, (cnt + 31) // 32 * 32))
                b = bounds[0][5]
            for (k, nb), ns in gr.items():
                cnt = len(ns) * (prog.EG << nb)
                pad = (cnt + 31) // 32 * 32
                bounds.append((k, nb, index[ns[0].name], len(ns), b, b + pad))
                b += pad
            w("    // step %d: %s%s" % (si, "momentum table, " if si == 0 else "", ", ".join("%d x %s/%d bits" % (len(ns), k, nb) for (k, nb), ns in gr.items())))
            w("    for (int t = gt; t < %d; t += NTG) {" % b)
            for i, (k, nb, first, nfam, lo, hi) in enumerate(bounds):
                cond = "" if len(bounds) == 1 else ("if (t < %d) " % hi if i == 0 else ("else if (t < %d) " % hi if i < len(bounds) - 1 else "else "))
                if k == "MOMTAB":
                    w("      %src::run_momtab<%s>(s, t, mt, eb);" % (cond, name))
                else:
                    w("      %src::run_group<%s, SM, rc::K_%s, %d>(s, %d, %d, t - %d, mt, eb);" % (cond, name, k, nb, first, nfam, lo))
            w("    }")
            w("    rc::sync_group<%s>(grp);" % name)
        else:
            w("    // step %d: %d inner products" % (si, len(items)))
            cur_b = None
            w("    {")
            # the operand held in registers across consecutive inner products (B) is the one more closures of the step
            # share: fewer shared-memory loads per inner product (both products are symmetric in their operands)
            mult = {}
            for c in items:
                for x in (c.a, c.b):
                    mult[x.name] = mult.get(x.name, 0) + 1
            pairs = []
            for c in items:
                held, other = (c.b, c.a) if mult[c.b.name] >= mult[c.a.name] else (c.a, c.b)
                pairs.append((held, other, c))
            pairs.sort(key=lambda t: (t[0].name, t[1].name))
            for held, other, c in pairs:
                ld_b = "ldv" if c.kind == "DOTV" else "lds"
                typ = "Vec4<T>" if c.kind == "DOTV" else "Spinor<T>"
                if held.name != cur_b:
                    if cur_b is not None:
                        w("      }")
                    w("      { const %s B = ev.%s(%d + rc::pextc<%d>(h));   // %s" % (typ, ld_b, held.slot, _hmask(held), held.name))
                    cur_b = held.name
                fn = "mdot" if c.kind == "DOTV" else "row_col"
                w("        { const cx<T> a = %s(ev.%s(%d + rc::pextc<%d>(h)), B);   // %s" % (fn, ld_b, other.slot, _hmask(other), other.name))
                for fl, sg in c.flows:
                    if fl not in seen:
                        seen.add(fl)
                        w("          jamp[%d] = %sa;" % (fl, "" if sg > 0 else "-"))
                    else:
                        w("          jamp[%d] = jamp[%d] %s a;" % (fl, fl, "+" if sg > 0 else "-"))
                w("        }")
            w("      }")
            w("    }")
            if si != len(prog.steps) - 1 and not prog.relaxed(si):
                w("    rc::sync_group<%s>(grp);" % name)
    assert len(seen) == nf
    num, den = prog.num, prog.den
    w("  }")
    w("")
    w("  // A10: colour sum  sum_f C_ff |J_f|^2 + 2 sum_{f<g} C_fg Re(J_f^* J_g),  C = numerators / %d" % den)
    w("  template <class T> static __device__ __forceinline__ T colour(const cx<T> (&jamp)[NFLOW]) {")
    w("    T me = (T)0;")
    for f in range(nf):
        w("    { T zr = (T)%d * jamp[%d].re, zi = (T)%d * jamp[%d].im;" % (num[f][f], f, num[f][f], f))
        for hh in range(f + 1, nf):
            if num[f][hh] == 0:
                continue
            w("      zr = fma_<T>((T)%d, jamp[%d].re, zr); zi = fma_<T>((T)%d, jamp[%d].im, zi);" % (2 * num[f][hh], hh, 2 * num[f][hh], hh))
        w("      me = fma_<T>(jamp[%d].re, zr, fma_<T>(jamp[%d].im, zi, me)); }" % (f, f))
    w("    return me * (T)%s;" % repr(1.0 / den))
    w("  }")
    w("")
    w("  // |M|^2 of helicity h of event el (no g_s^(2 n_g)/denominator)")
    w("  template <class T, class SM> static __device__ __forceinline__ T run(const SM& s, int tid, int el, int h, T mt) {")
    w("    cx<T> jamp[NFLOW];")
    w("    amplitudes<T, SM>(s, tid, el, h, mt, jamp);")
    w("    return colour<T>(jamp);")
    w("  }")
    w("};")
    w("}  // namespace mg")
    return "\n".join(L) + "\n"


def _hmask(n):
    return sum(1 << p for p in n.dep)


def generate(ng):
    prog = Program(ng)
    return prog, emit(prog)


def tables(progs):
    out = "// GENERATED by paper_2106_12631_b200/gen/recycle.py — do not edit.\n#pragma once\nnamespace mg {\n"
    for ng, prog in progs:
        if ng not in EMITTED:
            continue
        out += "static const long kFlopsRecycle_%d = %d;   // per event: setup %d + tasks %d + %d helicities x %d + reduction\n" % (
            ng, prog.flops_event, prog.flops_setup, prog.flops_nodes, prog.nhel, prog.flops_hel)
        out += "static const long kFlopsRecycleFp64_%d = %d;   // FP64 kernels: setup %d (line momenta squared in double-double)\n" % (
            ng, prog.flops_event - prog.flops_setup + prog.flops_setup_dd, prog.flops_setup_dd)
    return out + "}  // namespace mg\n"


EMITTED = (3, 4)      # g g -> t t~ runs one thread per event (gen_ggtt.cuh): its recycling program is only interpreted by the tests


def main():
    progs = []
    for ng in (2, 3, 4):
        prog, src = generate(ng)
        progs.append((ng, prog))
        if ng not in EMITTED:
            continue
        with open(os.path.join(CSRC, FILE_NAME[ng]), "w") as f:
            f.write(src)
        print("ng=%d: %d nodes, %d tasks/event, %d closures, %d slots (%.1f KB/event FP64), %d steps, flops/event %d (per hel %d)" %
              (ng, len(prog.all_nodes), sum(n.nvar for n in prog.all_nodes), len(prog.closures), prog.nslot,
               prog.nslot * 64 / 1024.0, len(prog.steps), prog.flops_event, prog.flops_hel))
    with open(os.path.join(CSRC, "gen_rc_tables.cuh"), "w") as f:
        f.write(tables(progs))


if __name__ == "__main__":
    main()
