"""numpy interpreter of the helicity-recycling PROGRAM written by paper_2106_12631_b200/gen/recycle.py.

Test infrastructure for the HOST logic of the generator: it executes the program's steps exactly as the kernel
does (same task tables, same shared-memory slots with entries poisoned after their last reader, same variant
indexing, same +-1 colour-flow sums) with the reduced vertex rules of csrc/helas.cuh restated in numpy, so that
a mistake in tables, liveness or signs shows up on the CPU against the oracle before any GPU run.  It is not
the oracle and not the product: the product's arithmetic runs only in the CUDA kernels.
"""
import numpy as np

R2 = 0.70710678118654752440


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def polvec(p, lam, outgoing):
    px, py, pz = p[1], p[2], p[3]
    pt2 = px * px + py * py
    cj = -1.0 if outgoing else 1.0
    if pt2 == 0:
        sg = 1.0 if pz >= 0 else -1.0
        return np.array([0, -lam * sg * R2, -1j * cj * R2, 0], dtype=complex)
    ipt, iP = 1 / np.sqrt(pt2), 1 / np.sqrt(pz * pz + pt2)
    ct, st, cp, sp = pz * iP, pt2 * ipt * iP, px * ipt, py * ipt
    return np.array([0, -lam * ct * cp * R2 + 1j * cj * sp * R2, -lam * ct * sp * R2 - 1j * cj * cp * R2, lam * st * R2], dtype=complex)


def chi(p, P, lam):
    px, py, pz = p[1], p[2], p[3]
    pt2 = px * px + py * py
    if pt2 == 0:
        up = (pz >= 0) == (lam > 0)
        return np.array([(1.0 if pz >= 0 else -1.0) if up else 0.0, 0.0 if up else 1.0], dtype=complex)
    Ppz = P + pz if pz >= 0 else pt2 / (P - pz)
    nrm = 1 / np.sqrt(2 * P * Ppz)
    if lam > 0:
        return np.array([Ppz * nrm, (px + 1j * py) * nrm])
    return np.array([(-px + 1j * py) * nrm, Ppz * nrm])


def omegas(E, P, m):
    if m == 0:
        return np.sqrt(2 * P), 0.0
    em = E + m
    return (em + P) / np.sqrt(2 * em), (em - P) / np.sqrt(2 * em)


def spinor_u(p, m, lam):
    P = np.sqrt(p[1] ** 2 + p[2] ** 2 + p[3] ** 2)
    wp, wm = omegas(p[0], P, m)
    x = chi(p, P, lam)
    wl, wr = (wm, wp) if lam > 0 else (wp, wm)
    return np.array([wl * x[0], wl * x[1], wr * x[0], wr * x[1]])


def spinor_v(p, m, lam):
    P = np.sqrt(p[1] ** 2 + p[2] ** 2 + p[3] ** 2)
    wp, wm = omegas(p[0], P, m)
    x = chi(p, P, -lam)
    wl, wr = (wp, -wm) if lam > 0 else (wm, -wp)
    return np.array([wl * x[0], wl * x[1], wr * x[0], wr * x[1]])


def bar(s):
    return np.array([np.conj(s[2]), np.conj(s[3]), np.conj(s[0]), np.conj(s[1])])


def slash_col(V, x):
    p03, m03, p12, m12 = V[0] + V[3], V[0] - V[3], V[1] + 1j * V[2], V[1] - 1j * V[2]
    return np.array([m03 * x[2] - m12 * x[3], -p12 * x[2] + p03 * x[3], p03 * x[0] + m12 * x[1], p12 * x[0] + m03 * x[1]])


def slash_row(V, x):
    p03, m03, p12, m12 = V[0] + V[3], V[0] - V[3], V[1] + 1j * V[2], V[1] - 1j * V[2]
    return np.array([x[2] * p03 + x[3] * p12, x[2] * m12 + x[3] * m03, x[0] * m03 - x[1] * p12, -x[0] * m12 + x[1] * p03])


def ff_current(bq, x):
    a0, a1, b0, b1 = bq
    l0, l1, r0, r1 = x
    return np.array([(a0 * r0 + a1 * r1) + (b0 * l0 + b1 * l1), (a0 * r1 + a1 * r0) - (b0 * l1 + b1 * l0),
                     1j * ((a1 * r0 - a0 * r1) - (b1 * l0 - b0 * l1)), (a0 * r0 - a1 * r1) - (b0 * l0 - b1 * l1)])


def vvv_cur(sign, J1, k1, J2, k2):
    d, e, f = k1 - k2, k1 + 2 * k2, -(2 * k1 + k2)
    return sign * (mdot(J1, J2) * d + mdot(J1, e) * J2 + mdot(J2, f) * J1)


def vvvv_cur(sign, which, A, B, C):
    if which == 1:
        return sign * (mdot(A, C) * B - mdot(B, C) * A)
    if which == 2:
        return sign * (mdot(A, B) * C - mdot(B, C) * A)
    return sign * (mdot(A, B) * C - mdot(A, C) * B)


def pext(v, mask):
    r = j = 0
    for b in range(8):
        if (mask >> b) & 1:
            r |= ((v >> b) & 1) << j
            j += 1
    return r


def run(prog, mom, mt, gs):
    """mom[npar, 4] -> (ME, per-helicity |M|^2 without normalisation) following prog.steps."""
    npar, nhel, nf = prog.npar, prog.nhel, len(prog.g.flows)
    tab = np.array([sum(c * mom[i] for i, c in enumerate(coef)) for coef, _ in prog.mom_defs])
    ip = np.array([0.0 if kind == 0 else 1.0 / (mdot(q, q) - (mt * mt if kind == 2 else 0.0)) for q, (_, kind) in zip(tab, prog.mom_defs)])
    ent = np.full((prog.nslot, 4), np.nan + 0j)
    jamp = np.zeros((nhel, nf), dtype=complex)

    def get(node, consumer_variant, consumer):
        return ent[node.slot + pext(consumer_variant, consumer.local_mask(node))]

    for si, (kind, items) in enumerate(prog.steps):
        if kind == "P":
            out = []
            for n in items:
                for v in range(n.nvar):
                    lam = 1 if v else -1
                    if n.kind == "POLVEC":
                        r = polvec(mom[n.params["mom"]], lam, n.params["outgoing"])
                    elif n.kind == "UBAR":
                        r = bar(spinor_u(mom[n.params["mom"]], mt, lam))
                    elif n.kind == "VSP":
                        r = spinor_v(mom[n.params["mom"]], mt, lam)
                    elif n.kind == "VCUR":
                        r = np.zeros(4, dtype=complex)
                        for t in n.params["terms"]:
                            o = [get(x, v, n) for x in t["ops"]]
                            if t["type"] == 0:
                                r = r + vvv_cur(t["sign"], o[0], tab[t["momA"]], o[1], tab[t["momB"]])
                            else:
                                r = r + vvvv_cur(t["sign"], t["type"], o[0], o[1], o[2])
                        if n.params.get("prop") is not None:
                            r = r * ip[n.params["prop"]]
                    elif n.kind == "ROWPROP":
                        q = tab[n.params["mom"]]
                        r = ip[n.params["prop"]] * (slash_row(q, slash_row(get(n.ops[1], v, n), get(n.ops[0], v, n))) + mt * slash_row(get(n.ops[1], v, n), get(n.ops[0], v, n)))
                    elif n.kind == "COLPROP":
                        q = tab[n.params["mom"]]
                        r = ip[n.params["prop"]] * (slash_col(q, slash_col(get(n.ops[1], v, n), get(n.ops[0], v, n))) + mt * slash_col(get(n.ops[1], v, n), get(n.ops[0], v, n)))
                    elif n.kind == "FFCUR":
                        r = ip[n.params["prop"]] * ff_current(get(n.ops[0], v, n), get(n.ops[1], v, n))
                    elif n.kind in ("ROWPROPN", "COLPROPN", "SLASHCOLN", "SLASHROWN"):
                        # the same operations on a signed sum of slash products (gen/recycle.py _presum)
                        sl = slash_row if n.kind in ("ROWPROPN", "SLASHROWN") else slash_col
                        r = sum(t["sign"] * sl(get(t["ops"][1], v, n), get(t["ops"][0], v, n)) for t in n.params["terms"])
                        if n.kind.endswith("PROPN"):
                            q = tab[n.params["mom"]]
                            r = ip[n.params["prop"]] * (sl(q, r) + mt * r)
                    elif n.kind == "SLASHCOL":
                        r = slash_col(get(n.ops[1], v, n), get(n.ops[0], v, n))
                    elif n.kind == "SLASHROW":
                        r = slash_row(get(n.ops[1], v, n), get(n.ops[0], v, n))
                    else:
                        raise AssertionError(n.kind)
                    assert np.all(np.isfinite(r)), (n.name, v)
                    out.append((n.slot + v, r))
            for i, r in out:                       # all reads of the step happen before its writes become visible
                ent[i] = r
        else:
            for h in range(nhel):
                for c in items:
                    a = ent[c.a.slot + pext(h, sum(1 << p for p in c.a.dep))]
                    b = ent[c.b.slot + pext(h, sum(1 << p for p in c.b.dep))]
                    amp = mdot(a, b) if c.kind == "DOTV" else np.sum(a * b)
                    assert np.isfinite(amp), (c.a.name, c.b.name, h)
                    for fl, sg in c.flows:
                        jamp[h, fl] += sg * amp
        for n in prog.all_nodes:                   # poison what the kernel is allowed to overwrite from now on
            if n.last == si:
                ent[n.slot:n.slot + n.nvar] = np.nan
    C = prog.num / prog.den
    per_hel = np.einsum("hf,fg,hg->h", jamp.conj(), C, jamp).real
    denom = {2: 256, 3: 256, 4: 512}[prog.ng]
    # FLIP programs carry one member of every (h, complement) pair of helicity combinations: each counts twice
    return (2 if getattr(prog, "flip", False) else 1) * per_hel.sum() * gs ** (2 * prog.ng) / denom, per_hel
