"""ORACLE — test infrastructure only (see oracle/philox.hpp for the rules): plain numpy / Python restatement of the
two steps that follow the hot path, SURVEY.md §8(f) N3.

Serves PAPER.md:90 (§4: "a fiducial cross section for the collision process and a sample of N_unw unweighted events.
Both results are obtained using Monte Carlo methods, starting from a larger set of N_wgt randomly generated weighted
events ... an event weight, which varies for weighted events, but is a constant equal to +1 for unweighted events")
and PAPER.md:94 (§4: "event unweighting, where data stream compaction should in principle be straight-forward").
The paper gives no formula for either (cross sections and unweighting are future work); the readings
are listed in DESIGN.md:

  R27  cross section at fixed partonic energy:  sigma = <w> / (2 s) * (hbar c)^2,  w = W_ps * ME (R18), flux factor
       1/(2 s) for massless beams, (hbar c)^2 = 0.3893793721e9 pb GeV^2 (CODATA); MC error = sqrt((<w^2>-<w>^2)/n).
  R28  the random number that decides on event e is word 0 of Philox4x32-10 with key = seed and counter
       (event_lo32, event_hi32, 0xFFFFFFFF, 0): the same global event index as the momenta (R2), a particle slot no
       process uses, hence independent of the momenta and of how the batch is split.
  R29  hit-or-miss: event e is kept iff u_e * w_max < w_e, evaluated in the precision of the weights, u_e mapped to
       (0,1) as in R3; kept events are listed in increasing event order (stable compaction) and carry weight +1.

Pins: tests/test_oracle_xsec.py (closed-form total cross sections of e+ e- -> mu+ mu- and g g -> t t~, acceptance
fraction <w>/w_max, limiting cases, independence of the decision stream from the momentum stream).
"""
import math

import numpy as np

from . import philox4x32_10

GEV2_TO_PB = 0.3893793721e9       # (hbar c)^2 in pb GeV^2
UNWEIGHT_SLOT = 0xFFFFFFFF        # counter word 2 of the decision stream (R28)


def weight_sums(w):
    """(sum w, sum w^2, max w) of a batch, exactly rounded sums (math.fsum) of the weights promoted to double."""
    w = np.asarray(w, dtype=np.float64)
    if w.size == 0:
        return 0.0, 0.0, 0.0
    return math.fsum(w.tolist()), math.fsum((w * w).tolist()), float(w.max())


def cross_section(w, sqrt_s):
    """R27: (sigma, MC error) in pb from the event weights of n flat phase-space points."""
    n = len(w)
    s1, s2, _ = weight_sums(w)
    mean = s1 / n
    var = max(s2 / n - mean * mean, 0.0)
    f = GEV2_TO_PB / (2.0 * sqrt_s * sqrt_s)
    return f * mean, f * math.sqrt(var / n)


def decision_uniform(seed, event, dtype=np.float64):
    """R28 + R3: the uniform in (0,1) that decides on the event with GLOBAL index `event`."""
    ctr = [event & 0xFFFFFFFF, (event >> 32) & 0xFFFFFFFF, UNWEIGHT_SLOT, 0]
    key = [seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF]
    x = int(philox4x32_10(ctr, key)[0])
    if np.dtype(dtype) == np.float64:
        return np.float64((x + 0.5) * (1.0 / 4294967296.0))
    return np.float32((np.float32(x >> 9) + np.float32(0.5)) * np.float32(1.0 / 8388608.0))


def unweight(seed, first_event, w, w_max):
    """R29: indices (relative to the batch, increasing) of the events kept by hit-or-miss against w_max."""
    w = np.asarray(w)
    t = w.dtype.type
    wm = t(w_max)
    kept = []
    for e in range(len(w)):
        u = decision_uniform(seed, first_event + e, w.dtype)
        if t(u) * wm < w[e]:               # one rounded product in the weights' precision, then the comparison
            kept.append(e)
    return np.asarray(kept, dtype=np.int64)
