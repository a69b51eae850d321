"""Pins of oracle/xsec.py (cross-section estimate and unweighting).  CPU only.

The paper prints neither formula nor value, so the pins are textbook closed forms and
properties that any correct hit-or-miss implementation must have:
  * sigma(e+ e- -> mu+ mu-), QED only, tree level, massless:  4 pi alpha^2 / (3 s);
    with the Z: the same angular integral of the closed-form ME of SURVEY.md C5, <t^2> = <u^2> = s^2/3;
  * sigma(g g -> Q Qbar) at LO:  pi alpha_s^2 / (3 s) [ (1 + rho + rho^2/16) ln((1+beta)/(1-beta)) - beta (7/4 + 31 rho/16) ],
    rho = 4 m^2/s (heavy-quark hadroproduction, e.g. Ellis-Stirling-Webber);
  * acceptance of hit-or-miss = <w>/w_max; all kept for w = w_max; none for w = 0; scale invariance;
  * the decision stream is not one of the momentum streams.
"""
import math

import numpy as np
import pytest

import oracle
from oracle import xsec

SQRT_S = 1500.0


def _closed_form_eemumu(par, with_z=True):
    s = par.sqrt_s ** 2
    e2 = 4 * math.pi / par.alpha_em_inv
    sw2 = 1 - par.mW ** 2 / par.mZ ** 2
    cw2 = 1 - sw2
    gl, gr = -0.5 + sw2, sw2
    bw = 1.0 / (sw2 * cw2 * (s - par.mZ ** 2 + 1j * par.mZ * par.gammaZ)) if with_z else 0.0
    amp2 = sum(abs(e2 * (1.0 / s + ga * gb * bw)) ** 2 for ga in (gl, gr) for gb in (gl, gr))
    return xsec.GEV2_TO_PB / (2 * s) * (1 / (8 * math.pi)) * (s * s / 3) * amp2


def test_cross_section_eemumu_closed_form():
    par = oracle.default_params()
    n = 1 << 17
    me, w = oracle.pipeline(0, 7, 0, n, par)
    sigma, err = xsec.cross_section(w * me, par.sqrt_s)
    ref = _closed_form_eemumu(par)
    assert abs(sigma - ref) < 4 * err and err / ref < 5e-3
    # the QED limit of the closed form is the textbook 4 pi alpha^2 / (3 s)
    qed = _closed_form_eemumu(par, with_z=False)
    assert qed == pytest.approx(xsec.GEV2_TO_PB * 4 * math.pi / (3 * par.sqrt_s ** 2 * par.alpha_em_inv ** 2), rel=1e-13)


def test_cross_section_ggtt_closed_form():
    par = oracle.default_params()
    n = 1 << 17
    me, w = oracle.pipeline(1, 7, 0, n, par)
    sigma, err = xsec.cross_section(w * me, par.sqrt_s)
    s = par.sqrt_s ** 2
    rho = 4 * par.mt ** 2 / s
    beta = math.sqrt(1 - rho)
    ref = xsec.GEV2_TO_PB * math.pi * par.alpha_s ** 2 / (3 * s) * (
        (1 + rho + rho * rho / 16) * math.log((1 + beta) / (1 - beta)) - beta * (7 / 4 + 31 * rho / 16))
    assert abs(sigma - ref) < 4 * err and err / ref < 1e-2


def test_weight_sums_are_exactly_rounded():
    w = np.array([1e16, 1.0, -1e16, 3.0, 0.5])           # naive left-to-right summation returns 3.5
    s1, s2, mx = xsec.weight_sums(w)
    assert s1 == 4.5 and mx == 1e16
    assert xsec.weight_sums([]) == (0.0, 0.0, 0.0)
    assert xsec.weight_sums(np.array([2.0, 3.0], dtype=np.float32)) == (5.0, 13.0, 3.0)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_unweighting_acceptance_and_limits(dtype):
    rng = np.random.default_rng(5)
    n = 20000
    w = rng.random(n).astype(dtype)                        # <w> = 1/2
    kept = xsec.unweight(11, 1000, w, 1.0)
    acc = len(kept) / n
    assert abs(acc - w.mean()) < 4 * math.sqrt(0.25 / n)    # acceptance = <w>/w_max
    assert np.all(np.diff(kept) > 0)                        # increasing event order
    assert np.array_equal(xsec.unweight(11, 1000, 4 * w, 4.0), kept)          # scale invariance (powers of two: exact)
    ones = np.ones(50, dtype=dtype)
    assert len(xsec.unweight(3, 0, ones, 1.0)) == 50        # u < 1 strictly: w = w_max is always kept
    assert len(xsec.unweight(3, 0, 0 * ones, 1.0)) == 0
    # the decision depends on the global event index only: splitting the batch changes nothing
    a = xsec.unweight(11, 1000, w[:300], 1.0)
    b = xsec.unweight(11, 1300, w[300:600], 1.0) + 300
    assert np.array_equal(np.concatenate([a, b]), kept[kept < 600])


def test_decision_stream_is_uniform_and_not_a_momentum_stream():
    n = 4096
    u = np.array([xsec.decision_uniform(7, e) for e in range(n)])
    assert 0 < u.min() and u.max() < 1
    assert abs(u.mean() - 0.5) < 4 / math.sqrt(12 * n)
    # Kolmogorov-Smirnov distance to the uniform law
    d = np.abs(np.sort(u) - (np.arange(n) + 0.5) / n).max()
    assert d < 1.95 / math.sqrt(n)
    # none of the (event, particle) words of the momentum streams (R2) coincides with the decision word (R28)
    mom_words = oracle.rng_words(7, 0, 256, 4)[:, :, 0]
    dec_words = np.array([int(oracle.philox4x32_10([e, 0, xsec.UNWEIGHT_SLOT, 0], [7, 0])[0]) for e in range(256)])
    assert not np.any(mom_words == dec_words[:, None])
    # FP32 mapping of R3: 23 bits, strictly inside (0,1)
    u32 = np.array([xsec.decision_uniform(7, e, np.float32) for e in range(512)])
    assert u32.dtype == np.float32 and 0 < u32.min() and u32.max() < 1
    assert np.all(np.abs(u32.astype(np.float64) - u[:512]) < 2.0 ** -23)
