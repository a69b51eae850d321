"""Pins of the oracle's RNG and phase-space steps.  CPU only."""
import math
import os

import numpy as np
import pytest
from scipy import integrate

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")
SQRT_S = 1500.0


def _hexwords(s):
    return [int(x, 16) for x in s.split()]


def test_philox_known_answer_vectors():
    n = 0
    for line in open(os.path.join(GOLD, "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        lhs, out = line.split("->")
        ctr, key = lhs.split("|")
        got = oracle.philox4x32_10(_hexwords(ctr), _hexwords(key))
        assert [int(x) for x in got] == _hexwords(out)
        n += 1
    assert n == 3


def test_philox_event_particle_mapping():
    for line in open(os.path.join(GOLD, "philox_mapping.txt")):
        if line.startswith("#") or not line.strip():
            continue
        lhs, out = line.split("->")
        seed, ev, ip = [int(x) for x in lhs.split()]
        w = oracle.rng_words(seed, ev, 1, ip + 1)[0, ip]
        assert [int(x) for x in w] == _hexwords(out)
        # same words straight from the block function with the R2 counter/key layout
        w2 = oracle.philox4x32_10([ev & 0xFFFFFFFF, ev >> 32, ip, 0], [seed & 0xFFFFFFFF, seed >> 32])
        assert (w == w2).all()


def test_philox_counter_is_global_event_index():
    a = oracle.rng_words(7, 0, 64, 3)
    b = oracle.rng_words(7, 40, 24, 3)
    assert (a[40:] == b).all()
    hi = oracle.rng_words(7, (1 << 32) + 5, 1, 1)[0, 0]
    assert (hi == oracle.philox4x32_10([5, 1, 0, 0], [7, 0])).all()


def test_uniform_maps_are_exact_and_open():
    w = oracle.rng_words(42, 0, 4096, 2)
    u64 = oracle.uniforms(42, 0, 4096, 2, np.float64)
    u32 = oracle.uniforms(42, 0, 4096, 2, np.float32)
    # (x + 0.5) 2^-32 and ((x>>9) + 0.5) 2^-23 evaluated in exact integer arithmetic
    assert (u64 * 2.0**33 == 2.0 * w.astype(np.float64) + 1.0).all()
    assert (u32.astype(np.float64) * 2.0**24 == 2.0 * (w >> 9).astype(np.float64) + 1.0).all()
    assert u64.min() > 0 and u64.max() < 1 and u32.min() > 0 and u32.max() < 1
    # extreme words
    assert ((0xFFFFFFFF >> 9) + 0.5) * 2.0**-23 < 1.0 and np.float32(((0xFFFFFFFF >> 9) + 0.5) * 2.0**-23) < np.float32(1.0)


def test_rambo_w0_closed_forms():
    # n = 2: two-body massless phase space 1/(8 pi), independent of s
    assert oracle.rambo_w0(2, SQRT_S) == pytest.approx(1 / (8 * math.pi), rel=1e-15)
    assert oracle.rambo_w0(2, 91.0) == pytest.approx(1 / (8 * math.pi), rel=1e-15)
    s = SQRT_S**2
    # n = 3: s/(2^8 pi^3);  n = 4: s^2/(2^13 * 3 * pi^5)  (massless n-body volume)
    assert oracle.rambo_w0(3, SQRT_S) == pytest.approx(s / (256 * math.pi**3), rel=1e-14)
    assert oracle.rambo_w0(4, SQRT_S) == pytest.approx(s * s / (24576 * math.pi**5), rel=1e-14)
    assert oracle.rambo_w0(3, SQRT_S) == pytest.approx(283.4607518542924, rel=1e-13)
    assert oracle.rambo_w0(4, SQRT_S) == pytest.approx(673138.5678286852, rel=1e-13)


@pytest.mark.parametrize("nf", [2, 3, 4])
def test_rambo_massless_invariants(nf):
    rho = oracle.uniforms(7, 0, 4096, nf)
    mom, w, xi = oracle.rambo(rho, np.zeros(nf), SQRT_S)
    assert (xi == 1).all() and np.allclose(w, oracle.rambo_w0(nf, SQRT_S), rtol=1e-15)
    assert (mom[:, 0] == [750, 0, 0, 750]).all() and (mom[:, 1] == [750, 0, 0, -750]).all()
    tot = mom[:, 2:].sum(axis=1)
    assert np.abs(tot - [SQRT_S, 0, 0, 0]).max() < 1e-12 * SQRT_S
    m2 = mom[:, 2:, 0] ** 2 - (mom[:, 2:, 1:] ** 2).sum(-1)
    assert np.abs(m2).max() < 1e-12 * SQRT_S**2
    assert (mom[:, 2:, 0] > 0).all()
    if nf == 2:
        assert np.abs(mom[:, 2:, 0] - SQRT_S / 2).max() < 1e-12 * SQRT_S
    # isotropy: <cos theta> = 0, <pz> = 0 within 5 sigma
    cz = mom[:, 2, 3] / np.sqrt((mom[:, 2, 1:] ** 2).sum(-1))
    assert abs(cz.mean()) < 5 * (1 / math.sqrt(3)) / math.sqrt(len(cz))


@pytest.mark.parametrize("nf", [2, 3, 4])
def test_rambo_massive_invariants(nf):
    m = np.array([173.0, 173.0, 0.0, 0.0][:nf])
    rho = oracle.uniforms(7, 0, 4096, nf)
    mom, w, xi = oracle.rambo(rho, m, SQRT_S)
    tot = mom[:, 2:].sum(axis=1)
    assert np.abs(tot - [SQRT_S, 0, 0, 0]).max() < 1e-12 * SQRT_S
    m2 = mom[:, 2:, 0] ** 2 - (mom[:, 2:, 1:] ** 2).sum(-1)
    assert np.abs(m2 - m**2).max() < 1e-12 * SQRT_S**2
    assert ((xi > 0) & (xi < 1)).all()
    # long-double run agrees
    mom_ld, w_ld, _ = oracle.rambo(rho, m, SQRT_S, long_double=True)
    assert np.abs(mom - mom_ld).max() < 1e-12 * SQRT_S and np.abs(w / w_ld - 1).max() < 1e-12
    if nf == 2:
        beta = math.sqrt(1 - 4 * 173.0**2 / SQRT_S**2)
        # double run: rounding of the massless step is amplified by (Q0/M)^2 <~ 4096 on this sample
        assert np.abs(w / (beta / (8 * math.pi)) - 1).max() < 2e-12
        assert np.abs(w_ld / (beta / (8 * math.pi)) - 1).max() < 2e-15
        assert beta / (8 * math.pi) == pytest.approx(0.038715746184201860, rel=1e-14)


def test_rambo_massless_limit_of_massive():
    rho = oracle.uniforms(3, 0, 256, 3)
    a = oracle.rambo(rho, np.zeros(3), SQRT_S)
    b = oracle.rambo(rho, np.array([1e-9, 1e-9, 0.0]), SQRT_S)
    assert np.abs(a[0] - b[0]).max() < 1e-9 and np.abs(a[1] / b[1] - 1).max() < 1e-12


def _phi2(s, ma, mb):
    lam = (s - (ma + mb) ** 2) * (s - (ma - mb) ** 2)
    return math.sqrt(max(lam, 0.0)) / (8 * math.pi * s)


def _phi3(s, m1, m2, m3):
    f = lambda sp: _phi2(s, math.sqrt(sp), m3) * _phi2(sp, m1, m2) / (2 * math.pi)
    return integrate.quad(f, (m1 + m2) ** 2, (math.sqrt(s) - m3) ** 2, epsabs=0, epsrel=1e-10, limit=200)[0]


def _phi4(s, m1, m2, m3, m4):
    f = lambda sp: _phi2(s, math.sqrt(sp), m4) * _phi3(sp, m1, m2, m3) / (2 * math.pi)
    return integrate.quad(f, (m1 + m2 + m3) ** 2, (math.sqrt(s) - m4) ** 2, epsabs=0, epsrel=1e-9, limit=200)[0]


@pytest.mark.parametrize("nf", [3, 4])
def test_rambo_massive_mean_weight_is_phase_space_volume(nf):
    """<W> over flat RAMBO points = massive n-body phase-space volume, by nested 1-D quadrature of
    the two-body recursion (independent of RAMBO).  Statistical pin, 4 sigma."""
    s = SQRT_S**2
    if nf == 3:
        vol = _phi3(s, 173.0, 173.0, 0.0)
        assert vol == pytest.approx(219.27236, rel=2e-7)
    else:
        vol = _phi4(s, 173.0, 173.0, 0.0, 0.0)
        assert vol == pytest.approx(3.854605e5, rel=2e-6)
    n = 200000
    rho = oracle.uniforms(11, 0, n, nf)
    _, w, _ = oracle.rambo(rho, np.array([173.0, 173.0, 0.0, 0.0][:nf]), SQRT_S)
    err = w.std() / math.sqrt(n)
    assert abs(w.mean() - vol) < 4 * err
    assert err / vol < 2e-3
