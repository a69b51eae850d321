"""Pins of the oracle's matrix elements.  CPU only.

Each pin is independent of the oracle's own formulation: closed forms from the literature,
invariances, a second brute-force formulation, values printed in SURVEY.md.
"""
import math
import os

import numpy as np
import pytest

import oracle
from inputs import random_lorentz, read_worked_examples, transform

GOLD = os.path.join(os.path.dirname(__file__), "golden")
SQRT_S = 1500.0


def _events(process, n, seed=7, first=0):
    nf = oracle.N_FINAL[process]
    rho = oracle.uniforms(seed, first, n, nf)
    # long-double RAMBO rounded to double: on-shell and momentum-conserving to ~1 ulp, so that
    # closed forms (which assume exact kinematics) can be compared at 1e-13
    mom, w, _ = oracle.rambo(rho, oracle.masses(process), SQRT_S, long_double=True)
    return mom


def _mdot(a, b):
    return a[..., 0] * b[..., 0] - (a[..., 1:] * b[..., 1:]).sum(-1)


# ----------------------------------------------------------------------------- P0
def _eemumu_closed_form(mom, par, with_z=True):
    """ME = (|A_LL|^2+|A_RR|^2) u^2 + (|A_LR|^2+|A_RL|^2) t^2,
    A_ab = e^2 [1/s + g_a g_b/(sW^2 cW^2 (s - mZ^2 + i mZ GZ))]; t=(p_e- - p_mu-)^2, u=(p_e- - p_mu+)^2."""
    e2 = 4 * math.pi / par.alpha_em_inv
    sw2 = 1 - par.mW**2 / par.mZ**2
    cw2 = 1 - sw2
    gl, gr = -0.5 + sw2, sw2
    pep, pem, pmup, pmum = (mom[:, i] for i in range(4))
    s = _mdot(pep + pem, pep + pem)
    t = _mdot(pem - pmum, pem - pmum)
    u = _mdot(pem - pmup, pem - pmup)
    bw = 1.0 / (sw2 * cw2 * (s - par.mZ**2 + 1j * par.mZ * par.gammaZ)) if with_z else 0.0
    A = lambda ga, gb: e2 * (1.0 / s + ga * gb * bw)
    return (abs(A(gl, gl)) ** 2 + abs(A(gr, gr)) ** 2) * u**2 + (abs(A(gl, gr)) ** 2 + abs(A(gr, gl)) ** 2) * t**2


def test_eemumu_photon_plus_z_closed_form():
    par = oracle.default_params()
    mom = _events(0, 2048, seed=42)
    me = oracle.me(0, mom, par)
    ref = _eemumu_closed_form(mom, par)
    assert np.abs(me / ref - 1).max() < 1e-13
    # constants of reading R14/R15
    assert 1 - par.mW**2 / par.mZ**2 == pytest.approx(0.22224653309289089, rel=1e-14)
    assert math.sqrt(4 * math.pi / par.alpha_em_inv) == pytest.approx(0.3079537672443688, rel=1e-14)


def test_eemumu_qed_limit():
    """Z decoupled (mZ -> 1e12 GeV at fixed sW): ME -> 2 e^4 (t^2+u^2)/s^2 (north_star)."""
    par = oracle.default_params(mZ=1.0e12, mW=1.0e12 * math.sqrt(1 - 0.22224653309289089))
    mom = _events(0, 512, seed=42)
    me = oracle.me(0, mom, par)
    e4 = (4 * math.pi / par.alpha_em_inv) ** 2
    pep, pem, pmup, pmum = (mom[:, i] for i in range(4))
    s = _mdot(pep + pem, pep + pem)
    t = _mdot(pem - pmum, pem - pmum)
    u = _mdot(pem - pmup, pem - pmup)
    assert np.abs(me / (2 * e4 * (t * t + u * u) / s**2) - 1).max() < 1e-12


def test_eemumu_at_other_energies_including_z_pole():
    par = oracle.default_params()
    for rs in (91.188, 200.0, 40.0):
        rho = oracle.uniforms(5, 0, 64, 2)
        mom, _, _ = oracle.rambo(rho, np.zeros(2), rs)
        assert np.abs(oracle.me(0, mom, par) / _eemumu_closed_form(mom, par) - 1).max() < 1e-12


def test_eemumu_four_of_sixteen_helicities():
    """only four of the sixteen combinations are allowed."""
    mom = _events(0, 64, seed=42)
    me, hel = oracle.me(0, mom, per_helicity=True)
    share = hel / hel.sum(1, keepdims=True)
    good = (share > 1e-10).any(0)
    assert good.sum() == 4
    # bit k = particle k (e+, e-, mu+, mu-): opposite e+/e- and opposite mu+/mu- helicities
    for h in range(16):
        b = [(h >> k) & 1 for k in range(4)]
        assert good[h] == (b[0] != b[1] and b[2] != b[3])
    assert (share[:, ~good] < 1e-25).all()  # zeros up to rounding (Dirac representation)
    assert np.allclose(hel.sum(1) / 4, me, rtol=1e-15)


# ----------------------------------------------------------------------------- P1
def _ggtt_closed_form(mom, par):
    """Heavy-quark production gg -> QQbar, spin/colour averaged (Ellis-Stirling-Webber, table 10.x form):
    ME = gs^4 (1/(6 t1 t2) - 3/8)(t1^2 + t2^2 + rho - rho^2/(4 t1 t2))."""
    gs4 = (4 * math.pi * par.alpha_s) ** 2
    p1, p2, p3 = mom[:, 0], mom[:, 1], mom[:, 2]
    s = _mdot(p1 + p2, p1 + p2)
    t1 = 2 * _mdot(p1, p3) / s
    t2 = 2 * _mdot(p2, p3) / s
    rho = 4 * par.mt**2 / s
    return gs4 * (1 / (6 * t1 * t2) - 3.0 / 8) * (t1**2 + t2**2 + rho - rho**2 / (4 * t1 * t2))


def test_ggtt_closed_form():
    par = oracle.default_params()
    mom = _events(1, 1024)
    me = oracle.me(1, mom, par)
    assert np.abs(me / _ggtt_closed_form(mom, par) - 1).max() < 1e-12
    assert math.sqrt(4 * math.pi * par.alpha_s) == pytest.approx(1.2177157847767197, rel=1e-14)


def test_ggtt_closed_form_other_mass_and_energy():
    for mt, rs in ((4.7, 100.0), (173.0, 400.0), (500.0, 1500.0)):
        par = oracle.default_params(mt=mt, sqrt_s=rs)
        rho = oracle.uniforms(9, 0, 128, 2)
        mom, _, _ = oracle.rambo(rho, np.array([mt, mt]), rs)
        assert np.abs(oracle.me(1, mom, par) / _ggtt_closed_form(mom, par) - 1).max() < 1e-11


# ----------------------------------------------------------------------------- colour
def test_colour_matrices():
    c2, c3, c4 = (oracle.colour_matrix(n) for n in (2, 3, 4))
    assert np.allclose(c2 * 3, [[16, -2], [-2, 16]], atol=1e-12)
    assert np.allclose(c3[0] * 9, [64, -8, -8, 1, 1, 10], atol=1e-12)
    row = [512, -64, -64, 8, 8, 80, -64, 8, 8, -1, -1, -10, 8, -1, 80, -10, 71, 62, -1, -10, -10, 62, 62, -28]
    assert np.allclose(c4[0] * 54, row, atol=1e-10)
    for n, c in ((2, c2), (3, c3), (4, c4)):
        assert np.allclose(c, c.T, atol=1e-13)
        assert np.allclose(np.diag(c), 3 * (4.0 / 3) ** n, atol=1e-12)  # Nc CF^n
        ev = np.linalg.eigvalsh(c)
        assert ev.min() > 0
        num = np.round(c * 54)
        assert np.abs(c * 54 - num).max() < 1e-9
    assert set(np.unique(np.round(c4 * 54)).astype(int)) == {512, 80, 71, 62, 8, -1, -10, -28, -64}
    ev4 = np.linalg.eigvalsh(c4)
    assert ev4.min() == pytest.approx(3.896, abs=2e-3) and ev4.max() == pytest.approx(14.847, abs=2e-3)


# ----------------------------------------------------------------------------- invariances
@pytest.mark.parametrize("process,nev", [(1, 4), (2, 4), (3, 2)])
def test_gauge_invariance_of_every_partial_amplitude(process, nev):
    """eps_g -> p_g/E_g makes every colour-ordered partial amplitude vanish, for every helicity of the others."""
    mom = _events(process, nev)
    npar = oracle.N_PAR[process]
    ng = npar - 2
    for e in range(nev):
        hels = range(1 << npar) if process < 3 else range(0, 64, 5)
        for h in hels:
            full = np.abs(oracle.partial_amplitudes(process, mom[e], h)).max()
            for g in range(ng):
                a = oracle.partial_amplitudes(process, mom[e], h, gauge_gluon=g)
                ref = max(full, np.abs(oracle.partial_amplitudes(process, mom[e], h ^ 0)).max())
                # scale: the same amplitudes with a physical polarisation (|eps| ~ 1 like p/E)
                scale = max(np.abs(oracle.partial_amplitudes(process, mom[e], hh)).max() for hh in (h, h ^ (1 << [0, 1, 4, 5][g])))
                assert np.abs(a).max() < 1e-10 * scale, (process, e, h, g, np.abs(a).max(), scale, ref)


@pytest.mark.parametrize("process,nev,tol", [(0, 32, 1e-12), (1, 32, 1e-12), (2, 16, 1e-11), (3, 6, 1e-11)])
def test_lorentz_invariance(process, nev, tol):
    """Helicity-summed ME is unchanged under a common rotation+boost of all momenta."""
    mom = _events(process, nev)
    me0 = oracle.me(process, mom)
    for k in range(2):
        lam = random_lorentz(100 + k)
        me1 = oracle.me(process, transform(mom, lam))
        assert np.abs(me1 / me0 - 1).max() < tol


# ----------------------------------------------------------------------------- second formulation
@pytest.mark.parametrize("process,nev", [(1, 8), (2, 3)])
def test_colour_dressed_brute_force_agrees(process, nev):
    mom = _events(process, nev)
    a = oracle.me(process, mom)
    b = oracle.me_dressed(process, mom)
    assert np.abs(a / b - 1).max() < 1e-12


def test_colour_dressed_brute_force_agrees_ggttgg():
    """One gg -> tt~gg event, |M|^2 summed over all 8^4*9 colour assignments with explicit f^{abc}, T^a."""
    mom = _events(3, 1, first=3)
    a = oracle.me(3, mom)
    b = oracle.me_dressed(3, mom)
    assert np.abs(a / b - 1).max() < 1e-12


# ----------------------------------------------------------------------------- helicities, examples
@pytest.mark.parametrize("process,ngood", [(1, 12), (2, 32), (3, 64)])
def test_good_helicity_counts(process, ngood):
    """Reading R16: good iff max over probe events of share > 1e-10.  12/32/64."""
    mom = _events(process, 32 if process < 3 else 8)
    me, hel = oracle.me(process, mom, per_helicity=True)
    share = hel / hel.sum(1, keepdims=True)
    good = (share > 1e-10).any(0)
    assert good.sum() == ngood
    assert np.allclose(hel.sum(1) / oracle.DENOM[process], me, rtol=1e-14)
    if process == 1:
        # (g g t t~) = (+,+,+,-), (+,+,-,+), (-,-,+,-), (-,-,-,+) vanish in the 2 -> 2 CM frame
        bad = {h for h in range(16) if not good[h]}
        assert bad == {0b0111, 0b1011, 0b0100, 0b1000}


def test_worked_examples():
    for ex in read_worked_examples(os.path.join(GOLD, "worked_examples.txt")):
        got = oracle.me(ex["process"], ex["mom"], long_double=True)[0]
        assert got == pytest.approx(ex["me"], rel=1e-12)
        got = oracle.me(ex["process"], ex["mom"])[0]
        assert got == pytest.approx(ex["me"], rel=1e-12)


def test_long_double_and_double_agree():
    for process, n in ((0, 64), (1, 64), (2, 16), (3, 4)):
        mom = _events(process, n)
        a = oracle.me(process, mom)
        b = oracle.me(process, mom, long_double=True)
        assert np.abs(a / b - 1).max() < 1e-12


def test_pipeline_equals_steps():
    for process in (0, 1, 2):
        me, w, mom = oracle.pipeline(process, 7, 100, 16, want_momenta=True)
        rho = oracle.uniforms(7, 100, 16, oracle.N_FINAL[process])
        mom2, w2, _ = oracle.rambo(rho, oracle.masses(process), SQRT_S)
        assert (mom == mom2).all() and (w == w2).all()
        assert (me == oracle.me(process, mom2)).all()
