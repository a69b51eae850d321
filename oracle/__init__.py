"""ORACLE — test infrastructure only.

ctypes front-end of the plain scalar C++ oracle (oracle/*.hpp).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package; the product (paper_2106_12631_b200) never does.

Arrays are event-major numpy arrays: rho[n, n_final, 4], mom[n, npar, 4] (E, px, py, pz).
Process ids: 0 = e+e- -> mu+mu-, 1 = gg -> tt~, 2 = gg -> tt~g, 3 = gg -> tt~gg, 4 = u u~ -> t t~, 5 = u u~ -> t t~ g.

Parity pins (tests/test_oracle_*.py): Philox KAT vectors; RAMBO closed-form weights, momentum
conservation, on-shellness, 2-body beta/(8 pi); e+e- -> mu+mu- photon+Z closed form and QED limit;
gg -> tt~ heavy-quark closed form; gauge invariance of every partial amplitude; Lorentz invariance;
colour-ordered vs colour-dressed brute force; colour-matrix values; u u~ -> t t~ (g): q q~ -> Q Q~ closed form,
gauge and Lorentz invariance, initial-state collinear limit.  "Event weight" (W_ps * ME) is
a definition with no independent pin: parity unpinned (reading R18).
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

N_FINAL = {0: 2, 1: 2, 2: 3, 3: 4, 4: 2, 5: 3}
N_PAR = {k: v + 2 for k, v in N_FINAL.items()}
DENOM = {0: 4, 1: 256, 2: 256, 3: 512, 4: 36, 5: 36}


class Params(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("sqrt_s", "alpha_em_inv", "mZ", "gammaZ", "mW", "mt", "alpha_s")]


def default_params(**kw):
    """BASELINE.json configs: sqrt(s)=1500, 1/alpha=132.507, mZ=91.188, GammaZ=2.441, mW=80.419, mt=173, alpha_s=0.118."""
    d = dict(sqrt_s=1500.0, alpha_em_inv=132.507, mZ=91.188, gammaZ=2.441, mW=80.419, mt=173.0, alpha_s=0.118)
    d.update(kw)
    return Params(**d)


def masses(process, par=None):
    par = par or default_params()
    m = [0.0] * N_FINAL[process]
    if process >= 1:
        m[0] = m[1] = par.mt
    return np.array(m, dtype=np.float64)


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.oracle_rambo_w0.restype = C.c_double
        _lib.oracle_rambo_w0.argtypes = [C.c_int, C.c_double]
        _lib.oracle_hardware_threads.restype = C.c_int
    return _lib


def _p(a, t=C.c_double):
    return a.ctypes.data_as(C.POINTER(t))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def rng_words(seed, first_event, n, n_final):
    out = np.zeros((n, n_final, 4), dtype=np.uint32)
    lib().oracle_rng_words(C.c_uint64(seed), C.c_uint64(first_event), C.c_int64(n), C.c_int(n_final), _p(out, C.c_uint32))
    return out


def uniforms(seed, first_event, n, n_final, dtype=np.float64):
    out = np.zeros((n, n_final, 4), dtype=dtype)
    if dtype == np.float64:
        lib().oracle_uniforms_f64(C.c_uint64(seed), C.c_uint64(first_event), C.c_int64(n), C.c_int(n_final), _p(out))
    else:
        lib().oracle_uniforms_f32(C.c_uint64(seed), C.c_uint64(first_event), C.c_int64(n), C.c_int(n_final), _p(out, C.c_float))
    return out


def rambo_w0(n_final, sqrt_s):
    return lib().oracle_rambo_w0(n_final, sqrt_s)


def rambo(rho, mass, sqrt_s, long_double=False):
    """rho[n, n_final, 4] (float64) -> (mom[n, n_final+2, 4], weight[n], xi[n])."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    n, nf = rho.shape[0], rho.shape[1]
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    mom = np.zeros((n, nf + 2, 4))
    w = np.zeros(n)
    xi = np.zeros(n)
    lib().oracle_rambo(C.c_int(nf), _p(mass), C.c_double(sqrt_s), _p(rho), C.c_int64(n), _p(mom), _p(w), _p(xi), C.c_int(int(long_double)))
    return mom, w, xi


def me(process, mom, par=None, per_helicity=False, long_double=False, nthreads=0):
    par = par or default_params()
    mom = np.ascontiguousarray(mom, dtype=np.float64)
    n = mom.shape[0]
    assert mom.shape[1:] == (N_PAR[process], 4)
    out = np.zeros(n)
    hel = np.zeros((n, 1 << N_PAR[process])) if per_helicity else None
    nthreads = nthreads or hardware_threads()
    lib().oracle_me(C.c_int(process), C.byref(par), _p(mom), C.c_int64(n), _p(out), _p(hel) if per_helicity else None,
                    C.c_int(int(long_double)), C.c_int(nthreads))
    return (out, hel) if per_helicity else out


def me_dressed(process, mom, par=None, nthreads=0):
    par = par or default_params()
    mom = np.ascontiguousarray(mom, dtype=np.float64)
    n = mom.shape[0]
    out = np.zeros(n)
    lib().oracle_me_dressed(C.c_int(process), C.byref(par), _p(mom), C.c_int64(n), _p(out), C.c_int(nthreads or hardware_threads()))
    return out


def qq_gauge(mom1, par=None):
    """u u~ -> t t~ g: (largest |M| over colours and helicities with eps -> k/k0, the same with physical polarisations)."""
    par = par or default_params()
    mom1 = np.ascontiguousarray(mom1, dtype=np.float64)
    out = np.zeros(2)
    lib().oracle_qq_gauge(C.byref(par), _p(mom1), _p(out))
    return out[0], out[1]


def colour_matrix(ng):
    nperm = int(np.prod(np.arange(1, ng + 1)))
    out = np.zeros((nperm, nperm))
    lib().oracle_colour_matrix(C.c_int(ng), _p(out))
    return out


def partial_amplitudes(process, mom1, ihel, gauge_gluon=-1, par=None, long_double=False):
    par = par or default_params()
    mom1 = np.ascontiguousarray(mom1, dtype=np.float64)
    ng = N_PAR[process] - 2
    nperm = int(np.prod(np.arange(1, ng + 1)))
    out = np.zeros(2 * nperm)
    lib().oracle_partial_amplitudes(C.c_int(process), C.byref(par), _p(mom1), C.c_int(ihel), C.c_int(gauge_gluon), _p(out), C.c_int(int(long_double)))
    return out[0::2] + 1j * out[1::2]


def pipeline(process, seed, first_event, n, par=None, want_momenta=False, nthreads=0):
    """Philox -> RAMBO -> ME for events [first_event, first_event+n) in FP64.  Returns (me, weight[, mom])."""
    par = par or default_params()
    me_out = np.zeros(n)
    w = np.zeros(n)
    mom = np.zeros((n, N_PAR[process], 4)) if want_momenta else None
    lib().oracle_pipeline(C.c_int(process), C.byref(par), C.c_uint64(seed), C.c_uint64(first_event), C.c_int64(n),
                          _p(me_out), _p(w), _p(mom) if want_momenta else None, C.c_int(nthreads or hardware_threads()))
    return (me_out, w, mom) if want_momenta else (me_out, w)


def hardware_threads():
    return max(1, lib().oracle_hardware_threads())
