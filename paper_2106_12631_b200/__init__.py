"""paper_2106_12631_b200 — thin Python binding of libmg_b200.so (include/mg.h).

Argument marshalling only: every step of the path (Philox, RAMBO, helicity amplitudes, colour sum)
runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams.  There is
no CPU fallback: if the shared library is missing or there is no sm_100 device the calls raise.

Names follow include/mg.h: mg_init_process -> Process(...), mg_rng -> Process.rng, etc.
Layouts (mg.h): SoA with the event index fastest; tensors are [rows, ld] with ld >= n.
"""
import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmg_b200.so")

EEMUMU, GGTT, GGTTG, GGTTGG, QQTT, QQTTG = 0, 1, 2, 3, 4, 5
FP64, FP32 = 0, 1
STAGE_RNG, STAGE_RAMBO, STAGE_SIGMAKIN, STAGE_GENERATE = 0, 1, 2, 3
PROCESS_NAMES = {"eemumu": EEMUMU, "ggtt": GGTT, "ggttg": GGTTG, "ggttgg": GGTTGG, "qqtt": QQTT, "qqttg": QQTTG}


class MgError(RuntimeError):
    pass


class Params(C.Structure):
    _fields_ = [("process", C.c_int32), ("precision", C.c_int32), ("device", C.c_int32), ("reserved", C.c_int32),
                ("sqrt_s", C.c_double), ("alpha_em_inv", C.c_double), ("mZ", C.c_double), ("gammaZ", C.c_double),
                ("mW", C.c_double), ("mt", C.c_double), ("alpha_s", C.c_double)]


_lib = None


def lib():
    """Loads libmg_b200.so (fails loudly if it has not been built: python -m paper_2106_12631_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise MgError("libmg_b200.so not built (run `python -m paper_2106_12631_b200.build`); there is no CPU fallback")
    L = C.CDLL(LIB_PATH)
    vp, i64, u64 = C.c_void_p, C.c_int64, C.c_uint64
    sig = {
        "mg_default_params": (C.c_int, [C.c_int, C.c_int, C.POINTER(Params)]),
        "mg_init_process": (C.c_int, [C.POINTER(Params), C.POINTER(vp)]),
        "mg_free_process": (C.c_int, [vp]),
        "mg_n_external": (C.c_int, [vp]), "mg_n_final": (C.c_int, [vp]), "mg_n_helicities": (C.c_int, [vp]),
        "mg_n_colour_flows": (C.c_int, [vp]), "mg_n_diagrams": (C.c_int, [vp]), "mg_n_amplitudes": (C.c_int, [vp]),
        "mg_me_denominator": (C.c_int, [vp]),
        "mg_colour_matrix": (C.c_int, [vp, C.POINTER(C.c_double)]),
        "mg_padded_stride": (i64, [i64]),
        "mg_rng_words": (C.c_int, [vp, u64, u64, i64, i64, vp, vp]),
        "mg_rng": (C.c_int, [vp, u64, u64, i64, i64, vp, vp]),
        "mg_rambo": (C.c_int, [vp, vp, i64, i64, vp, vp, vp]),
        "mg_generate": (C.c_int, [vp, u64, u64, i64, i64, vp, vp, vp]),
        "mg_filter_helicities": (C.c_int, [vp, vp, i64, i64, C.POINTER(u64), vp]),
        "mg_set_helicity_mask": (C.c_int, [vp, u64]),
        "mg_get_helicity_mask": (C.c_int, [vp, C.POINTER(u64)]),
        "mg_sigmakin": (C.c_int, [vp, vp, i64, i64, vp, vp, vp, vp]),
        "mg_sigmakin_per_helicity": (C.c_int, [vp, vp, i64, i64, vp, vp]),
        "mg_sigmakin_fused": (C.c_int, [vp, u64, u64, i64, vp, vp, vp, vp]),
        "mg_sigmakin_split": (C.c_int, [vp, vp, i64, i64, vp, vp, vp, i64, vp]),
        "mg_weight_sums": (C.c_int, [vp, vp, i64, C.POINTER(C.c_double), vp]),
        "mg_unweight": (C.c_int, [vp, u64, u64, vp, i64, C.c_double, vp, C.POINTER(i64), vp]),
        "mg_sigmakin_host": (C.c_int, [vp, vp, i64, i64, vp]),
        "mg_run_host": (C.c_int, [vp, u64, u64, i64, i64, vp, vp, vp]),
        "mg_flops_per_event": (i64, [vp, C.c_int]),
        "mg_bytes_per_event": (i64, [vp, C.c_int]),
        "mg_last_kernel_ms": (C.c_double, [vp]),
        "mg_weight_sums_async": (C.c_int, [vp, vp, i64, vp, vp]),
        "mg_weight_sums_static": (C.c_int, [vp, vp, i64, vp, vp]),
        "mg_weight_sums_static_max_events": (i64, []),
        "mg_unweight_async": (C.c_int, [vp, u64, u64, vp, i64, C.c_double, vp, vp, vp]),
        "mg_set_fp32_rescue": (C.c_int, [vp, C.c_double]),
        "mg_get_fp32_rescue": (C.c_double, [vp]),
        "mg_last_rescued": (C.c_int, [vp, C.POINTER(i64)]),
        "mg_strerror": (C.c_char_p, [C.c_int]),
        "mg_version": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    _lib = L
    return L


EXPORTED = ["mg_default_params", "mg_init_process", "mg_free_process", "mg_n_external", "mg_n_final", "mg_n_helicities",
            "mg_n_colour_flows", "mg_n_diagrams", "mg_n_amplitudes", "mg_me_denominator", "mg_colour_matrix",
            "mg_padded_stride", "mg_rng_words", "mg_rng", "mg_rambo", "mg_generate", "mg_filter_helicities",
            "mg_set_helicity_mask", "mg_get_helicity_mask", "mg_sigmakin", "mg_sigmakin_per_helicity", "mg_sigmakin_fused", "mg_sigmakin_split", "mg_weight_sums", "mg_unweight",
            "mg_sigmakin_host", "mg_run_host", "mg_flops_per_event", "mg_bytes_per_event", "mg_last_kernel_ms",
            "mg_weight_sums_async", "mg_unweight_async", "mg_weight_sums_static", "mg_weight_sums_static_max_events", "mg_set_fp32_rescue", "mg_get_fp32_rescue", "mg_last_rescued",
            "mg_strerror", "mg_version"]


def _check(rc):
    if rc != 0:
        raise MgError("mg error %d: %s" % (rc, lib().mg_strerror(rc).decode()))


def padded_stride(n):
    return int(lib().mg_padded_stride(n))


def weight_sums_static_max_events():
    """Largest n mg_weight_sums_static accepts (its partial sums live in a fixed device array of the library)."""
    return int(lib().mg_weight_sums_static_max_events())


def default_params(process, precision=FP64, device=0, **kw):
    p = Params()
    _check(lib().mg_default_params(process, precision, C.byref(p)))
    p.device = device
    for k, v in kw.items():
        setattr(p, k, v)
    return p


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(None)


def _stream(device):
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


class Process:
    """Handle of one (process, precision) on one device — mg_init_process / mg_free_process."""

    def __init__(self, process, precision=FP64, device=0, **physics):
        if isinstance(process, str):
            process = PROCESS_NAMES[process]
        self.params = default_params(process, precision, device, **physics)
        self._h = C.c_void_p()
        _check(lib().mg_init_process(C.byref(self.params), C.byref(self._h)))
        self.process, self.precision, self.device = process, precision, torch.device("cuda", device)
        self.dtype = torch.float64 if precision == FP64 else torch.float32
        L = lib()
        self.n_external = L.mg_n_external(self._h)
        self.n_final = L.mg_n_final(self._h)
        self.n_helicities = L.mg_n_helicities(self._h)
        self.n_colour_flows = L.mg_n_colour_flows(self._h)
        self.n_diagrams = L.mg_n_diagrams(self._h)
        self.n_amplitudes = L.mg_n_amplitudes(self._h)
        self.denominator = L.mg_me_denominator(self._h)

    def close(self):
        if self._h:
            lib().mg_free_process(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- allocation helpers (torch owns the memory)
    def empty(self, rows, n, ld=None, dtype=None):
        ld = ld or padded_stride(n)
        return torch.empty((rows, ld), dtype=dtype or self.dtype, device=self.device)

    # ---- stages
    def rng_words(self, seed, first_event, n, out=None):
        out = out if out is not None else self.empty(4 * self.n_final, n, dtype=torch.int32)
        _check(lib().mg_rng_words(self._h, seed, first_event, n, out.shape[1], _ptr(out), _stream(self.device)))
        return out

    def rng(self, seed, first_event, n, out=None):
        out = out if out is not None else self.empty(4 * self.n_final, n)
        _check(lib().mg_rng(self._h, seed, first_event, n, out.shape[1], _ptr(out), _stream(self.device)))
        return out

    def rambo(self, rnd, n, momenta=None, ps_weight=None):
        ld = rnd.shape[1]
        momenta = momenta if momenta is not None else self.empty(4 * self.n_external, n, ld)
        ps_weight = ps_weight if ps_weight is not None else torch.empty(ld, dtype=self.dtype, device=self.device)
        assert momenta.shape[1] == ld
        _check(lib().mg_rambo(self._h, _ptr(rnd), n, ld, _ptr(momenta), _ptr(ps_weight), _stream(self.device)))
        return momenta, ps_weight

    def generate(self, seed, first_event, n, momenta=None, ps_weight=None):
        momenta = momenta if momenta is not None else self.empty(4 * self.n_external, n)
        ld = momenta.shape[1]
        ps_weight = ps_weight if ps_weight is not None else torch.empty(ld, dtype=self.dtype, device=self.device)
        _check(lib().mg_generate(self._h, seed, first_event, n, ld, _ptr(momenta), _ptr(ps_weight), _stream(self.device)))
        return momenta, ps_weight

    def filter_helicities(self, momenta, probe_n=32):
        mask = C.c_uint64()
        _check(lib().mg_filter_helicities(self._h, _ptr(momenta), probe_n, momenta.shape[1], C.byref(mask), _stream(self.device)))
        return mask.value

    def set_helicity_mask(self, mask):
        _check(lib().mg_set_helicity_mask(self._h, mask))

    def helicity_mask(self):
        m = C.c_uint64()
        _check(lib().mg_get_helicity_mask(self._h, C.byref(m)))
        return m.value

    def sigmakin(self, momenta, n, me=None, ps_weight=None, event_weight=None):
        ld = momenta.shape[1]
        me = me if me is not None else torch.empty(ld, dtype=self.dtype, device=self.device)
        _check(lib().mg_sigmakin(self._h, _ptr(momenta), n, ld, _ptr(me), _ptr(ps_weight), _ptr(event_weight), _stream(self.device)))
        return me

    def sigmakin_split(self, momenta, n, me=None, ps_weight=None, event_weight=None, chunk_events=0):
        """mg_sigmakin_split: the same values as sigmakin from two kernels per chunk of events under a CUDA graph."""
        ld = momenta.shape[1]
        me = me if me is not None else torch.empty(ld, dtype=self.dtype, device=self.device)
        _check(lib().mg_sigmakin_split(self._h, _ptr(momenta), n, ld, _ptr(me), _ptr(ps_weight), _ptr(event_weight),
                                       chunk_events, _stream(self.device)))
        return me

    def sigmakin_per_helicity(self, momenta, n, out=None):
        ld = momenta.shape[1]
        out = out if out is not None else self.empty(self.n_helicities, n, ld)
        _check(lib().mg_sigmakin_per_helicity(self._h, _ptr(momenta), n, ld, _ptr(out), _stream(self.device)))
        return out

    def sigmakin_fused(self, seed, first_event, n, me=None, ps_weight=None, event_weight=None):
        """mg_sigmakin_fused: random numbers -> momenta -> matrix element in one pass, momenta never stored."""
        me = me if me is not None else torch.empty(n, dtype=self.dtype, device=self.device)
        _check(lib().mg_sigmakin_fused(self._h, seed, first_event, n, _ptr(me),
                                       _ptr(ps_weight) if ps_weight is not None else None,
                                       _ptr(event_weight) if event_weight is not None else None, _stream(self.device)))
        return me

    def weight_sums(self, weights, n):
        """mg_weight_sums: (sum w, sum w^2, max w) of the first n event weights, in double."""
        out = (C.c_double * 3)()
        _check(lib().mg_weight_sums(self._h, _ptr(weights), n, out, _stream(self.device)))
        return out[0], out[1], out[2]

    def unweight(self, seed, first_event, weights, n, w_max, kept=None):
        """mg_unweight: batch-relative indices of the events kept by hit-or-miss against w_max (int64 tensor view)."""
        kept = kept if kept is not None else torch.empty(max(n, 1), dtype=torch.int64, device=self.device)
        cnt = C.c_int64()
        _check(lib().mg_unweight(self._h, seed, first_event, _ptr(weights), n, float(w_max), _ptr(kept), C.byref(cnt), _stream(self.device)))
        return kept[:cnt.value]

    def weight_sums_async(self, weights, n, out=None):
        """mg_weight_sums_async: (sum w, sum w^2, max w) left on the device (float64[3]); no host synchronisation."""
        out = out if out is not None else torch.empty(3, dtype=torch.float64, device=self.device)
        _check(lib().mg_weight_sums_async(self._h, _ptr(weights), n, _ptr(out), _stream(self.device)))
        return out

    def weight_sums_static(self, weights, n, out):
        """mg_weight_sums_static: mg_weight_sums_async with its partial sums in a fixed device array of the library: no
        allocation anywhere (`out`, float64[3] on the device, is the caller's); n <= weight_sums_static_max_events()."""
        _check(lib().mg_weight_sums_static(self._h, _ptr(weights), n, _ptr(out), _stream(self.device)))
        return out

    def unweight_async(self, seed, first_event, weights, n, w_max, kept=None, count=None):
        """mg_unweight_async: kept indices and their number (int64[1]) left on the device; no host synchronisation."""
        kept = kept if kept is not None else torch.empty(max(n, 1), dtype=torch.int64, device=self.device)
        count = count if count is not None else torch.empty(1, dtype=torch.int64, device=self.device)
        _check(lib().mg_unweight_async(self._h, seed, first_event, _ptr(weights), n, float(w_max), _ptr(kept), _ptr(count), _stream(self.device)))
        return kept, count

    # ---- mixed precision of the FP32 handles of g g -> t t~ g (g)
    def set_fp32_rescue(self, kappa_max):
        _check(lib().mg_set_fp32_rescue(self._h, float(kappa_max)))

    def fp32_rescue(self):
        return float(lib().mg_get_fp32_rescue(self._h))

    def last_rescued(self):
        c = C.c_int64()
        _check(lib().mg_last_rescued(self._h, C.byref(c)))
        return c.value

    # ---- host-buffer (end-to-end) forms; tensors are CPU tensors (pinned for speed)
    def sigmakin_host(self, h_momenta, n, h_me):
        assert not h_momenta.is_cuda and not h_me.is_cuda
        _check(lib().mg_sigmakin_host(self._h, _ptr(h_momenta), n, h_momenta.shape[1], _ptr(h_me)))
        return h_me

    def run_host(self, seed, first_event, n, h_me, h_momenta=None, h_ps_weight=None, ld=None):
        ld = ld or (h_momenta.shape[1] if h_momenta is not None else padded_stride(n))
        _check(lib().mg_run_host(self._h, seed, first_event, n, ld, _ptr(h_momenta), _ptr(h_ps_weight), _ptr(h_me)))
        return h_me

    # ---- roofline bookkeeping
    def flops_per_event(self, stage=STAGE_SIGMAKIN):
        return int(lib().mg_flops_per_event(self._h, stage))

    def bytes_per_event(self, stage):
        return int(lib().mg_bytes_per_event(self._h, stage))

    def last_kernel_ms(self):
        return float(lib().mg_last_kernel_ms(self._h))

    def colour_matrix(self):
        nf = self.n_colour_flows
        buf = (C.c_double * (nf * nf))()
        _check(lib().mg_colour_matrix(self._h, buf))
        return torch.tensor(list(buf), dtype=torch.float64).reshape(nf, nf)
