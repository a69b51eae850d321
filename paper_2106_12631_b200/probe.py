"""Binding of libmg_probe.so (include/mg_probe.h): on-box ALU microbenchmarks used by bench.py.  Measurement
tooling, not part of the product library."""
import ctypes as C
import os

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libmg_probe.so")
_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libmg_probe.so not built (run `python -m paper_2106_12631_b200.build`)")
        _lib = C.CDLL(LIB_PATH)
        _lib.mg_probe_alu.restype = C.c_int
        _lib.mg_probe_alu.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double)]
    return _lib


def alu_tflops(precision=0, device=0, mode=0):
    """TFLOP/s of mg_probe_alu: mode 0 = FMA chain, 1 = three distinct register operands, 2 = FP64 mma.sync m8n8k4."""
    v = C.c_double()
    rc = lib().mg_probe_alu(precision, device, mode, C.byref(v))
    if rc != 0:
        raise RuntimeError("mg_probe_alu failed: %d" % rc)
    return v.value
