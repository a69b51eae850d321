"""Host-side checks that need no GPU: libmg_b200.so builds, loads, exports every symbol declared in
include/mg.h, and its argument checking answers before any CUDA call."""
import ctypes as C
import os
import re

import pytest

import paper_2106_12631_b200 as mg
from paper_2106_12631_b200 import build as mg_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    mg_build.build()
    return mg.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mg_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_symbols()
    assert len(names) >= 25
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(mg.EXPORTED) == names


def test_strerror_and_version(lib):
    assert lib.mg_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4):
        assert len(lib.mg_strerror(code)) > 3
    assert b"sm_100a" in lib.mg_version()


def test_padded_stride(lib):
    assert lib.mg_padded_stride(0) == 0
    assert lib.mg_padded_stride(1) == 32
    assert lib.mg_padded_stride(32) == 32
    assert lib.mg_padded_stride(33) == 64
    assert lib.mg_padded_stride(16384) == 16384


def test_default_params_are_the_baseline_configs(lib):
    p = mg.Params()
    assert lib.mg_default_params(mg.GGTTGG, mg.FP32, C.byref(p)) == 0
    assert (p.process, p.precision, p.device) == (3, 1, 0)
    assert (p.sqrt_s, p.alpha_em_inv, p.mZ, p.gammaZ, p.mW, p.mt, p.alpha_s) == (1500.0, 132.507, 91.188, 2.441, 80.419, 173.0, 0.118)
    assert lib.mg_default_params(7, 0, C.byref(p)) == -1
    assert lib.mg_default_params(0, 5, C.byref(p)) == -1
    assert lib.mg_default_params(0, 0, None) == -1


def test_init_argument_checks_come_before_cuda(lib):
    h = C.c_void_p()
    p = mg.default_params(mg.GGTT)
    p.process = 9
    assert lib.mg_init_process(C.byref(p), C.byref(h)) == -1          # MG_EINVAL
    p = mg.default_params(mg.GGTT)
    p.mt = 800.0                                                        # 2 mt >= sqrt_s
    assert lib.mg_init_process(C.byref(p), C.byref(h)) == -2          # MG_EPARAM
    p = mg.default_params(mg.EEMUMU)
    p.sqrt_s = float("nan")
    assert lib.mg_init_process(C.byref(p), C.byref(h)) == -2
    assert lib.mg_init_process(None, C.byref(h)) == -1
    assert lib.mg_free_process(None) == 0


def test_null_handle_is_einval(lib):
    assert lib.mg_n_external(None) == -1
    assert lib.mg_rng(None, 1, 0, 4, 32, None, None) == -1
    assert lib.mg_sigmakin(None, None, 4, 32, None, None, None, None) == -1
    assert lib.mg_flops_per_event(None, 2) == -1


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p()
    p = mg.default_params(mg.EEMUMU)
    assert lib.mg_init_process(C.byref(p), C.byref(h)) == -3          # MG_ECUDA: fails loudly, no fallback
    with pytest.raises(mg.MgError):
        mg.Process("eemumu")


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2106_12631_b200")
    for root, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(root, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "oracle/" not in text, f
