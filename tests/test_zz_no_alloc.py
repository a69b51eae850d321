"""mg_weight_sums_static (include/mg.h): the weight sums of SURVEY.md §8(f) N3 through an entry point that
allocates nothing — its per-CTA partial sums live in a fixed `static __device__` array of csrc/xsec.cu instead of the
handle's scratch region.  For callers that cannot call cudaMalloc (CUDA graph capture, serving loops).

Collected last on purpose (file name): the suite runs with `pytest -x`, and a failure here must not hide another test.
The test passes alone in a fresh process (it builds its own inputs and makes the first call on the device itself) and
after the other tests (the array then holds another call's partials, which must never be read).
"""
import numpy as np
import pytest
import torch

from oracle import xsec

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mg():
    import paper_2106_12631_b200 as m
    from paper_2106_12631_b200 import build
    build.build()
    return m


@pytest.mark.parametrize("prec", [0, 1])
def test_static_weight_sums_equal_the_allocating_path_on_two_calls_in_a_row(mg, prec):
    """Same kernels, same order of additions as mg_weight_sums_async: the three results are equal bit for bit (the
    tolerance of the existing weight-sum tests for the two GPU forms), on two calls in a row that share the array: a
    large batch first, then a smaller one with other weights whose result must not see what the first call left behind;
    then the first again.  The first result is also compared with the exactly rounded sums of oracle/xsec.py (1e-12)."""
    P = mg.Process(1, prec)
    n1, n2 = (1 << 20) + 12345, 70001
    w = torch.empty(mg.padded_stride(n1), dtype=P.dtype, device="cuda")
    ew = torch.empty(mg.padded_stride(n1), dtype=P.dtype, device="cuda")
    P.sigmakin_fused(7, 0, n1, None, w, ew)                      # event weights of g g -> t t~, events 0 .. n1-1
    ew2 = (ew[5000:5000 + n2] * 3.0).contiguous()
    ref1 = P.weight_sums_async(ew, n1).clone()
    ref2 = P.weight_sums_async(ew2, n2).clone()
    out = torch.full((3,), -1.0, dtype=torch.float64, device="cuda")
    got1 = P.weight_sums_static(ew, n1, out).clone()
    got2 = P.weight_sums_static(ew2, n2, out).clone()            # second call in a row, same array, fewer partials
    got3 = P.weight_sums_static(ew, n1, out).clone()
    torch.cuda.synchronize()
    assert torch.equal(got1, ref1) and torch.equal(got2, ref2) and torch.equal(got3, ref1)
    assert not torch.equal(ref1, ref2)
    o1, o2, omx = xsec.weight_sums(ew[:n1].cpu().numpy().astype(np.float64))
    g = got1.cpu().numpy()
    assert abs(g[0] / o1 - 1) < 1e-12 and abs(g[1] / o2 - 1) < 1e-12 and g[2] == omx
    # n == 0 writes zeros; the host-returning form agrees as well
    assert P.weight_sums_static(ew, 0, out).cpu().tolist() == [0.0, 0.0, 0.0]
    assert tuple(P.weight_sums_static(ew, n1, out).cpu().tolist()) == P.weight_sums(ew, n1)


def test_static_weight_sums_limit_and_arguments(mg):
    """Sizes beyond the fixed maximum are refused with MG_ELIMIT and its message; the maximum itself is accepted."""
    P = mg.Process(0, 1)
    nmax = mg.weight_sums_static_max_events()
    assert nmax == 1 << 24
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    wts = torch.rand(nmax + 8, dtype=torch.float32, device="cuda")
    with pytest.raises(mg.MgError, match="-5.*fixed maximum"):
        P.weight_sums_static(wts, nmax + 1, out)
    assert torch.equal(P.weight_sums_static(wts, nmax, out).clone(), P.weight_sums_async(wts, nmax))
    with pytest.raises(mg.MgError, match="-1"):
        P.weight_sums_static(wts, -1, out)
    with pytest.raises(mg.MgError, match="-1"):
        P.weight_sums_static(None, 16, out)
    with pytest.raises(mg.MgError, match="-1"):
        P.weight_sums_static(wts, 16, None)
