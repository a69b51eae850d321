"""Host logic of the helicity-recycling generator (paper_2106_12631_b200/gen/recycle.py), CPU only.

The PROGRAM the generator writes for `sigmakin_recycle_kernel` (nodes, producer steps, shared-memory slots assigned
by liveness, closures, +-1 colour-flow sums) is executed by the numpy interpreter tests/rc_interp.py
and compared with the oracle (plain colour-ordered recursion, oracle/me_qcd.hpp) on RAMBO events: a wrong operand,
a slot reused too early (the interpreter poisons entries after their last reader), a wrong helicity-variant index
or a wrong sign fails here before any GPU run.  Structural pins: task and closure counts follow from the diagram
counts of SURVEY.md §8(c) C6.
"""
import numpy as np
import pytest

import oracle
import rc_interp
from paper_2106_12631_b200.gen import recycle

SQRT_S = 1500.0


@pytest.fixture(scope="module")
def programs():
    return {ng: recycle.Program(ng) for ng in (2, 3, 4)}


def _events(process, n, seed=7):
    rho = oracle.uniforms(seed, 0, n, oracle.N_FINAL[process])
    mom, w, _ = oracle.rambo(rho, oracle.masses(process), SQRT_S)
    return mom


@pytest.mark.parametrize("ng,n", [(2, 6), (3, 4), (4, 2)])
def test_program_reproduces_the_oracle(programs, ng, n):
    prog = programs[ng]
    par = oracle.default_params()
    process = ng - 1
    mom = _events(process, n)
    ref = oracle.me(process, mom, par)
    gs = np.sqrt(4 * np.pi * par.alpha_s)
    for e in range(n):
        me, per_hel = rc_interp.run(prog, mom[e], par.mt, gs)
        assert abs(me / ref[e] - 1) < 1e-11, (ng, e, me, ref[e])
        assert np.all(per_hel > -1e-30)


@pytest.mark.parametrize("ng,n", [(3, 6), (4, 2)])
def test_program_is_the_same_function_of_momenta_rounded_to_fp32(programs, ng, n):
    """The FP32 kernels get momenta that conserve 4-momentum and sit on their mass shells only to 1e-7.  The
    program (line-momentum routing from the t end, textbook form of the massive spinors) must be the SAME rational
    function of the 4 N input numbers as the plain definition, not one that agrees only on the physical manifold:
    evaluated in double on FP32-rounded momenta it still reproduces the oracle to rounding.  With
    K - p_tbar routing or omega_- = m/omega_+ this fails at the 1e-7 .. 1e-5 level."""
    prog = programs[ng]
    par = oracle.default_params()
    process = ng - 1
    mom = _events(process, n, seed=11).astype(np.float32).astype(np.float64)
    ref = oracle.me(process, mom, par)
    gs = np.sqrt(4 * np.pi * par.alpha_s)
    for e in range(n):
        me, _ = rc_interp.run(prog, mom[e], par.mt, gs)
        assert abs(me / ref[e] - 1) < 1e-10, (ng, e, me / ref[e] - 1)


def test_program_shape(programs):
    # one closure per colour-ordered amplitude of the diagram list: 3 / 18 / 159 amplitudes collapse to
    # 3 / 15 / 105 inner products once diagrams that differ only in a gluon sub-tree share an off-shell current;
    # g g -> t t~ g g: 75 after the rows and columns that enter the same colour-flow sums are added up before the
    # product (PRESUM: the six classes with two gluons on either side of the cut go from 9 products and 16 updates to 4 and 4)
    assert [len(programs[ng].closures) for ng in (2, 3, 4)] == [3, 15, 75]
    assert len(recycle.Program(4, PRESUM=False).closures) == 105
    assert sum(len(c.flows) for c in programs[4].closures) == 264 and sum(len(c.flows) for c in recycle.Program(4, PRESUM=False).closures) == 336
    for ng, prog in programs.items():
        assert prog.nhel == 1 << (ng + 2 - (1 if prog.flip else 0))       # threads per event (FLIP: the last helicity is fixed)
        # every node is written before it is read and its slots lie inside the allocated entries
        for n in prog.all_nodes:
            assert n.born < n.last and n.slot + n.nvar <= prog.nslot
            for o in n.operands():
                assert o.born < n.born and set(o.dep) <= set(n.dep)
        # two nodes alive at the same time never overlap in shared memory (a node owns its entries from the step
        # that writes it to the step of its last reader, both included)
        nodes = prog.all_nodes
        for i, a in enumerate(nodes):
            for b in nodes[i + 1:]:
                if max(a.born, b.born) <= min(a.last, b.last):
                    assert a.slot + a.nvar <= b.slot or b.slot + b.nvar <= a.slot, (a.name, b.name)
        # explicit flop tally: every part is counted
        assert prog.flops_event == prog.flops_setup + prog.flops_nodes + prog.nhel * prog.flops_hel + prog.nhel + 1


def test_generated_sources_are_current(programs):
    import os
    for ng in recycle.EMITTED:
        path = os.path.join(recycle.CSRC, recycle.FILE_NAME[ng])
        assert open(path).read() == recycle.emit(programs[ng]), "run python -m paper_2106_12631_b200.gen.recycle"
