"""Host logic of the kernel generator (paper_2106_12631_b200/gen/qcdgen.py): diagram and amplitude
counts (BASELINE.json configs: 3/16/123 diagrams; 3/18/159 amplitudes), colour
matrices against the oracle's brute force and the values listed in SURVEY.md C6, coefficients +-1,
and that the committed generated sources are what the generator writes."""
import os

import numpy as np
import pytest

import oracle
from paper_2106_12631_b200.gen import qcdgen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def gens():
    return {ng: qcdgen.generate(ng) for ng in (2, 3, 4)}


def test_diagram_and_amplitude_counts(gens):
    assert [gens[ng][0].n_diag for ng in (2, 3, 4)] == [3, 16, 123]
    assert [gens[ng][0].n_amp for ng in (2, 3, 4)] == [3, 18, 159]


def test_gluon_tree_recurrence():
    # off-shell gluon trees over |S| leaves: 1, 1, 4, 25
    g = qcdgen.Generator(4)
    assert sum(3 * (s.namp - s.namp4) + s.namp4 for s in g.cur[frozenset([0, 1])]) == 3 * 1
    assert sum(3 * (s.namp - s.namp4) + s.namp4 for s in g.cur[frozenset([0, 1, 2])]) == 3 * 4
    full = g._combine(frozenset(range(4)), as_current=False)
    assert sum(3 * (s.namp - s.namp4) + s.namp4 for s in full) == 3 * 25


def test_colour_flow_coefficients_are_signs(gens):
    for ng in (2, 3, 4):
        g = gens[ng][0]
        covered = set()
        for col, terms in g.closures:
            assert all(c in (1, -1) for c in col.values())
            assert all(t[0] in (1, -1) for t in terms)
            covered.update(col.keys())
        assert covered == set(g.flows)


@pytest.mark.parametrize("ng", [2, 3, 4])
def test_colour_matrix_matches_oracle_brute_force(gens, ng):
    num, den = gens[ng][3], gens[ng][4]
    C = oracle.colour_matrix(ng)
    assert np.abs(num / den - C).max() < 1e-12
    assert den == {2: 3, 3: 9, 4: 54}[ng]


def test_colour_matrix_first_rows(gens):
    assert gens[2][3].tolist() == [[16, -2], [-2, 16]]
    assert gens[3][3][0].tolist() == [64, -8, -8, 1, 1, 10]
    assert gens[4][3][0].tolist() == [512, -64, -64, 8, 8, 80, -64, 8, 8, -1, -1, -10, 8, -1, 80, -10, 71, 62, -1, -10, -10, 62, 62, -28]


def test_committed_sources_are_current(gens):
    for ng in qcdgen.EMITTED:
        path = os.path.join(ROOT, "paper_2106_12631_b200", "csrc", qcdgen.FILE_NAME[ng])
        assert open(path).read() == gens[ng][2], "run python -m paper_2106_12631_b200.gen.qcdgen"


def test_flop_tally_is_positive_and_ordered(gens):
    f = [gens[ng][1].flops_hel for ng in (2, 3, 4)]
    assert 500 < f[0] < f[1] < f[2] < 40000


# ----------------------------------------------------------------------------- quark-initiated channel (gen/qqgen.py)
def test_quark_channel_colour_matrices_and_sources():
    from paper_2106_12631_b200.gen import qqgen
    num0, den0 = qqgen.colour_matrix(0)
    assert num0.tolist() == [[2]] and den0 == 1                       # sum |T^c_ij T^c_lk|^2 = (N^2 - 1)/4
    num1, den1 = qqgen.colour_matrix(1)
    K = num1 / den1
    assert np.allclose(K, K.T) and np.linalg.matrix_rank(K) == 3       # five diagrams, two commutator relations (below)
    # emission off one line: C_F (N^2 - 1)/4 = 8/3 on the diagonal; three-gluon vertex: N (N^2 - 1)/4 = 6
    assert np.allclose(np.diag(K), [8 / 3] * 4 + [6])
    # [T^a, T^c] = i f^{acb} T^b on either line: the three-gluon tensor is the commutator of the two emission tensors
    C = [c.reshape(-1) for c in qqgen.colour_tensors(1)]
    assert np.abs(C[0] - C[1] - C[4]).max() < 1e-12 and np.abs(C[3] - C[2] + C[4]).max() < 1e-12
    src, tables = qqgen.emit()
    csrc = os.path.join(ROOT, "paper_2106_12631_b200", "csrc")
    assert open(os.path.join(csrc, "gen_qqtt.cuh")).read() == src, "run python -m paper_2106_12631_b200.gen.qqgen"
    assert open(os.path.join(csrc, "gen_qq_tables.cuh")).read() == tables
