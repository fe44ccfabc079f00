"""Host logic of the quark-channel generator (gen/quark.py): diagram counts, colour-flow expansion and
the exact colour matrix, the latter against an explicit Gell-Mann contraction written here with numpy (neither the
oracle's code nor the generator's Fierz reduction)."""
from itertools import product

import numpy as np
import pytest

from paper_2312_02898_b200.gen import quark as Q


def gell_mann():
    lam = np.zeros((8, 3, 3), dtype=complex)
    lam[0][0, 1] = lam[0][1, 0] = 1
    lam[1][0, 1], lam[1][1, 0] = -1j, 1j
    lam[2][0, 0], lam[2][1, 1] = 1, -1
    lam[3][0, 2] = lam[3][2, 0] = 1
    lam[4][0, 2], lam[4][2, 0] = -1j, 1j
    lam[5][1, 2] = lam[5][2, 1] = 1
    lam[6][1, 2], lam[6][2, 1] = -1j, 1j
    lam[7] = np.diag([1, 1, -2]) / np.sqrt(3)
    return lam / 2


@pytest.mark.parametrize("k,nterms,ndiag,nflow", [(0, 1, 1, 2), (1, 5, 5, 4), (2, 37, 36, 12)])
def test_diagram_and_flow_counts(k, nterms, ndiag, nflow):
    """1, 5 and 36 Feynman diagrams for q q~ -> t t~ + 0, 1, 2 gluons (any crossing has the same diagrams)."""
    terms = Q.diagram_terms(k)
    assert len(terms) == nterms and Q.n_feynman_diagrams(terms) == ndiag
    fl = Q.flows(k)
    assert len(fl) == nflow == 2 * np.prod(range(1, k + 2))
    index = {f: i for i, f in enumerate(fl)}
    fed = set()
    for t in terms:
        tf = Q.term_flows(t, k, index)
        assert tf and all(abs(s) == 1 for _, s in tf)
        fed.update(f for f, _ in tf)
    assert fed == set(range(nflow))


@pytest.mark.parametrize("k", [0, 1, 2])
def test_colour_matrix_equals_explicit_gell_mann_contraction(k):
    T = gell_mann()

    def string(seq, cols):
        m = np.eye(3, dtype=complex)
        for g in seq:
            m = m @ T[cols[g]]
        return m

    fl = Q.flows(k)
    cf = np.zeros((len(fl), len(fl)), dtype=complex)
    for cols in product(range(8), repeat=k):
        vecs = []
        for kind, s1, s2 in fl:
            a, b = string(s1, cols), string(s2, cols)
            if kind == "L":      # (T^S1)_{i n} (T^S2)_{o l}
                v = np.einsum("in,ol->ilon", a, b)
            else:                # -1/N (T^S1)_{i l} (T^S2)_{o n}
                v = -np.einsum("il,on->ilon", a, b) / 3
            vecs.append(v.ravel())
        v = np.array(vecs)
        cf += v.conj() @ v.T
    want = np.array([[float(x) for x in row] for row in Q.colour_matrix(k)])
    assert np.abs(cf.imag).max() < 1e-12
    assert np.abs(cf.real - want).max() < 1e-12


def test_colour_factor_of_the_born_process():
    """q q~ -> t t~: both flows carry the same amplitude, the colour factor is (N^2 - 1)/4 = 2."""
    cf = Q.colour_matrix(0)
    assert sum(sum(row) for row in cf) / 4 == 2


def test_every_subprocess_is_emitted_with_its_averaging_factor():
    want = {"qQtT": 36, "qQtTg": 36, "qgtTq": 96, "gQtTQ": 96, "qQtTgg": 72, "qgtTqg": 96, "ggtTqQ": 256}
    for spec in Q.SPECS:
        qp = Q.QProcess(spec)
        if spec in want:
            assert qp.denominator == want[spec]
    files, info = Q.emit_quark("qgtTqg")
    assert info["ndiagrams"] == 36 and info["ncol"] == 12 and info["proc"] == "q g > t t~ q g"
    assert "cur_pair" in files[0][1] and "mg_desc_qgttxqg" in files[0][1]


# ------------------------------------------------------------------------------------------- two light-quark lines
def test_two_line_term_colours_equal_the_explicit_gell_mann_tensors():
    """Each of the seven terms: sum over the pseudo-gluon colours of the T-strings on the three open lines (numpy, explicit
    Gell-Mann matrices) against the generator's Fierz-reduced combination of Kronecker deltas."""
    from paper_2312_02898_b200.gen import quark2 as Q2
    T = gell_mann()
    rows, cols = ("t", "e0", "e1"), ("T", "s0", "s1")
    eye = np.eye(3)
    for kind, strings in Q2.terms():
        want = np.zeros((3,) * 6, dtype=complex)           # indices: t, T, e0, s0, e1, s1
        for sign, top, l0, l1 in strings:
            for x0 in range(8):
                for x1 in range(8):
                    lab = {"P0": T[x0], "P1": T[x1]}

                    def mat(s):
                        m = eye.astype(complex)
                        for a in s:
                            m = m @ lab[a]
                        return m

                    want += sign * np.einsum("ab,cd,ef->abcdef", mat(top), mat(l0), mat(l1))
        got = np.zeros((3,) * 6, dtype=complex)
        pos = {"t": 0, "T": 1, "e0": 2, "s0": 3, "e1": 4, "s1": 5}
        for flow, coef in Q2.term_colour(strings, rows, cols, rows).items():
            letters = "abcdef"
            ops = []
            for r, c in zip(rows, flow):
                ops.append(letters[pos[r]] + letters[pos[c]])
            got += float(coef) * np.einsum("%s,%s,%s->abcdef" % tuple(ops), eye, eye, eye)
        assert np.abs(got - want).max() < 1e-12, kind


def test_two_line_flow_matrix_and_processes():
    from paper_2312_02898_b200.gen import quark2 as Q2
    rows = ("t", "e0", "e1")
    from itertools import permutations
    flows = list(permutations(("T", "s0", "s1")))
    cf = np.array(Q2.flow_matrix(flows, rows))
    assert cf.shape == (6, 6) and np.all(np.diag(cf) == 27) and set(cf.ravel()) == {3, 9, 27}
    assert np.array_equal(cf, cf.T) and np.linalg.matrix_rank(cf) == 6
    assert Q2.QProcess2("qQtTrR").denominator == 36 and Q2.QProcess2("qqtTqq").denominator == 72
    assert len(Q2.QProcess2("qQtTqQ").pairings) == 2 and len(Q2.QProcess2("qrtTqr").pairings) == 1
    files, info = Q2.emit_quark2("qQtTqQ")
    assert info["ndiagrams"] == 14 and info["ncol"] == 6 and info["proc"] == "q q~ > t t~ q q~"
    files, info = Q2.emit_quark2("qRtTqR")
    assert info["ndiagrams"] == 7 and "mg_desc_qrxttxqrx" in files[0][1]
