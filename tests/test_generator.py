"""Host-logic tests of the process generator K0 (pins of §8c C8 rows "Generator",
"Colour matrices").  CPU only."""
from fractions import Fraction

import numpy as np
import pytest

from paper_2312_02898_b200.gen import topology as topo
from paper_2312_02898_b200.gen.colour import colour_matrix, common_denominator
from paper_2312_02898_b200.gen.plan import Plan


def test_gluon_tree_counts_follow_the_recursion():
    # g(k) = sum_{2-partitions} g g + sum_{3-partitions} g g g -> 1, 1, 4, 25, 220 (k leaves + root)
    want = {1: 1, 2: 1, 3: 4, 4: 25, 5: 220}
    for k, w in want.items():
        terms = topo.gluon_tree_terms(tuple(range(k)))
        feyn = sum(Fraction(1, 1 << topo.n_four_vertices(t)) for t in terms)
        assert feyn == w


@pytest.mark.parametrize("n,ndiag", [(2, 3), (3, 16), (4, 123), (5, 1240)])
def test_feynman_diagram_counts(n, ndiag):
    terms = topo.diagram_terms(n)
    assert topo.n_feynman_diagrams(terms) == ndiag


@pytest.mark.parametrize("n", [2, 3, 4])
def test_every_flow_is_fed_and_signs_are_units(n):
    fi = topo.flow_index_table(n)
    seen = set()
    for t in topo.diagram_terms(n):
        for f, s in topo.term_flows(t, fi):
            assert s in (-1, 1, -2, 2)
            seen.add(f)
    assert seen == set(range(len(fi)))


def test_colour_matrix_pins():
    # n=2: 1/3 [[16,-2],[-2,16]]; n=3 (x1/9) row 0 = (64,-8,-8,1,1,10); diag = N CF^n
    cf2 = colour_matrix(2)
    assert cf2 == [[Fraction(16, 3), Fraction(-2, 3)], [Fraction(-2, 3), Fraction(16, 3)]]
    cf3 = colour_matrix(3)
    assert [v * 9 for v in cf3[0]] == [64, -8, -8, 1, 1, 10]
    cf4 = colour_matrix(4)
    assert [v * 54 for v in cf4[0]] == [512, -64, -64, 8, 8, 80, -64, 8, 8, -1, -1, -10, 8, -1, 80, -10, 71, 62, -1,
                                        -10, -10, 62, 62, -28]
    for n, cf in ((2, cf2), (3, cf3), (4, cf4)):
        a = np.array([[float(v) for v in row] for row in cf])
        assert np.array_equal(a, a.T)
        assert all(cf[i][i] == 3 * Fraction(4, 3) ** n for i in range(len(cf)))
        assert np.linalg.matrix_rank(a) == len(cf)


@pytest.mark.slow
def test_colour_matrix_n5_pins():
    cf = colour_matrix(5)
    den = common_denominator(cf)
    assert den == 324
    vals = {v * 324 for row in cf for v in row}
    assert cf[0][0] * 324 == 4096 and min(vals) == -512 and len(vals) == 24


def test_generator_colour_matrix_equals_the_oracles_gell_mann_sum(oracle):
    # two independent routes: exact Fierz reduction (generator) vs explicit Gell-Mann matrices (oracle)
    for n in (2, 3, 4):
        a = np.array([[float(v) for v in row] for row in colour_matrix(n)])
        assert np.allclose(a, oracle.colour_matrix(n), rtol=0, atol=1e-12)


def test_plan_counts_and_recycling():
    p4 = Plan(4)
    c = p4.counts()
    assert p4.ndiagrams == 123 and len(p4.terms) == c["amp"]
    # every internal current is defined before it is used
    defined = {"ub", "vv"} | {"e%d" % i for i in range(4)}
    from paper_2312_02898_b200.gen.plan import _inputs
    for op in p4.ops:
        for nm in _inputs(op):
            assert nm in defined
        if op[0] not in ("amp", "flush"):
            assert op[1] not in defined
            defined.add(op[1])


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_accumulator_blocks_reproduce_term_flows_and_groups_cover_all_terms(n):
    """Hierarchical JAMP accumulation (plan.py): expanding accumulators through their flush tables gives the
    same flow x term sign matrix as the direct expansion (also asserted per amplitude inside Plan), and the
    diagram groups are a partition of the terms that writes every colour flow."""
    from paper_2312_02898_b200.gen.plan import partition_terms
    all_terms = topo.diagram_terms(n)
    kernels = partition_terms(n, max_terms=60, max_phase=24)
    groups = [ph for k in kernels for ph in k]           # kernels -> phases -> terms
    assert sorted(map(repr, (t for g in groups for t in g))) == sorted(map(repr, all_terms))
    fi = topo.flow_index_table(n)
    direct = {}
    for t in all_terms:
        for f, s in topo.term_flows(t, fi):
            direct[f] = direct.get(f, 0) + abs(s)
    via = {}
    for g in groups:
        p = Plan(n, terms=g)
        nacc = {}
        for op in p.ops:
            if op[0] == "amp":
                for b, a, s in op[3]:
                    nacc[(b, a)] = nacc.get((b, a), 0) + 1
            elif op[0] == "flush":
                for f, s in op[3]:
                    via[f] = via.get(f, 0) + abs(s) * nacc[(op[1], op[2])]
    assert via == direct and set(via) == set(range(len(fi)))


def test_greedy_order_lowers_live_state_without_recomputation():
    """The register-pressure-aware amplitude order (plan._greedy_order) only permutes: same currents, same FLOPs."""
    from paper_2312_02898_b200.gen.plan import partition_terms
    terms = [t for ph in partition_terms(4, max_terms=40, max_phase=10 ** 6)[4] for t in ph]
    a = Plan(4, terms=terms, greedy=False)
    b = Plan(4, terms=terms)
    ca, cb = a.counts(), b.counts()
    keys = ("v3", "k", "lq", "rq", "bil", "amp")
    assert {k: ca.get(k, 0) for k in keys} == {k: cb.get(k, 0) for k in keys}
    assert b.max_live() <= a.max_live()
