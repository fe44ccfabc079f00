"""Pins for the colour matrices (SURVEY.md §8c C4 'Colour matrix', C8 row 'Colour matrices')."""
import itertools
from fractions import Fraction

import numpy as np
import pytest


def test_brute_equals_streamed(oracle):
    for n in (1, 2, 3):
        assert np.abs(oracle.colour_matrix(n, brute=True) - oracle.colour_matrix(n)).max() < 1e-12


@pytest.mark.parametrize("n,den", [(2, 3), (3, 9), (4, 54), (5, 324)])
def test_colour_matrix_tables(oracle, n, den):
    cf = oracle.colour_matrix(n)
    npm = cf.shape[0]
    assert np.allclose(cf, cf.T, atol=1e-10)
    # diagonal N C_F^n
    assert np.allclose(np.diag(cf), 3 * (4.0 / 3.0) ** n, atol=1e-10)
    # entries are integers over `den`
    scaled = cf * den
    assert np.abs(scaled - np.round(scaled)).max() < 1e-7
    # full rank, positive definite
    ev = np.linalg.eigvalsh(cf)
    assert ev.min() > 1e-6
    row0 = np.round(scaled[0]).astype(int).tolist()
    if n == 2:
        assert np.round(scaled).astype(int).tolist() == [[16, -2], [-2, 16]]
    if n == 3:
        assert row0 == [64, -8, -8, 1, 1, 10]
    if n == 4:
        assert row0 == [512, -64, -64, 8, 8, 80, -64, 8, 8, -1, -1, -10, 8, -1, 80, -10, 71, 62, -1, -10, -10, 62, 62, -28]
        assert len(set(np.round(scaled).astype(int).ravel().tolist())) == 9
    if n == 5:
        vals = set(np.round(scaled).astype(int).ravel().tolist())
        assert np.round(scaled[0, 0]) == 4096 and min(vals) == -512 and len(vals) == 24
    # relabelling invariance: CF[s,s'] depends only on s^-1 s'
    perms = list(itertools.permutations(range(n)))
    idx = {p: i for i, p in enumerate(perms)}
    rng = np.random.default_rng(0)
    for _ in range(50):
        a, b = perms[rng.integers(npm)], perms[rng.integers(npm)]
        inv = [0] * n
        for i, x in enumerate(a):
            inv[x] = i
        rel = tuple(inv[x] for x in b)
        assert abs(cf[idx[a], idx[b]] - cf[0, idx[rel]]) < 1e-10


def test_n2_against_fierz_by_hand():
    # Tr(T^a T^b T^b T^a) = N C_F^2 = 16/3 ; Tr(T^a T^b T^a T^b) = -C_F/2 ... = -2/3  (textbook SU(3))
    N = Fraction(3); CF = Fraction(4, 3)
    assert N * CF * CF == Fraction(16, 3)
    assert N * CF * (CF - N / 2) == Fraction(-2, 3)
