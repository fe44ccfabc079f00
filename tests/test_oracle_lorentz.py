"""Pins for conventions C1: gamma matrices, spinors, polarisation vectors."""
import numpy as np

G = np.diag([1.0, -1.0, -1.0, -1.0])


def _slash(orc, p):
    return sum(G[m, m] * p[m] * orc.gamma(m) for m in range(4))


def _momenta():
    rng = np.random.default_rng(12)
    out = []
    for m in (0.0, 173.0, 4.7):
        for _ in range(6):
            p3 = rng.normal(size=3) * 300
            out.append((np.array([np.sqrt(m * m + p3 @ p3), *p3]), m))
    # special directions: along +z, along -z
    out.append((np.array([750.0, 0, 0, 750.0]), 0.0)); out.append((np.array([750.0, 0, 0, -750.0]), 0.0))
    e = np.sqrt(173.0 ** 2 + 100.0 ** 2)
    out.append((np.array([e, 0, 0, -100.0]), 173.0)); out.append((np.array([e, 0, 0, 100.0]), 173.0))
    return out


def test_clifford_algebra_and_gamma5(oracle):
    g = [oracle.gamma(m) for m in range(4)]
    for m in range(4):
        for n in range(4):
            assert np.allclose(g[m] @ g[n] + g[n] @ g[m], 2 * G[m, n] * np.eye(4))
    g5 = 1j * g[0] @ g[1] @ g[2] @ g[3]
    assert np.allclose(g5, np.diag([-1, -1, 1, 1]))          # C1: gamma5 = diag(-1,-1,+1,+1)
    assert np.allclose(g[0].conj().T, g[0])


def test_dirac_equation_and_completeness(oracle_ld):
    orc = oracle_ld
    g0 = orc.gamma(0)
    for p, m in _momenta():
        ps = _slash(orc, p)
        su = np.zeros((4, 4), complex); sv = np.zeros((4, 4), complex)
        scale = p[0] * np.sqrt(p[0])
        for lam in (1, -1):
            u = orc.spinor("u", p, m, lam); v = orc.spinor("v", p, m, lam)
            assert np.abs((ps - m * np.eye(4)) @ u).max() < 1e-13 * scale
            assert np.abs((ps + m * np.eye(4)) @ v).max() < 1e-13 * scale
            ub = u.conj() @ g0; vb = v.conj() @ g0
            su += np.outer(u, ub); sv += np.outer(v, vb)
            # normalisation ubar u = 2m, vbar v = -2m
            assert abs(ub @ u - 2 * m) < 1e-12 * p[0] and abs(vb @ v + 2 * m) < 1e-12 * p[0]
            # helicity eigenstates: (Sigma.p/|p|) u = lam u
            pabs = np.linalg.norm(p[1:])
            sig = [np.array([[0, 1], [1, 0]]), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]])]
            sp = sum(p[i + 1] * sig[i] for i in range(3)) / pabs
            Sp = np.block([[sp, np.zeros((2, 2))], [np.zeros((2, 2)), sp]])
            assert np.abs(Sp @ u - lam * u).max() < 1e-13 * np.sqrt(2 * p[0])
            assert np.abs(Sp @ v + lam * v).max() < 1e-13 * np.sqrt(2 * p[0])
        assert np.abs(su - (ps + m * np.eye(4))).max() < 1e-13 * p[0]
        assert np.abs(sv - (ps - m * np.eye(4))).max() < 1e-13 * p[0]


def test_massless_spinor_has_exact_zero_components(oracle):
    p = np.array([100.0, 30.0, -40.0, np.sqrt(100.0 ** 2 - 2500.0)])
    u = oracle.spinor("u", p, 0.0, 1)
    assert u[0] == 0 and u[1] == 0          # omega_- = 0 exactly (C1)


def test_polarisation_vectors(oracle_ld):
    orc = oracle_ld
    for k, m in _momenta():
        if m != 0.0:
            continue
        e = {lam: orc.polvec(k, lam) for lam in (1, -1)}
        for lam in (1, -1):
            assert abs((e[lam] * np.diag(G)) @ k) < 1e-14 * k[0]                  # eps.k = 0
            assert abs((e[lam] * np.diag(G)) @ e[lam].conj() + 1) < 1e-14          # eps.eps* = -1
            assert abs((e[lam] * np.diag(G)) @ e[lam]) < 1e-14                     # eps.eps = 0
            assert e[lam][0] == 0
        assert abs((e[1] * np.diag(G)) @ e[-1].conj()) < 1e-14                     # orthogonal
        # completeness in the transverse plane: sum eps_i eps*_j = delta_ij - k_i k_j/|k|^2
        kk = k[1:] / np.linalg.norm(k[1:])
        S = sum(np.outer(e[l][1:], e[l][1:].conj()) for l in (1, -1))
        assert np.abs(S - (np.eye(3) - np.outer(kk, kk))).max() < 1e-14
        # helicity: rotation about k by angle a multiplies eps(lam) by exp(-i lam a) -> check via
        # (k_hat x eps) = -i lam eps
        assert np.abs(np.cross(kk, e[1][1:]) + 1j * e[1][1:]).max() < 1e-14
        assert np.abs(np.cross(kk, e[-1][1:]) - 1j * e[-1][1:]).max() < 1e-14
