"""Pins for the matrix-element half of the oracle.

Nothing here re-types the oracle's own formulas: the pins are closed forms (e+e- -> mu+mu- gamma+Z
angular formula, Combridge gg -> tt~), an independent colour-dressed evaluation with explicit
f^{abc}, gauge (Ward) invariance, Bose symmetry, Lorentz invariance, helicity-selection rules and
the survey's separately computed worked values.
"""
import math

import numpy as np
import pytest

import workloads
from oracle import oracle as O

PAR = O.default_params()
GS2 = 4 * math.pi * 0.118


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


# ---------------------------------------------------------------- closed forms
def eemumu_closed(p, par=PAR, photon_only=False):
    """|M|^2 = e^4 [A0 (1+c^2) + A1 c], c = cos angle(e-, mu-)."""
    e2 = 4 * math.pi / par.alpha_ew_inv
    sw2 = par.sw2; cw2 = 1 - sw2
    gv = -0.5 + 2 * sw2; ga = -0.5
    q = p[0] + p[1]; s = mdot(q, q)
    r = s / (4 * sw2 * cw2 * (s - par.mz ** 2 + 1j * par.mz * par.gamma_z))
    if photon_only:
        r = 0
    a0 = 1 + 2 * r.real * gv ** 2 + abs(r) ** 2 * (gv ** 2 + ga ** 2) ** 2 if r != 0 else 1.0
    a1 = 4 * r.real * ga ** 2 + 8 * abs(r) ** 2 * gv ** 2 * ga ** 2 if r != 0 else 0.0
    c = (p[1][1:] @ p[3][1:]) / (np.linalg.norm(p[1][1:]) * np.linalg.norm(p[3][1:]))
    return e2 * e2 * (a0 * (1 + c * c) + a1 * c)


def combridge(p, mt=173.0):
    """g^4/(2VN) (V/(t1 t2) - 2N^2)(t1^2 + t2^2 + rho - rho^2/(4 t1 t2))."""
    N, V = 3.0, 8.0
    s = mdot(p[0] + p[1], p[0] + p[1])
    t1 = 2 * mdot(p[0], p[2]) / s; t2 = 2 * mdot(p[1], p[2]) / s; rho = 4 * mt * mt / s
    return GS2 ** 2 / (2 * V * N) * (V / (t1 * t2) - 2 * N * N) * (t1 * t1 + t2 * t2 + rho - rho * rho / (4 * t1 * t2))


def test_default_sw2_is_the_A1_reading():
    assert abs(O.default_sw2() - 0.22224649) < 1e-8


def test_eemumu_closed_form(oracle, oracle_ld):
    pts = workloads.read_points("worked_examples.txt")
    p = np.array(pts[0]["momenta"])
    for orc in (oracle, oracle_ld):
        v = orc.me("e+ e- > mu+ mu-", p)
        assert abs(v / pts[0]["value"] - 1) < 1e-12
        assert abs(v / eemumu_closed(p) - 1) < 1e-13
    mom = oracle.rambo(1, 500, [0.0, 0.0], 500.0)
    for p in mom:
        assert abs(oracle_ld.me("e+ e- > mu+ mu-", p) / eemumu_closed(p) - 1) < 1e-12
    # photon-only limit: switch the Z off by making it infinitely heavy
    par = O.default_params(); par.mz = 1e9
    p = np.array(pts[0]["momenta"])
    assert abs(oracle.me("e+ e- > mu+ mu-", p, par) / eemumu_closed(p, photon_only=True) - 1) < 1e-9
    assert abs(eemumu_closed(p, photon_only=True) - 1.1242220471453e-2) < 1e-14


def test_eemumu_helicity_selection(oracle):
    p = np.array(workloads.read_points("worked_examples.txt")[0]["momenta"])
    tot, hel = oracle.me("e+ e- > mu+ mu-", p, per_helicity=True)
    assert np.count_nonzero(hel) == 4 and abs(hel.sum() / tot - 1) < 1e-14
    # opposite helicities on each massless line: h = (l1,l2,l3,l4) with l1 != l2, l3 != l4
    for h in np.nonzero(hel)[0]:
        b = [(h >> k) & 1 for k in (3, 2, 1, 0)]
        assert b[0] != b[1] and b[2] != b[3]


def test_ggtt_combridge(oracle, oracle_ld):
    pts = {q["name"]: q for q in workloads.read_points("worked_examples.txt")}
    p = np.array(pts["ggtt"]["momenta"])
    assert abs(combridge(p) / pts["ggtt"]["value"] - 1) < 1e-13
    mom = oracle.rambo(2, 300, [173.0, 173.0], 1500.0)
    for p in mom:
        c = combridge(p)
        assert abs(oracle_ld.me("g g > t t~", p) / c - 1) < 1e-11
        assert abs(oracle.me_ggtt_explicit(p) / c - 1) < 1e-11
    # other energies / masses
    par = O.default_params(); par.mt = 50.0
    mom = oracle.rambo(9, 50, [50.0, 50.0], 400.0)
    for p in mom:
        assert abs(oracle_ld.me("g g > t t~", p, par) / combridge(p, 50.0) - 1) < 1e-11


def test_ggtt_helicity_zeros_in_cm_frame(oracle):
    # C8 'Helicity counts': 12/16 in the CM frame; zeros = equal gluon helicities with opposite t, t~ ones
    p = oracle.rambo(2, 1, [173.0, 173.0], 1500.0)[0]
    tot, hel = oracle.me("g g > t t~", p, per_helicity=True)
    good = hel > 1e-14 * tot
    assert good.sum() == 12
    for h in range(16):
        l1, l2, lt, ltb = [(h >> k) & 1 for k in (3, 2, 1, 0)]
        assert good[h] == (not (l1 == l2 and lt != ltb))


def test_worked_examples(oracle_ld):
    for q in workloads.read_points("worked_examples.txt"):
        v = oracle_ld.me(q["proc"], np.array(q["momenta"]))
        assert abs(v / q["value"] - 1) < 1e-12, q["name"]


# ---------------------------------------------------------------- independent second route
@pytest.mark.parametrize("nfinal,nev", [(0, 5), (1, 5), (2, 3)])
def test_colour_ordered_equals_colour_dressed(oracle, nfinal, nev):
    masses = [173.0, 173.0] + [0.0] * nfinal
    mom = oracle.rambo(100 + nfinal, nev, masses, 1500.0)
    for p in mom:
        a = oracle.me(nfinal + 1, p); b = oracle.me_dressed(nfinal, p)
        assert abs(a / b - 1) < 1e-11


# ---------------------------------------------------------------- invariances
@pytest.mark.parametrize("nfinal", [0, 1, 2, 3])
def test_ward_identity(oracle_ld, nfinal):
    masses = [173.0, 173.0] + [0.0] * nfinal
    p = oracle_ld.rambo(200 + nfinal, 1, masses, 1500.0)[0]
    ref = oracle_ld.me(nfinal + 1, p)
    for g in range(2 + nfinal):
        # eps -> k: |M|^2 carries one factor (GeV)^2 more; compare to s * |M|^2
        assert oracle_ld.me_ward(nfinal, p, g) < 1e-24 * 1500.0 ** 2 * ref


@pytest.mark.parametrize("nfinal", [0, 1, 2, 3])
def test_bose_symmetry(oracle, nfinal):
    masses = [173.0, 173.0] + [0.0] * nfinal
    p = oracle.rambo(300 + nfinal, 1, masses, 1500.0)[0]
    ref = oracle.me(nfinal + 1, p)
    # swap the two beam gluons = rotate the event by pi about x (pz -> -pz, py -> -py) ... instead
    # exchange them as labels: same physical configuration with beams relabelled
    q = p.copy(); q[[0, 1]] = q[[1, 0]]
    # after relabelling, beam 1 flies along -z: the oracle takes general momenta
    assert abs(oracle.me(nfinal + 1, q) / ref - 1) < 1e-12
    if nfinal >= 2:
        q = p.copy(); q[[4, 5]] = q[[5, 4]]
        assert abs(oracle.me(nfinal + 1, q) / ref - 1) < 1e-12
    if nfinal >= 3:
        q = p.copy(); q[[4, 6]] = q[[6, 4]]
        assert abs(oracle.me(nfinal + 1, q) / ref - 1) < 1e-12


def _lorentz(rng):
    # random rotation (QR) times random boost
    A = rng.normal(size=(3, 3)); Q, _ = np.linalg.qr(A)
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    R = np.eye(4); R[1:, 1:] = Q
    beta = rng.normal(size=3); beta *= 0.6 / np.linalg.norm(beta)
    b2 = beta @ beta; g = 1 / math.sqrt(1 - b2)
    B = np.eye(4); B[0, 0] = g; B[0, 1:] = B[1:, 0] = g * beta
    B[1:, 1:] += (g - 1) * np.outer(beta, beta) / b2
    return B @ R


@pytest.mark.parametrize("proc,nfinal", [("e+ e- > mu+ mu-", -1), ("g g > t t~", 0), ("g g > t t~ g", 1),
                                         ("g g > t t~ g g", 2), ("g g > t t~ g g g", 3)])
def test_lorentz_invariance(oracle_ld, proc, nfinal):
    rng = np.random.default_rng(5)
    cfg = workloads.CONFIGS[workloads.PROC_TO_NAME[proc]]
    p = oracle_ld.rambo(400, 1, cfg["masses_final"], cfg["sqrt_s"])[0]
    ref = oracle_ld.me(proc, p)
    for _ in range(2):
        L = _lorentz(rng)
        q = p @ L.T
        assert abs(oracle_ld.me(proc, q) / ref - 1) < 1e-11


def test_ggtt_all_helicities_contribute_after_boost(oracle):
    # A7: 16/16 after a boost along z
    p = oracle.rambo(2, 1, [173.0, 173.0], 1500.0)[0]
    g = 1.25; b = math.sqrt(1 - 1 / g ** 2)
    L = np.eye(4); L[0, 0] = L[3, 3] = g; L[0, 3] = L[3, 0] = g * b
    tot, hel = oracle.me("g g > t t~", p @ L.T, per_helicity=True)
    assert (hel > 1e-14 * tot).sum() == 16


def test_batch_driver_matches_single_calls(oracle):
    mom = oracle.rambo(3, 16, [173.0, 173.0, 0.0], 1500.0)
    out = oracle.me_batch("g g > t t~ g", mom)
    for i in range(16):
        assert out[i] == oracle.me("g g > t t~ g", mom[i])
