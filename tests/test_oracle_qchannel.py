"""Pins of the quark-channel oracle (oracle/me_qchannel.c; "pp -> t t~ 0-2 j").

None of these re-types the oracle's recursion:
  * q q~ -> t t~ against the textbook closed form (Combridge 1979; e.g. Ellis-Stirling-Webber table 10.2)
        sum-bar |M|^2 = (4 g^4 / 9) [ (m^2 - t)^2 + (m^2 - u)^2 + 2 m^2 s ] / s^2
    — fixes the absolute normalisation, the spinors of both lines and the colour average;
  * the Ward identity (polarisation -> momentum gives zero) on every gluon of every process — fixes the relative
    signs and factors between the diagram classes (emission off either line, three- and four-gluon vertices);
  * initial-state collinear limits onto that closed form with the Altarelli-Parisi kernels
        q -> q g :  |M|^2 -> g^2 C_F (1 + x^2)/(1 - x) / (x p_a.k) |M_0(x p_a)|^2
        g -> q q~:  |M|^2 -> g^2 T_R (x^2 + (1 - x)^2) / (x p_a.k) |M_0(x p_a)|^2
    — fixes the normalisation of every 1-jet process (incoming-gluon colour and spin averages included), and of the
    2-jet processes q q~ -> t t~ g g, q g -> t t~ q g and g g -> t t~ q q~ against the 1-jet ones (their beam and C mirrors
    against them);
  * charge conjugation (q <-> q~ together with t <-> t~) and beam exchange;
  * two light-quark lines (flavours q and r): the final-state collinear limit r r~ -> g of q q~ -> t t~ r r~ onto
    q q~ -> t t~ g with <P_qg> = T_R (1 - 2 z (1 - z)) (two azimuths pi/2 apart cancel the spin correlation), the
    initial-state limit q -> g q of q r -> t t~ q r onto g r -> t t~ r with P_gq = C_F (1 + (1 - x)^2)/x, and the
    relabelling symmetries.  Same flavour twice (q q~ -> t t~ q q~, q q -> t t~ q q): the amplitude is the difference of the
    two ways of connecting the lines (Fermi statistics).  The sign is pinned by the Pauli principle: with the two identical
    final quarks at the same momentum, the configurations in which they also share helicity and colour must not contribute
    (they carry 13.5 % of |M|^2 with the opposite sign, 2-3 % on a generic event); the crossed processes use the same rule.
"""
import math
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from oracle import oracle as O

MT = 173.0
G2 = 4 * math.pi * 0.118
CF, TR = 4.0 / 3.0, 0.5


@pytest.fixture(scope="module")
def orc():
    return O.Oracle()


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def born_closed_form(pa, pb, pt):
    s = mdot(pa + pb, pa + pb)
    t = mdot(pa - pt, pa - pt)
    u = 2 * MT * MT - s - t
    return 4 * G2 * G2 / 9 * ((MT * MT - t) ** 2 + (MT * MT - u) ** 2 + 2 * MT * MT * s) / s ** 2


def test_qqbar_to_ttbar_equals_the_closed_form(orc):
    mom = orc.rambo(11, 16, [MT, MT], 1500.0)
    for p in mom:
        ref = born_closed_form(p[0], p[1], p[2])
        assert abs(orc.me_qchannel("qQtT", p) / ref - 1) < 1e-12
        # antiquark in the first beam: the same formula with the beams exchanged
        assert abs(orc.me_qchannel("QqtT", p) / born_closed_form(p[1], p[0], p[2]) - 1) < 1e-12


@pytest.mark.parametrize("spec", ["qQtTg", "QqtTg", "qgtTq", "gqtTq", "QgtTQ", "gQtTQ"])
def test_ward_identity_one_jet(orc, spec):
    mom = orc.rambo(12, 3, [MT, MT, 0.0], 1500.0)
    for p in mom:
        v = orc.me_qchannel(spec, p)
        assert v > 0
        assert orc.me_qchannel(spec, p, ward=0) / v < 1e-20


def test_ward_identity_two_jets(orc):
    p = orc.rambo(13, 1, [MT, MT, 0.0, 0.0], 1500.0)[0]
    jobs = [(spec, w) for spec in ("qQtTgg", "qgtTqg", "ggtTqQ") for w in (-1, 0, 1)]
    with ThreadPoolExecutor(9) as ex:
        res = dict(zip(jobs, ex.map(lambda j: orc.me_qchannel(j[0], p, ward=j[1]), jobs)))
    for spec in ("qQtTgg", "qgtTqg", "ggtTqQ"):
        assert res[(spec, -1)] > 0
        for w in (0, 1):
            assert res[(spec, w)] / res[(spec, -1)] < 1e-20


def _boost(p, Q):
    M = math.sqrt(mdot(Q, Q))
    b = Q[1:] / Q[0]
    g = Q[0] / M
    bp = b @ p[1:]
    out = np.zeros(4)
    out[0] = g * (p[0] + bp)
    out[1:] = p[1:] + ((g - 1) * bp / (b @ b) + g * p[0]) * b
    return out


def _collinear_event(x, theta, beam, E=750.0, extra=None):
    """2 -> t t~ + k (+ extra) with k = (1 - x) * beam momentum, tilted by theta; momentum conserved exactly."""
    pa = np.array([E, 0, 0, E])
    pb = np.array([E, 0, 0, -E])
    sgn = 1 if beam == 0 else -1
    k = (1 - x) * E * np.array([1, math.sin(theta) * math.cos(0.7), math.sin(theta) * math.sin(0.7), sgn * math.cos(theta)])
    Q = pa + pb - k
    if extra is not None:
        Q = Q - extra
    M = math.sqrt(mdot(Q, Q))
    pp = math.sqrt(M * M / 4 - MT * MT)
    ct, ph = 0.3, 1.1
    st = math.sqrt(1 - ct * ct)
    t = np.array([M / 2, pp * st * math.cos(ph), pp * st * math.sin(ph), pp * ct])
    tb = np.array([M / 2, -t[1], -t[2], -t[3]])
    return pa, pb, _boost(t, Q), _boost(tb, Q), k


@pytest.mark.parametrize("x", [0.6, 0.8])
def test_initial_state_collinear_limits_onto_the_closed_form(orc, x):
    err = {}
    for theta in (1e-2, 1e-3):
        pa, pb, t, tb, k = _collinear_event(x, theta, 0)
        p = np.array([pa, pb, t, tb, k])
        r1 = orc.me_qchannel("qQtTg", p) / (G2 * CF * (1 + x * x) / (1 - x) / (x * mdot(pa, k)) * born_closed_form(x * pa, pb, t))
        r3 = orc.me_qchannel("gQtTQ", p) / (G2 * TR * (x * x + (1 - x) ** 2) / (x * mdot(pa, k)) * born_closed_form(x * pa, pb, t))
        pa, pb, t, tb, k = _collinear_event(x, theta, 1)
        p = np.array([pa, pb, t, tb, k])
        r2 = orc.me_qchannel("qgtTq", p) / (G2 * TR * (x * x + (1 - x) ** 2) / (x * mdot(pb, k)) * born_closed_form(pa, x * pb, t))
        err[theta] = [abs(r - 1) for r in (r1, r2, r3)]
    assert max(err[1e-3]) < 2e-3
    for a, b in zip(err[1e-2], err[1e-3]):        # the correction is linear in the angle
        assert b < 0.2 * a


def test_two_jet_collinear_limit_onto_the_one_jet_process(orc):
    x = 0.7
    g1 = np.array([120.0, 60.0, -80.0, 66.332495807108])        # a hard, well-separated massless gluon
    g1[0] = math.sqrt(g1[1] ** 2 + g1[2] ** 2 + g1[3] ** 2)

    def ratio(theta):
        pa, pb, t, tb, k = _collinear_event(x, theta, 0, extra=g1)
        v = orc.me_qchannel("qQtTgg", np.array([pa, pb, t, tb, g1, k]))
        ref = orc.me_qchannel("qQtTg", np.array([x * pa, pb, t, tb, g1]))
        # the identical-gluon factor 1/2 of the 2-jet process: the collinear gluon is one specific gluon of the two
        return 2 * v / (G2 * CF * (1 + x * x) / (1 - x) / (x * mdot(pa, k)) * ref)

    with ThreadPoolExecutor(2) as ex:
        r2, r3 = ex.map(ratio, (1e-2, 1e-3))
    assert abs(r3 - 1) < 3e-3 and abs(r3 - 1) < 0.2 * abs(r2 - 1)


def test_charge_conjugation_and_beam_exchange(orc):
    mom = orc.rambo(14, 3, [MT, MT, 0.0], 1500.0)
    for p in mom:
        c = p[[0, 1, 3, 2, 4]]                   # t <-> t~
        assert abs(orc.me_qchannel("qQtTg", p) / orc.me_qchannel("QqtTg", c) - 1) < 1e-10
        assert abs(orc.me_qchannel("qgtTq", p) / orc.me_qchannel("QgtTQ", c) - 1) < 1e-10
        b = p[[1, 0, 2, 3, 4]]                   # beams exchanged
        assert abs(orc.me_qchannel("qgtTq", p) / orc.me_qchannel("gqtTq", b) - 1) < 1e-10


def test_other_two_jet_crossings_collinear_limits_and_mirrors(orc):
    """The 2-jet crossings with one light line that the test above does not reach: q g -> t t~ q g with the final gluon
    along the incoming quark (q -> q g onto q g -> t t~ q) and g g -> t t~ q q~ with the final antiquark along an incoming
    gluon (g -> q q~ onto q g -> t t~ q); then the beam- and C-mirrored processes against these two."""
    x, theta = 0.7, 1e-3
    hard = np.array([0.0, 60.0, -80.0, 66.0])
    hard[0] = np.linalg.norm(hard[1:])
    pa, pb, t, tb, k = _collinear_event(x, theta, 0, extra=hard)
    p6 = np.array([pa, pb, t, tb, hard, k])
    ref = np.array([x * pa, pb, t, tb, hard])
    jobs = {
        "qgtTqg": ("qgtTqg", p6), "ggtTqQ": ("ggtTqQ", p6), "ref": ("qgtTq", ref),
        "gqtTqg": ("gqtTqg", p6[[1, 0, 2, 3, 4, 5]]),                 # beams exchanged
        "QgtTQg": ("QgtTQg", p6[[0, 1, 3, 2, 4, 5]]),                 # charge conjugation: q <-> q~, t <-> t~
        "gQtTQg": ("gQtTQg", p6[[1, 0, 3, 2, 4, 5]]),
        "QqtTgg": ("QqtTgg", p6[[1, 0, 2, 3, 4, 5]]), "qQtTgg": ("qQtTgg", p6),
    }
    with ThreadPoolExecutor(8) as ex:
        val = dict(zip(jobs, ex.map(lambda kv: orc.me_qchannel(*kv), jobs.values())))
    pk = mdot(pa, k)
    r1 = val["qgtTqg"] / (G2 * CF * (1 + x * x) / (1 - x) / (x * pk) * val["ref"])
    r2 = val["ggtTqQ"] / (G2 * TR * (x * x + (1 - x) ** 2) / (x * pk) * val["ref"])
    assert abs(r1 - 1) < 3e-3 and abs(r2 - 1) < 3e-3, (r1, r2)
    assert abs(val["gqtTqg"] / val["qgtTqg"] - 1) < 1e-10
    assert abs(val["QgtTQg"] / val["qgtTqg"] - 1) < 1e-10
    assert abs(val["gQtTQg"] / val["qgtTqg"] - 1) < 1e-10
    assert abs(val["QqtTgg"] / val["qQtTgg"] - 1) < 1e-10


def _perp(k):
    k3 = k[1:] / np.linalg.norm(k[1:])
    a = np.cross(k3, [0.0, 0.0, 1.0])
    a /= np.linalg.norm(a)
    return a, np.cross(k3, a)


def test_two_lines_relabelling_symmetries(orc):
    p = orc.rambo(31, 1, [MT, MT, 0.0, 0.0], 1500.0)[0]
    v = orc.me_qchannel("qQtTrR", p)
    assert v > 0 and abs(orc.me_qchannel("qQtTRr", p[[0, 1, 2, 3, 5, 4]]) / v - 1) < 1e-12
    v = orc.me_qchannel("qrtTqr", p)
    assert abs(orc.me_qchannel("rqtTqr", p[[1, 0, 2, 3, 4, 5]]) / v - 1) < 1e-12
    assert abs(orc.me_qchannel("qrtTrq", p[[0, 1, 2, 3, 5, 4]]) / v - 1) < 1e-12
    assert abs(orc.me_qchannel("QRtTQR", p[[0, 1, 3, 2, 4, 5]]) / v - 1) < 1e-10          # charge conjugation
    v = orc.me_qchannel("qqtTqq", p)                                                        # identical quarks
    assert abs(orc.me_qchannel("qqtTqq", p[[0, 1, 2, 3, 5, 4]]) / v - 1) < 1e-12
    assert abs(orc.me_qchannel("qqtTqq", p[[1, 0, 2, 3, 4, 5]]) / v - 1) < 1e-12
    assert abs(orc.me_qchannel("QQtTQQ", p[[0, 1, 3, 2, 4, 5]]) / v - 1) < 1e-10
    # a pair of another flavour in the final state is one of the two pairings of the same-flavour process
    assert orc.me_qchannel("qQtTqQ", p) != orc.me_qchannel("qQtTrR", p)


def test_final_state_pair_collinear_limit_onto_the_one_jet_process(orc):
    """q q~ -> t t~ r r~ with r || r~  ->  (2 g^2 / s_rr~) T_R (1 - 2 z (1 - z)) |M(q q~ -> t t~ g)|^2."""
    ev = orc.rambo(32, 1, [MT, MT, 0.0], 1500.0)[0]
    ref = orc.me_qchannel("qQtTg", ev)
    k = ev[4]
    a, b = _perp(k)
    z = 0.3
    for kt, tol in ((1e-1, 1e-3), (1e-2, 1e-4)):
        tot = 0.0
        for phi in (0.4, 0.4 + math.pi / 2):
            n = math.cos(phi) * a + math.sin(phi) * b
            p1, p2 = np.zeros(4), np.zeros(4)
            p1[1:] = z * k[1:] + kt * n
            p2[1:] = (1 - z) * k[1:] - kt * n
            p1[0], p2[0] = np.linalg.norm(p1[1:]), np.linalg.norm(p2[1:])
            Q = ev[2] + ev[3] + p1 + p2                      # beams along z that carry exactly this total
            pa = np.array([(Q[0] + Q[3]) / 2, 0, 0, (Q[0] + Q[3]) / 2])
            pb = np.array([(Q[0] - Q[3]) / 2, 0, 0, -(Q[0] - Q[3]) / 2])
            v = orc.me_qchannel("qQtTrR", np.array([pa, pb, ev[2], ev[3], p1, p2]))
            tot += v * 2 * mdot(p1, p2) / (2 * G2) / (TR * (1 - 2 * z * (1 - z)))
        assert abs(tot / 2 / ref - 1) < tol, (kt, tot / 2 / ref)


def test_initial_state_quark_to_gluon_limit_of_the_two_line_process(orc):
    """q r -> t t~ q r with the final q along the incoming q: -> g^2 C_F (1 + (1-x)^2)/x / (x p_a.k) |M(g r -> t t~ r)|^2,
    the gluon's spin correlation cancelled by two azimuths pi/2 apart."""
    x = 0.7
    r_out = np.array([0.0, 70.0, -90.0, 40.0])
    r_out[0] = np.linalg.norm(r_out[1:])
    res = {}
    for theta in (1e-2, 1e-3):
        tot = 0.0
        for phi in (0.7, 0.7 + math.pi / 2):
            E = 750.0
            pa, pb = np.array([E, 0, 0, E]), np.array([E, 0, 0, -E])
            k = (1 - x) * E * np.array([1, math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])
            Q = pa + pb - k - r_out
            M = math.sqrt(mdot(Q, Q))
            pp = math.sqrt(M * M / 4 - MT * MT)
            t = np.array([M / 2, pp * 0.8 * math.cos(1.1), pp * 0.8 * math.sin(1.1), pp * 0.6])
            tb = np.array([M / 2, -t[1], -t[2], -t[3]])
            t, tb = _boost(t, Q), _boost(tb, Q)
            v = orc.me_qchannel("qrtTqr", np.array([pa, pb, t, tb, k, r_out]))
            ref = orc.me_qchannel("gqtTq", np.array([x * pa, pb, t, tb, r_out]))
            tot += v / (G2 * CF * (1 + (1 - x) ** 2) / x / (x * mdot(pa, k)) * ref)
        res[theta] = abs(tot / 2 - 1)
    assert res[1e-3] < 3e-3 and res[1e-3] < 0.2 * res[1e-2], res


def test_pauli_principle_fixes_the_sign_between_the_pairings(orc):
    ev = orc.rambo(41, 2, [MT, MT, 0.0], 1500.0)
    generic = orc.rambo(42, 1, [MT, MT, 0.0, 0.0], 1500.0)[0]
    for spec in ("qqtTqq", "QQtTQQ"):
        for e in ev:
            p = np.array([e[0], e[1], e[2], e[3], e[4] / 2, e[4] / 2])        # the two identical quarks at the same momentum
            tot = orc.me_qchannel(spec, p)
            assert tot > 0 and orc.me_qchannel_pauli(spec, p) < 1e-25 * tot
        # the restricted sum itself is not trivially zero
        assert orc.me_qchannel_pauli(spec, generic) > 1e-2 * orc.me_qchannel(spec, generic)
    assert orc.me_qchannel_pauli("qrtTqr", generic) == -1


def test_bad_specs_are_rejected(orc):
    p = np.zeros((5, 4))
    for spec in ("qqtTg", "qQTtg", "ggtTg", "qQtTq"):
        assert orc.me_qchannel(spec, p) == -1
