"""Independent normalisation pin of the oracle's gg -> tt~ + n g at the highest multiplicity.

Collinear factorisation: when two final-state gluons i, j become collinear (s_ij -> 0), the matrix element summed over
spins and colours factorises onto the one with one gluon less,
    |M_{n+1}|^2  ->  (8 pi alpha_s / s_ij) <P_gg(z)> |M_n|^2,      <P_gg(z)> = 2 C_A [ z/(1-z) + (1-z)/z + z(1-z) ],
after averaging over the azimuth of the splitting (the spin-correlation term is ~ cos 2 phi: two azimuths pi/2 apart
cancel it).  The values the oracle returns carry the 1/k! of k identical final-state gluons (A3), so the ratio of the
returned values picks up k!/(k+1)! = 1/(k+1).  Nothing in this relation is shared with the recursion: it fixes the
overall factor (the 1536 = 256 * 3! of gg -> tt~ggg), the colour matrix normalisation and the coupling power, given the
lower multiplicity — which is pinned by Combridge (n = 2) and by the colour-dressed route (n = 3, 4).
Kinematics: Catani-Seymour map of an n-body point (emitter = last gluon, spectator = the gluon before it) to an
(n+1)-body point with exact momentum conservation and mass shells.
"""
import math

import numpy as np
import pytest

import workloads

ALPHA_S, CA = 0.118, 3.0


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def split(ev, y, z, phi):
    """ev [npar][4] with massless last two particles -> [npar+1][4]: the last particle splits into two."""
    pij, pk = ev[-1], ev[-2]
    # transverse basis orthogonal to pij and pk
    rng = np.random.default_rng(11)
    basis = []
    for _ in range(2):
        v = rng.normal(size=4)
        v[0] = 0.0
        for _it in range(2):      # remove components along pij, pk (Minkowski) and earlier basis vectors
            pp = mdot(pij, pk)
            v = v - pk * (mdot(v, pij) / pp) - pij * (mdot(v, pk) / pp)
            for b in basis:
                v = v - b * (mdot(v, b) / mdot(b, b))
        basis.append(v / math.sqrt(-mdot(v, v)))
    kt = math.sqrt(2.0 * y * z * (1 - z) * mdot(pij, pk))
    kperp = kt * (math.cos(phi) * basis[0] + math.sin(phi) * basis[1])
    pi = z * pij + y * (1 - z) * pk + kperp
    pj = (1 - z) * pij + y * z * pk - kperp
    pkn = (1 - y) * pk
    out = np.vstack([ev[:-2], pkn[None], pi[None], pj[None]])
    return out, 2.0 * mdot(pi, pj)


def test_collinear_limit_fixes_the_normalisation_of_ggttggg(oracle, oracle_ld):
    """gg -> tt~ggg onto gg -> tt~gg (the final-state map needs two final-state gluons in the lower process).  A wrong
    identical-particle factor ((n-1)! for (n-2)!: ratio 1/4), a wrong colour-matrix normalisation or a wrong coupling
    power changes the ratio by O(1)."""
    name_hi, name_lo, kfinal = "ggttggg", "ggttgg", 2
    lo, hi = workloads.CONFIGS[name_lo], workloads.CONFIGS[name_hi]
    evs = oracle.rambo(lo["seed"] + 100, 3, lo["masses_final"], lo["sqrt_s"])
    z = 0.37
    for ev in evs:
        me_lo = oracle_ld.me(lo["proc"], ev)
        ratios = []
        for y in (1e-6, 1e-8):
            acc, sij = 0.0, None
            for phi in (0.3, 0.3 + math.pi / 2):
                ev5, sij = split(ev, y, z, phi)
                # on shell and momentum conserving by construction
                assert abs(mdot(ev5[-1], ev5[-1])) < 1e-6 and abs(mdot(ev5[-2], ev5[-2])) < 1e-6
                assert np.allclose(ev5[2:].sum(axis=0), ev[2:].sum(axis=0), atol=1e-9)
                acc += 0.5 * oracle_ld.me(hi["proc"], ev5)
            pgg = 2 * CA * (z / (1 - z) + (1 - z) / z + z * (1 - z))
            pred = 8 * math.pi * ALPHA_S / sij * pgg * me_lo / (kfinal + 1)
            ratios.append(acc / pred)
        # the limit is approached like sqrt(y): 1e-6 -> O(1e-3), 1e-8 -> O(1e-4)
        print("collinear ratios (y = 1e-6, 1e-8):", ratios)
        assert abs(ratios[1] - 1) < 2e-3, ratios
        assert abs(ratios[1] - 1) < abs(ratios[0] - 1) + 1e-4, ratios
