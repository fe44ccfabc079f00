"""Pins of the oracle's batch-unweighting primitive (oracle/weight.c; PAPER.md:99-:103): closed forms and exactness."""
import math

import numpy as np


def test_weight_max_closed_forms(oracle, oracle_ld):
    n = 10000
    me = np.arange(1, n + 1, dtype=np.float64)            # me_i = i, w_i = 2: products 2i are exact
    w = np.full(n, 2.0)
    for orc in (oracle, oracle_ld):
        prod, (mx, su, s2) = orc.weight_max(me, w)
        assert np.array_equal(prod, 2.0 * me)
        assert mx == 2.0 * n                               # the maximum of exact products is exact
        assert su == n * (n + 1)                           # 2 * n(n+1)/2, exactly representable
        assert s2 == 4 * n * (n + 1) * (2 * n + 1) // 6    # 4 * sum i^2
    # the maximum does not depend on the order, and is attained by a product of the inputs
    rng = np.random.default_rng(7)
    me = rng.lognormal(size=5000); w = rng.uniform(0.1, 3.0, size=5000)
    prod, (mx, su, s2) = oracle_ld.weight_max(me, w)
    assert mx == max(float(a) * float(b) for a, b in zip(w, me))
    assert abs(su / math.fsum(prod) - 1) < 1e-15 and abs(s2 / math.fsum(p * p for p in prod) - 1) < 1e-15
    # single precision products are rounded once to float
    prod32, _ = oracle.weight_max(me, w, single=True)
    assert np.array_equal(prod32, (w * me).astype(np.float32).astype(np.float64))
    # empty batch
    _, out = oracle.weight_max(np.zeros(0), np.zeros(0))
    assert out[0] == -math.inf and out[1] == 0 and out[2] == 0
