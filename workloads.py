"""Seeded synthetic workloads shared by the CUDA path's tests/bench and the oracle's tests.

Holds NO arithmetic of the method: only the table of configurations from BASELINE.json
(`configs`) — process string, sqrt(s), event count, Philox seed, final-state
masses — and a reader for the text fixtures in tests/golden/.  Momenta themselves are produced
by each side's own Philox+RAMBO (compared separately), or by the CUDA path and handed to the
oracle as plain doubles for |M|^2 parity (SURVEY §8c "parity protocol").
"""
import os

MT = 173.0

# name -> configuration.  `index` is the position in BASELINE.json `configs`.
CONFIGS = {
    "eemumu": dict(index=0, proc="e+ e- > mu+ mu-", sqrt_s=500.0, nevt=16384, seed=1,
                   masses_final=[0.0, 0.0], precisions=("fp64",)),
    "ggtt": dict(index=1, proc="g g > t t~", sqrt_s=1500.0, nevt=524288, seed=2,
                 masses_final=[MT, MT], precisions=("fp64",)),
    "ggttg": dict(index=2, proc="g g > t t~ g", sqrt_s=1500.0, nevt=524288, seed=3,
                  masses_final=[MT, MT, 0.0], precisions=("fp64", "fp32")),
    "ggttgg": dict(index=3, proc="g g > t t~ g g", sqrt_s=1500.0, nevt=524288, seed=4,
                   masses_final=[MT, MT, 0.0, 0.0], precisions=("fp64", "fp32")),
    "ggttggg": dict(index=4, proc="g g > t t~ g g g", sqrt_s=1500.0, nevt=262144, seed=5,
                    masses_final=[MT, MT, 0.0, 0.0, 0.0], precisions=("fp64",)),
}
PROC_TO_NAME = {v["proc"]: k for k, v in CONFIGS.items()}

# Quark channels of p p -> t t~ + 0..2 jets with one light-quark line.  Key: one character
# per particle in process order ('q' light quark, 'Q' light antiquark, 'g' gluon, 'tT' = t t~); not BASELINE.json
# configs: parity-test workloads only (sqrt(s) and the RAMBO recipe as for the gluon channels).
_QNAMES = {"q": "q", "Q": "q~", "r": "r", "R": "r~", "g": "g", "t": "t", "T": "t~"}
QUARK_SPECS = ("qQtT", "QqtT",
               "qQtTg", "QqtTg", "qgtTq", "gqtTq", "QgtTQ", "gQtTQ",
               "qQtTgg", "QqtTgg", "qgtTqg", "gqtTqg", "QgtTQg", "gQtTQg", "ggtTqQ")
# two light-quark lines ('r' / 'R': quark / antiquark of a second light flavour), no gluon
QUARK2_SPECS = ("qQtTrR", "QqtTrR", "qrtTqr", "qRtTqR", "QrtTQr", "QRtTQR",
                "qQtTqQ", "QqtTqQ", "qqtTqq", "QQtTQQ")
QUARK_CHANNELS = {
    spec: dict(proc=" ".join(_QNAMES[c] for c in spec[:2]) + " > " + " ".join(_QNAMES[c] for c in spec[2:]),
               sqrt_s=1500.0, seed=20 + i, masses_final=[MT, MT] + [0.0] * (len(spec) - 4))
    for i, spec in enumerate(QUARK_SPECS + QUARK2_SPECS)
}

GOLDEN_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tests", "golden")


def read_points(filename):
    """Parse a tests/golden/*.txt fixture: blocks of
         point <name> <proc...> | value <float>
         <E> <px> <py> <pz>     (one line per particle, process order)
       '#' starts a comment.  Returns list of dict(name, proc, value, momenta)."""
    pts, cur = [], None
    with open(os.path.join(GOLDEN_DIR, filename)) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            if line.startswith("point"):
                head, val = line.split("|")
                toks = head.split()
                cur = dict(name=toks[1], proc=" ".join(toks[2:]), value=float(val.split()[1]), momenta=[])
                pts.append(cur)
            else:
                cur["momenta"].append([float(x) for x in line.split()])
    return pts
