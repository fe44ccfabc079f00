"""Exact SU(3) colour matrix for the T-string colour-flow basis (K0 of SURVEY.md §8a; K6 consumes it).

CF[s, s'] = sum over adjoint indices a_1..a_n and fundamental indices of
            [(T^{a_s1}..T^{a_sn})_{ij}]^* (T^{a_s'1}..T^{a_s'n})_{ij}
          = Tr( T^{a_s'1} .. T^{a_s'n} T^{a_sn} .. T^{a_s1} )       (all a's contracted pairwise)
evaluated *symbolically* in exact rational arithmetic by repeated use of the Fierz identity
    (T^a)_{ij} (T^a)_{kl} = 1/2 ( delta_il delta_jk - 1/N delta_ij delta_kl ),
i.e.  Tr(X T^a Y T^a) = 1/2 Tr(X) Tr(Y) - 1/(2N) Tr(X Y)   and   Tr(X T^a) Tr(Y T^a) = 1/2 Tr(X Y) - 1/(2N) Tr(X) Tr(Y).
This shares nothing with the oracle, which multiplies explicit Gell-Mann matrices numerically.
Because CF depends only on the relative permutation, n! traces suffice.
"""
from fractions import Fraction
from functools import lru_cache
from itertools import permutations

NC = 3


@lru_cache(maxsize=None)
def _traces(state):
    """state: tuple of tuples of labels (a product of traces of generators, every label appearing exactly
    twice over the whole product).  Returns the fully contracted value as a Fraction."""
    state = tuple(t for t in state)
    # empty traces contribute Tr(1) = N
    val = Fraction(1)
    rest = []
    for t in state:
        if len(t) == 0:
            val *= NC
        else:
            rest.append(t)
    if not rest:
        return val
    t0 = rest[0]
    a = t0[0]
    others = rest[1:]
    if a in t0[1:]:
        # Tr(T^a X T^a Y) with t0 = (a,) + X + (a,) + Y
        k = t0.index(a, 1)
        X, Y = t0[1:k], t0[k + 1:]
        v1 = _traces(_canon((X, Y) + tuple(others)))
        v2 = _traces(_canon((X + Y,) + tuple(others)))
        return val * (Fraction(1, 2) * v1 - Fraction(1, 2 * NC) * v2)
    # a sits in another trace: Tr(T^a X) Tr(T^a Y) = 1/2 Tr(X Y) - 1/(2N) Tr(X) Tr(Y)
    for idx, t in enumerate(others):
        if a in t:
            k = t.index(a)
            Y = t[k + 1:] + t[:k]
            X = t0[1:]
            remaining = tuple(others[:idx] + others[idx + 1:])
            v1 = _traces(_canon((X + Y,) + remaining))
            v2 = _traces(_canon((X, Y) + remaining))
            return val * (Fraction(1, 2) * v1 - Fraction(1, 2 * NC) * v2)
    raise ValueError("unpaired colour index")


def _canon(state):
    """Canonical form: rotate each trace so its smallest label comes first, relabel by first appearance."""
    rot = []
    for t in state:
        if t:
            k = t.index(min(t))
            t = t[k:] + t[:k]
        rot.append(tuple(t))
    rot.sort(key=lambda t: (len(t), t))
    relabel = {}
    out = []
    for t in rot:
        nt = []
        for x in t:
            if x not in relabel:
                relabel[x] = len(relabel)
            nt.append(relabel[x])
        out.append(tuple(nt))
    return tuple(out)


def colour_matrix(n):
    """Exact CF (list of lists of Fraction), flows = permutations of range(n) in lexicographic order."""
    perms = list(permutations(range(n)))
    index = {p: i for i, p in enumerate(perms)}
    # value depends on rho = s^-1 o s' only:  CF[id, rho]
    base = {}
    ident = tuple(range(n))
    for rho in perms:
        tr = tuple(rho) + tuple(reversed(ident))
        base[rho] = _traces(_canon((tr,)))
    cf = [[None] * len(perms) for _ in perms]
    for s in perms:
        inv = [0] * n
        for pos, lab in enumerate(s):
            inv[lab] = pos
        for sp in perms:
            rho = tuple(inv[lab] for lab in sp)   # relabel gluons so that s becomes the identity
            cf[index[s]][index[sp]] = base[rho]
    return cf


def common_denominator(cf):
    from math import lcm
    d = 1
    for row in cf:
        for v in row:
            d = lcm(d, v.denominator)
    return d
