"""Tree-diagram enumeration and colour-flow expansion for  g g -> t t~ + (n-2) g.

K0 of SURVEY.md §8(a) ("Madgraph5_aMC@NLO is a code generator": process -> source of the
matrix element).  Build-time host code; nothing here runs on the timed path.

Feynman rules (QCD + top): vertices {t t~ g, g g g, g g g g}.  With a single quark line every
tree diagram is an ordered sequence of *blocks* along the line from the top (colour index i) to the antitop
(colour index j~); a block is a rooted gluon tree whose root propagator ends on a quark-gluon vertex and
whose leaves are external gluons.  Internal gluon vertices have 2 (ggg) or 3 (gggg) children.

Colour: with f^{abc} T^c = -i [T^a, T^b] every ggg vertex turns into a commutator, so a diagram contributes
its kinematic value, up to a sign, to the colour flows (= orderings sigma of all gluons along the T-string
T^{sigma_1}..T^{sigma_n}) compatible with its planar embeddings.  We fix an embedding per tree (children
ordered by their smallest leaf label) and evaluate the tree with the *colour-ordered* vertex functions in
that order:
   ('g', i)                         external gluon i
   ('v3', A, B)                     three-gluon vertex, value antisymmetric in (A, B)
   ('k', A, M, C)                   one kinematic structure of the four-gluon vertex,
                                    K_M = (A.M) C + (M.C) A - 2 (A.C) M      (symmetric in A <-> C)
An unordered gggg vertex {X, Y, Z} gives K_mid for the ordering with `mid` in the middle; since
K_X + K_Y + K_Z = 0 only two structures are evaluated (K_X, K_Y) and K_Z = -K_X - K_Y.  A Feynman
diagram with q four-gluon vertices therefore becomes 2^q *terms*.
   orderings(leaf i)        = { (i,): +1 }
   orderings(v3(A, B))      = { a+b: s_a s_b } u { b+a: -s_a s_b }
   orderings(k(A, M, C))    = { a+m+c: +, c+m+a: +, m+c+a: -, a+c+m: - } (x sub-signs)
"""
from functools import lru_cache
from itertools import permutations


def set_partitions_2(items):
    """Unordered splits of the tuple `items` (sorted) into two non-empty parts; the part holding items[0]
    comes first."""
    first, rest = items[0], items[1:]
    n = len(rest)
    for mask in range(1 << n):
        a = (first,) + tuple(rest[i] for i in range(n) if mask >> i & 1)
        b = tuple(rest[i] for i in range(n) if not mask >> i & 1)
        if b:
            yield a, b


def set_partitions_3(items):
    """Unordered splits into three non-empty parts, ordered by smallest element."""
    for a, bc in set_partitions_2(items):
        if len(bc) >= 2:
            for b, c in set_partitions_2(bc):
                yield a, b, c


@lru_cache(maxsize=None)
def gluon_tree_terms(leaves):
    """All terms (see module doc) of rooted gluon trees over the sorted tuple `leaves`.
    Returns a tuple of (tree, n_feynman_weight) where trees with four-gluon vertices appear once per
    kinematic structure."""
    if len(leaves) == 1:
        return (("g", leaves[0]),)
    out = []
    for a, b in set_partitions_2(leaves):
        for ta in gluon_tree_terms(a):
            for tb in gluon_tree_terms(b):
                out.append(("v3", ta, tb))
    if len(leaves) >= 3:
        for x, y, z in set_partitions_3(leaves):
            for tx in gluon_tree_terms(x):
                for ty in gluon_tree_terms(y):
                    for tz in gluon_tree_terms(z):
                        out.append(("k", ty, tx, tz))   # K_X : X in the middle
                        out.append(("k", tx, ty, tz))   # K_Y : Y in the middle
    return tuple(out)


def n_four_vertices(tree):
    if tree[0] == "g":
        return 0
    return (1 if tree[0] == "k" else 0) + sum(n_four_vertices(t) for t in tree[1:])


def leaves_of(tree):
    if tree[0] == "g":
        return (tree[1],)
    out = ()
    for t in tree[1:]:
        out += leaves_of(t)
    return out


def leafmask(tree):
    m = 0
    for i in leaves_of(tree):
        m |= 1 << i
    return m


@lru_cache(maxsize=None)
def orderings(tree):
    """dict-like tuple of ((ordering tuple), sign) for a tree term."""
    if tree[0] == "g":
        return (((tree[1],), 1),)
    acc = {}

    def add(o, s):
        acc[o] = acc.get(o, 0) + s

    if tree[0] == "v3":
        for oa, sa in orderings(tree[1]):
            for ob, sb in orderings(tree[2]):
                add(oa + ob, sa * sb)
                add(ob + oa, -sa * sb)
    else:
        for oa, sa in orderings(tree[1]):
            for om, sm in orderings(tree[2]):
                for oc, sc in orderings(tree[3]):
                    s = sa * sm * sc
                    add(oa + om + oc, s)
                    add(oc + om + oa, s)
                    add(om + oc + oa, -s)
                    add(oa + oc + om, -s)
    return tuple(sorted((o, s) for o, s in acc.items() if s != 0))


def ordered_block_partitions(items):
    """All ordered sequences of disjoint non-empty blocks (sorted tuples) covering `items`."""
    items = tuple(items)
    if not items:
        yield ()
        return
    n = len(items)
    for mask in range(1, 1 << n):
        first = tuple(items[i] for i in range(n) if mask >> i & 1)
        rest = tuple(items[i] for i in range(n) if not mask >> i & 1)
        for tail in ordered_block_partitions(rest):
            yield (first,) + tail


def diagram_terms(n):
    """All diagram terms of g g -> t t~ + (n-2) g: list of tuples of trees (blocks from t to t~)."""
    out = []
    for blocks in ordered_block_partitions(range(n)):
        def rec(i, acc):
            if i == len(blocks):
                out.append(tuple(acc))
                return
            for t in gluon_tree_terms(blocks[i]):
                rec(i + 1, acc + [t])
        rec(0, [])
    return out


def n_feynman_diagrams(terms):
    """Feynman-diagram count: a diagram with q four-gluon vertices was split into 2^q terms."""
    tot = 0
    for d in terms:
        q = sum(n_four_vertices(t) for t in d)
        tot += 1.0 / (1 << q)
    return int(round(tot))


def flow_index_table(n):
    """Colour flows = permutations of range(n) in lexicographic order -> index."""
    return {p: i for i, p in enumerate(permutations(range(n)))}


def term_flows(term, flow_index):
    """[(flow index, sign)] for one diagram term (tuple of block trees)."""
    acc = [((), 1)]
    for t in term:
        acc = [(o + ot, s * st) for o, s in acc for ot, st in orderings(t)]
    d = {}
    for o, s in acc:
        d[flow_index[o]] = d.get(flow_index[o], 0) + s
    return tuple(sorted((f, s) for f, s in d.items() if s != 0))
