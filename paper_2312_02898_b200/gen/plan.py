"""Current scheduling for g g -> t t~ + (n-2) g  (K0 -> K4/K5 of SURVEY.md §8a).

Every diagram term (topology.py) is a sequence of gluon-tree blocks tau_1..tau_m along the quark line.  It is
evaluated by closing the line on one block c:
     A = Lbar(tau_1..tau_{c-1}) . Gslash(tau_c) . R(tau_{c+1}..tau_m) = B_mu(L, R) G^mu(tau_c)
with  Lbar(chain) the row-spinor current grown from ubar(p_t),  R(chain) the column-spinor current grown from
v(p_t~), G(tree) the off-shell gluon current of a block, and B the fermion bilinear shared by all terms with
the same (L, R).  Currents are memoised by structure, so sub-diagrams are computed once per helicity pass
(the "wavefunction recycling" of the diagram-based method, PAPER.md:45/:97 `matrix1_`).

Diagram *groups* (north_star subsystem (2): "per-diagram-group splitting ... where register pressure would
spill"): the terms of a process are partitioned into groups; each group gets its own Plan (it recomputes the
few low-multiplicity currents it shares with other groups) and becomes one kernel.

Hierarchical JAMP accumulation: the amplitude of a term feeds the colour flows
     prefix(L) . orderings(mid tree) . suffix(R),
and orderings() factorises over the tree (topology.py).  Amplitudes whose mid trees share a *skeleton* (the
tree truncated to a frontier of sub-trees, identified by their leaf sets) and the same (L, R) form an
accumulation *block*: they are summed into a few register accumulators indexed by the frontier sub-trees'
own orderings, and each accumulator is flushed once to all flows of the skeleton.  This turns
sum_terms |flows(term)| complex additions on the JAMPs into far fewer.

The plan is a flat list of ops in evaluation order:
   ("v3", out, A, B, maskA, maskB)      gluon current from a ggg vertex
   ("k",  out, A, M, C, mask)           gluon current from one gggg kinematic structure
   ("lq", out, Lprev, G, mask)          quark line, top side;    mask = gluons absorbed so far (incl. G)
   ("rq", out, Rnext, G, mask)          quark line, antitop side
   ("bil", out, L, R)                   B_mu = L gamma_mu R
   ("amp", B, G, accs)                  A = B.G ; acc[block][a] += sign*A for (block, a, sign) in accs
   ("flush", block, a, flows)           JAMP[f] += sign*acc[block][a] for (f, sign) in flows
Names: external gluons "e<i>", "ub" (ubar(p_t)), "vv" (v(p_t~)); internal "w<k>".
"""
from math import factorial

from . import topology as topo

# static FLOP counts per routine (DFMA = 2, DMUL/DADD = 1), counted from mg_wave.cuh by hand; used only
# for mg_process_info()'s algorithmic FLOP figure — measured FLOPs come from ncu.
FLOPS = {"v3": 4 * 7 + 2 * 7 * 2 + 12 + 6 + 4 * (1 + 9 * 2 + 1), "k": 3 * 4 * 7 + 8 + 4 * 2 * 11,
         "lq": 8 + 2 * 28 + 8 + 8 * 9, "rq": 8 + 2 * 28 + 8 + 8 * 9, "bil": 16 * 3 + 24, "amp": 4 * 7,
         "ext_g": 30, "ext_q": 50, "jamp_add": 2}


def closure_block(term):
    """Index of the block the quark line is closed on: the largest one, ties -> the most central."""
    sizes = [len(topo.leaves_of(t)) for t in term]
    m = len(term)
    return max(range(m), key=lambda i: (sizes[i], -abs(i - (m - 1) / 2.0)))


# ------------------------------------------------------------------------------------------ skeletons
def _nperm(tree):
    return factorial(len(topo.leaves_of(tree)))


def skeleton(tree, acc_max):
    """Truncates `tree` to a frontier of sub-trees such that prod |leaves(sub)|! <= acc_max.
    Returns (skel, frontier): skel is the tree with frontier sub-trees replaced by ("g", -1-k) pseudo leaves
    (k = index into frontier), frontier the list of cut sub-trees (in pseudo-leaf order)."""
    frontier = [tree]

    def cost():
        c = 1
        for t in frontier:
            c *= _nperm(t)
        return c

    while cost() > acc_max:
        # expand the largest frontier sub-tree into its children
        k = max(range(len(frontier)), key=lambda i: _nperm(frontier[i]))
        t = frontier[k]
        assert t[0] != "g"
        frontier[k:k + 1] = list(t[1:])
    fr_ids = {id(t): None for t in frontier}

    def build(t):
        for k, f in enumerate(frontier):
            if f is t:
                return ("g", -1 - k)
        if t[0] == "g":
            raise AssertionError("leaf not in frontier")
        return (t[0],) + tuple(build(c) for c in t[1:])

    return build(tree), frontier


def skeleton_key(skel, frontier):
    """Hashable identity of a skeleton: structure + the leaf sets of its frontier sub-trees."""
    return (skel, tuple(tuple(sorted(topo.leaves_of(f))) for f in frontier))


class Plan:
    """Ops for an ordered list of terms (default: all terms of the process, sorted for locality)."""

    def __init__(self, n, terms=None, acc_max=6, sort=True):
        self.n = n
        self.flow_index = topo.flow_index_table(n)
        self.ncol = len(self.flow_index)
        all_terms = topo.diagram_terms(n)
        self.ndiagrams = topo.n_feynman_diagrams(all_terms)
        self.terms = list(all_terms if terms is None else terms)
        self.acc_max = acc_max
        self.ops = []
        self._g = {}
        self._l = {(): "ub"}
        self._r = {(): "vv"}
        self._b = {}
        self._next = 0
        self.gmasks = set()      # gluon-propagator subsets
        self.lmasks = set()      # top-side quark propagators
        self.rmasks = set()      # antitop-side quark propagators
        self.blocks = {}         # block key -> dict(id, nacc, flows[a] = [(flow, sign)], last_amp_index)
        self._build(sort)

    def _new(self):
        self._next += 1
        return "w%d" % (self._next - 1)

    # ---- currents ----
    def g(self, tree):
        if tree[0] == "g":
            return "e%d" % tree[1]
        if tree in self._g:
            return self._g[tree]
        mask = topo.leafmask(tree)
        self.gmasks.add(mask)
        if tree[0] == "v3":
            a, b = self.g(tree[1]), self.g(tree[2])
            out = self._new()
            self.ops.append(("v3", out, a, b, topo.leafmask(tree[1]), topo.leafmask(tree[2])))
        else:
            a, m, c = self.g(tree[1]), self.g(tree[2]), self.g(tree[3])
            out = self._new()
            self.ops.append(("k", out, a, m, c, mask))
        self._g[tree] = out
        return out

    def l(self, chain):
        if chain in self._l:
            return self._l[chain]
        prev = self.l(chain[:-1])
        gc = self.g(chain[-1])
        mask = 0
        for t in chain:
            mask |= topo.leafmask(t)
        self.lmasks.add(mask)
        out = self._new()
        self.ops.append(("lq", out, prev, gc, mask))
        self._l[chain] = out
        return out

    def r(self, chain):
        if chain in self._r:
            return self._r[chain]
        nxt = self.r(chain[1:])
        gc = self.g(chain[0])
        mask = 0
        for t in chain:
            mask |= topo.leafmask(t)
        self.rmasks.add(mask)
        out = self._new()
        self.ops.append(("rq", out, nxt, gc, mask))
        self._r[chain] = out
        return out

    def b(self, lname, rname):
        key = (lname, rname)
        if key not in self._b:
            out = self._new()
            self.ops.append(("bil", out, lname, rname))
            self._b[key] = out
        return self._b[key]

    # ---- accumulation blocks ----
    def _block(self, lchain, rchain, mid):
        """Returns [(block id, acc index, sign)] for the amplitude of (lchain, mid, rchain), creating the
        block (and its flush table) on first use."""
        skel, frontier = skeleton(mid, self.acc_max)
        key = (lchain, rchain, skeleton_key(skel, frontier))
        fr_ord = [topo.orderings(f) for f in frontier]
        if key not in self.blocks:
            prefix = [((), 1)]
            for t in lchain:
                prefix = [(o + ot, s * st) for o, s in prefix for ot, st in topo.orderings(t)]
            suffix = [((), 1)]
            for t in rchain:
                suffix = [(o + ot, s * st) for o, s in suffix for ot, st in topo.orderings(t)]
            # accumulators: one per combination of frontier orderings (all permutations of each leaf set)
            from itertools import permutations, product
            fr_perms = [list(permutations(sorted(topo.leaves_of(f)))) for f in frontier]
            combos = list(product(*fr_perms))
            sk_ord = topo.orderings(skel)         # orderings of pseudo leaves -1-k
            flows = []
            for combo in combos:
                d = {}
                for po, ps in prefix:
                    for so, ss in suffix:
                        for o, s in sk_ord:
                            mid_o = ()
                            for lab in o:
                                mid_o += combo[-1 - lab]
                            f = self.flow_index[po + mid_o + so]
                            d[f] = d.get(f, 0) + ps * ss * s
                flows.append(tuple(sorted((f, s) for f, s in d.items() if s != 0)))
            self.blocks[key] = dict(id=len(self.blocks), combos={c: i for i, c in enumerate(combos)}, flows=flows,
                                    used=set(), last=None)
        blk = self.blocks[key]
        out = []
        from itertools import product
        for choice in product(*fr_ord):
            combo = tuple(c[0] for c in choice)
            sign = 1
            for c in choice:
                sign *= c[1]
            a = blk["combos"][combo]
            blk["used"].add(a)
            out.append((blk["id"], a, sign))
        return blk, out

    def _build(self, sort):
        keyed = []
        for term in self.terms:
            c = closure_block(term)
            keyed.append((term[:c], term[c + 1:], term[c], term))
        if sort:
            keyed.sort(key=lambda k: amp_sort_key(k[0], k[1], k[2], self.acc_max, self.n))
        self.namps = 0
        open_blocks = []
        for lchain, rchain, mid, term in keyed:
            ln = self.l(lchain)
            rn = self.r(rchain)
            bn = self.b(ln, rn)
            gn = self.g(mid)
            blk, accs = self._block(lchain, rchain, mid)
            # consistency: expanding the accumulators reproduces the term's flow list exactly
            d = {}
            for _, a, s in accs:
                for f, fs in blk["flows"][a]:
                    d[f] = d.get(f, 0) + s * fs
            assert tuple(sorted((f, s) for f, s in d.items() if s != 0)) == topo.term_flows(term, self.flow_index)
            self.ops.append(("amp", bn, gn, tuple(accs)))
            blk["last"] = len(self.ops) - 1
            self.namps += 1
        # insert the flushes after the last amplitude of each block
        flush_at = {}
        for blk in self.blocks.values():
            flush_at.setdefault(blk["last"], []).append(blk)
        ops = []
        for i, op in enumerate(self.ops):
            ops.append(op)
            for blk in flush_at.get(i, []):
                for a in sorted(blk["used"]):
                    ops.append(("flush", blk["id"], a, blk["flows"][a]))
        self.ops = ops
        self.block_first = {}
        for i, op in enumerate(self.ops):
            if op[0] == "amp":
                for b_, a, _ in op[3]:
                    self.block_first.setdefault((b_, a), i)

    # ---- statistics ----
    def counts(self):
        c = {}
        for op in self.ops:
            c[op[0]] = c.get(op[0], 0) + 1
        c["acc_add"] = sum(len(op[3]) for op in self.ops if op[0] == "amp")
        c["jamp_add"] = sum(len(op[3]) for op in self.ops if op[0] == "flush")
        return c

    def flops_per_helicity(self, colour=True, externals=True):
        c = self.counts()
        f = sum(FLOPS[k] * v for k, v in c.items() if k in FLOPS)
        f += 2 * c.get("acc_add", 0)
        if externals:
            f += self.n * FLOPS["ext_g"] + 2 * FLOPS["ext_q"]
        if colour:
            # symmetric quadratic form: per i: 2 FMA per j>i, plus 2 FMA + 2 FMA
            f += 2 * (self.ncol * (self.ncol - 1) // 2) * 2 + self.ncol * 8
        return f

    def flows_touched(self):
        s = set()
        for op in self.ops:
            if op[0] == "flush":
                s.update(f for f, _ in op[3])
        return s

    def max_live(self):
        """Peak number of simultaneously live internal currents in program order (register-pressure proxy)."""
        last = {}
        for i, op in enumerate(self.ops):
            for nm in _inputs(op):
                last[nm] = i
        live, peak = set(), 0
        for i, op in enumerate(self.ops):
            if op[0] not in ("amp", "flush"):
                live.add(op[1])
            peak = max(peak, len(live))
            for nm in _inputs(op):
                if last.get(nm) == i and nm in live:
                    live.discard(nm)
        return peak


def anchor_of(mid, th=4):
    """The sub-tree whose current is the transient object shared by neighbouring amplitudes: for a mid tree
    v3(T, leaf) with |T| >= th the big child T, else the mid tree itself."""
    if mid[0] == "v3":
        for big, small in ((mid[1], mid[2]), (mid[2], mid[1])):
            if small[0] == "g" and len(topo.leaves_of(big)) >= th:
                return big
    return mid


def group_key(term, n):
    """Locality key of a term: terms with the same key share their expensive currents."""
    th = max(n - 1, 2)
    c = closure_block(term)
    mid = term[c]
    anc = anchor_of(mid, th)
    la = topo.leaves_of(anc)
    if th <= len(la) < n:
        # sub-key: the (|anchor|-1)-gluon sub-tree the anchor is built on, if it is v3(sub-tree, leaf)
        sub = "x"
        if n >= 5 and anc[0] == "v3":
            for big, small in ((anc[1], anc[2]), (anc[2], anc[1])):
                if small[0] == "g" and len(topo.leaves_of(big)) == len(la) - 1:
                    sub = tuple(sorted(topo.leaves_of(big)))
        return ("A", tuple(sorted(la)), sub)
    if len(la) >= n:
        return ("T", mid[0])
    if c > 0:
        return ("L", tuple(sorted(topo.leaves_of(term[0]))))
    return ("R", tuple(sorted(topo.leaves_of(term[-1]))))


def amp_sort_key(lchain, rchain, mid, acc_max, n):
    term = lchain + (mid,) + rchain
    gk = group_key(term, n)
    anc = anchor_of(mid, max(n - 1, 2))
    skel, frontier = skeleton(anc, acc_max)
    big = gk[0] in ("A", "T")
    return (gk, 0 if big else len(lchain) + len(rchain), "" if big else repr(lchain), "" if big else repr(rchain),
            repr(skeleton_key(skel, frontier)), repr(anc), repr(mid), repr(lchain), repr(rchain))


def _inputs(op):
    k = op[0]
    if k == "v3":
        return [op[2], op[3]]
    if k == "k":
        return [op[2], op[3], op[4]]
    if k in ("lq", "rq"):
        return [op[2], op[3]]
    if k == "bil":
        return [op[2], op[3]]
    if k == "amp":
        return [op[1], op[2]]
    return []


# ------------------------------------------------------------------------------------------ diagram groups
def partition_terms(n, max_terms=170):
    """Splits the terms of g g -> t t~ + (n-2) g into diagram groups (one kernel each).
    Terms anchored on a >= 4-gluon sub-tree go with that sub-tree's leaf set (its current is computed once and
    used by every amplitude that contains it); the rest are keyed by the outermost quark-line block they share
    and bin-packed."""
    terms = topo.diagram_terms(n)
    buckets = {}
    for term in terms:
        buckets.setdefault(group_key(term, n), []).append(term)
    total = len(terms)
    if total <= max_terms:
        return [terms]
    groups = []
    small = []
    for key in sorted(buckets, key=lambda k: (k[0], k[1])):
        b = buckets[key]
        if key[0] in ("A", "T"):
            groups.append(b)
        else:
            small.append(b)
    cur = []
    for b in small:
        if cur and len(cur) + len(b) > max_terms:
            groups.append(cur)
            cur = []
        cur = cur + b
    if cur:
        groups.append(cur)
    assert sum(len(g) for g in groups) == total
    return groups
