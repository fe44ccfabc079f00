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

# static FLOP counts per routine (DFMA = 2, DMUL/DADD = 1), counted from the expressions in mg_wave.cuh as ptxas
# contracts them (a complex product component = 1 mul + 1 fma; a 4-term dot product component = 1 mul + 7 fma, ...):
#   v3  wdot 30 + 2 pwdot 28 + (2 PB + PA, 2 PA + PB) 16 + scalings 6 + 4 components x (1 + 9 + 9) = 156
#   k   3 wdot 45 + scalings 8 + 4 components x (11 + 11) = 141
#   lq/rq  slash blocks 8 + two 2x2 complex row/column products 56 + 8 components x (1 mul + 3 fma) = 120
#   bil 16 real products-of-complex (3 each) + 24 adds = 72;  amp 2 x (1 mul + 7 fma) = 30
# Cross-checked against ncu's dadd/dmul/dfma thread-instruction counters for whole mg_sigma calls
# (profiles/r2_flops.md: static / measured = 1.00-1.03); mg_process_info() reports the static figures.
FLOPS = {"v3": 156, "k": 141, "lq": 120, "rq": 120, "bil": 72, "amp": 30, "ext_g": 30, "ext_q": 50, "jamp_add": 2}


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

    def __init__(self, n, terms=None, acc_max=6, sort=True, max_keep=0, tables=None, greedy=True):
        self.n = n
        self.tables = tables     # tables.Tables: currents that come from the per-event helicity tables are leaves
        self.flow_index = topo.flow_index_table(n)
        self.ncol = len(self.flow_index)
        all_terms = topo.diagram_terms(n)
        self.ndiagrams = topo.n_feynman_diagrams(all_terms)
        self.terms = list(all_terms if terms is None else terms)
        self.acc_max = acc_max
        self.ops = []
        # memo of internal currents, least recently used first.  max_keep > 0 bounds it: a current that has not
        # been used for a while is dropped and *recomputed* if it is needed again (rematerialisation), which keeps
        # the number of simultaneously live currents — registers — bounded at the price of a few extra FLOPs.
        from collections import OrderedDict
        self._memo = OrderedDict()
        self.max_keep = max_keep
        self._next = 0
        self.gmasks = set()      # gluon-propagator subsets
        self.lmasks = set()      # top-side quark propagators
        self.rmasks = set()      # antitop-side quark propagators
        self.blocks = {}         # block key -> dict(id, nacc, flows[a] = [(flow, sign)], last_amp_index)
        self._build(sort, greedy)

    def _new(self):
        self._next += 1
        return "w%d" % (self._next - 1)

    # ---- currents ----
    def _get(self, key):
        if key in self._memo:
            self._memo.move_to_end(key)
            return self._memo[key]
        return None

    def _put(self, key, name):
        self._memo[key] = name
        if self.max_keep:
            while len(self._memo) > self.max_keep:
                self._memo.popitem(last=False)
        return name

    def g(self, tree):
        if self.tables is not None and self.tables.has_gluon(tree):
            return self.tables.gluon(tree)["name"]
        if tree[0] == "g":
            return "e%d" % tree[1]
        hit = self._get(("g", tree))
        if hit:
            return hit
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
        return self._put(("g", tree), out)

    def l(self, chain):
        if self.tables is not None and self.tables.has_chain(chain):
            return self.tables.lchain(chain)["name"]
        if not chain:
            return "ub"
        hit = self._get(("l", chain))
        if hit:
            return hit
        prev = self.l(chain[:-1])
        gc = self.g(chain[-1])
        mask = 0
        for t in chain:
            mask |= topo.leafmask(t)
        self.lmasks.add(mask)
        out = self._new()
        self.ops.append(("lq", out, prev, gc, mask))
        return self._put(("l", chain), out)

    def r(self, chain):
        if self.tables is not None and self.tables.has_chain(chain):
            return self.tables.rchain(chain)["name"]
        if not chain:
            return "vv"
        hit = self._get(("r", chain))
        if hit:
            return hit
        nxt = self.r(chain[1:])
        gc = self.g(chain[0])
        mask = 0
        for t in chain:
            mask |= topo.leafmask(t)
        self.rmasks.add(mask)
        out = self._new()
        self.ops.append(("rq", out, nxt, gc, mask))
        return self._put(("r", chain), out)

    def b(self, lchain, rchain):
        hit = self._get(("b", lchain, rchain))
        if hit:
            return hit
        ln, rn = self.l(lchain), self.r(rchain)
        out = self._new()
        self.ops.append(("bil", out, ln, rn))
        return self._put(("b", lchain, rchain), out)

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

    def _build(self, sort, greedy=True):
        keyed = []
        for term in self.terms:
            c = closure_block(term)
            keyed.append((term[:c], term[c + 1:], term[c], term))
        if sort:
            keyed.sort(key=lambda k: amp_sort_key(k[0], k[1], k[2], self.acc_max, self.n))
            if greedy:
                keyed = _greedy_order(keyed, self.acc_max, self.tables)
        self.namps = 0
        open_blocks = []
        for lchain, rchain, mid, term in keyed:
            bn = self.b(lchain, rchain)
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
        """Peak live state in program order, in units of one current (8 doubles): internal currents plus open
        JAMP accumulators (a quarter each) — the register-pressure proxy the phase splitting is steered by."""
        last = {}
        for i, op in enumerate(self.ops):
            for nm in _inputs(op):
                last[nm] = i
        acc_last = {}
        for i, op in enumerate(self.ops):
            if op[0] == "flush":
                acc_last[(op[1], op[2])] = i
        live, accs, peak = set(), set(), 0.0
        for i, op in enumerate(self.ops):
            if op[0] not in ("amp", "flush"):
                live.add(op[1])
            if op[0] == "amp":
                accs.update((b_, a) for b_, a, _ in op[3])
            peak = max(peak, len(live) + 0.25 * len(accs))
            for nm in _inputs(op):
                if last.get(nm) == i and nm in live:
                    live.discard(nm)
            if op[0] == "flush" and acc_last.get((op[1], op[2])) == i:
                accs.discard((op[1], op[2]))
        return int(peak + 0.75)


# ------------------------------------------------------------------------------------------ amplitude order
def _tabled(key, tables):
    if tables is None:
        return False
    if key[0] == "g":
        return tables.has_gluon(key[1])
    if key[0] in ("l", "r"):
        return tables.has_chain(key[1])
    return False


def _deps(key, tables=None):
    """Direct inputs (as memo keys) of an internal current; external wavefunctions and currents that come from the
    per-event tables are not listed."""
    if tables is not None:
        return [d for d in _deps(key) if not _tabled(d, tables)]
    kind = key[0]
    if kind == "g":
        return [("g", c) for c in key[1][1:] if c[0] != "g"]
    if kind == "l":
        chain = key[1]
        return ([("l", chain[:-1])] if len(chain) > 1 else []) + ([("g", chain[-1])] if chain[-1][0] != "g" else [])
    if kind == "r":
        chain = key[1]
        return ([("r", chain[1:])] if len(chain) > 1 else []) + ([("g", chain[0])] if chain[0][0] != "g" else [])
    if kind == "b":
        return ([("l", key[1])] if key[1] else []) + ([("r", key[2])] if key[2] else [])
    raise AssertionError(kind)


def _amp_accs(mid, acc_max):
    """(skeleton key, accumulator ids) of the amplitude of a mid tree: see Plan._block."""
    from itertools import product
    skel, frontier = skeleton(mid, acc_max)
    combos = [tuple(c[0] for c in choice) for choice in product(*[topo.orderings(f) for f in frontier])]
    return skeleton_key(skel, frontier), combos


def _greedy_order(keyed, acc_max, tables=None):
    """Register-pressure-aware order of the amplitudes (list scheduling on the current DAG): repeatedly take the
    amplitude that adds the least live state — not-yet-computed currents (8 doubles each) and newly opened JAMP
    accumulators (2 doubles each) — net of what it lets die (currents whose consumers are all done, accumulator
    blocks whose last amplitude this is); ties keep the locality order given.  No current is computed twice."""
    namp = len(keyed)
    roots, closure, blocks, accs = [], [], [], []
    consumers = {}           # current key -> number of direct consumers (currents or amplitudes) still to come
    block_left = {}          # block key -> amplitudes still to come
    seen_nodes = set()
    for lchain, rchain, mid, term in keyed:
        r_ = [("b", lchain, rchain)] + ([("g", mid)] if mid[0] != "g" and not _tabled(("g", mid), tables) else [])
        roots.append(r_)
        clo, stack = [], list(r_)
        while stack:
            k = stack.pop()
            if k in clo:
                continue
            clo.append(k)
            stack.extend(_deps(k, tables))
        closure.append(clo)
        sk, combos = _amp_accs(mid, acc_max)
        bkey = (lchain, rchain, sk)
        blocks.append(bkey)
        accs.append([(bkey, c) for c in combos])
        block_left[bkey] = block_left.get(bkey, 0) + 1
        for k in r_:
            consumers[k] = consumers.get(k, 0) + 1
        for k in clo:
            if k not in seen_nodes:
                seen_nodes.add(k)
                for d in _deps(k, tables):
                    consumers[d] = consumers.get(d, 0) + 1
    computed = set()
    open_accs = {}           # block key -> set of open accumulator ids
    remaining = list(range(namp))
    order = []
    while remaining:
        best, best_score = None, None
        for pos, i in enumerate(remaining):
            new = [k for k in closure[i] if k not in computed]
            dec = {}
            for k in new:
                for d in _deps(k, tables):
                    dec[d] = dec.get(d, 0) + 1
            for k in roots[i]:
                dec[k] = dec.get(k, 0) + 1
            freed = sum(1 for k, v in dec.items() if consumers[k] - v == 0)
            opened = open_accs.get(blocks[i], ())
            new_acc = sum(1 for a in accs[i] if a not in opened)
            freed_acc = (len(opened) + new_acc) if block_left[blocks[i]] == 1 else 0
            score = (8 * (len(new) - freed) + 2 * (new_acc - freed_acc), len(new), pos)
            if best_score is None or score < best_score:
                best, best_score = i, score
            if score[0] < 0 or (score[0] == 0 and score[1] == 0):
                break           # shrinks (or keeps) the live set right away: take it
        i = best
        for k in closure[i]:
            if k not in computed:
                computed.add(k)
                for d in _deps(k, tables):
                    consumers[d] -= 1
        for k in roots[i]:
            consumers[k] -= 1
        block_left[blocks[i]] -= 1
        if block_left[blocks[i]] == 0:
            open_accs.pop(blocks[i], None)
        else:
            open_accs.setdefault(blocks[i], set()).update(accs[i])
        order.append(keyed[i])
        remaining.remove(i)
    return order


def anchor_of(mid, th=4):
    """The sub-tree whose current is the transient object shared by neighbouring amplitudes: for a mid tree
    v3(T, leaf) with |T| >= th the big child T, else the mid tree itself."""
    if mid[0] == "v3":
        for big, small in ((mid[1], mid[2]), (mid[2], mid[1])):
            if small[0] == "g" and len(topo.leaves_of(big)) >= th:
                return big
    return mid


def group_key(term, n):
    """(coarse, fine) locality key of a term.  Terms with the same coarse key go into the same kernel (they feed
    the same few colour flows); terms with the same fine key share their expensive currents and form a *phase*
    (its own Plan: the few low-multiplicity currents it shares with other phases are recomputed, so that very
    little is live across phases)."""
    th = max(n - 1, 2)
    c = closure_block(term)
    mid = term[c]
    anc = anchor_of(mid, th)
    la = topo.leaves_of(anc)

    def big_child(t):
        if t[0] == "g":
            return ()
        kids = sorted(t[1:], key=lambda k: -len(topo.leaves_of(k)))
        return tuple(sorted(topo.leaves_of(kids[0])))

    if th <= len(la) < n:
        return ("A", tuple(sorted(la))), big_child(anc)
    if len(la) >= n:
        return ("T", "all"), (mid[0], big_child(mid))      # one coarse class: every T kernel touches most flows
    # quark-line dominated terms: keyed by the gluon *set* on the top side of the closing block (the terms of a set
    # share all their top-side chains and need antitop-side chains over the complement only), then by the closing
    # block; terms closed on their first block are keyed by that block
    def mask(ts):
        out = ()
        for t in ts:
            out += tuple(topo.leaves_of(t))
        return tuple(sorted(out))

    if c > 0:
        return ("L", mask(term[:c])), tuple(sorted(topo.leaves_of(mid)))
    return ("R", tuple(sorted(topo.leaves_of(mid)))), mask(term[c + 1:c + 2])


def family_key(term, n):
    """Permutation-equivariant class of a term: (kind, gluon set).  Classes of one kind and set size are relabelings of
    each other (emit_coop.py runs the code of one of them for all).  Kinds: "A" the (n-1)-gluon set of the closing
    tree, "L" the gluon set on the top side of the closing block, "R" the closing block itself (terms closed on their
    first block), "Tv3"/"Tk" the big child of the root vertex of a single-block n-gluon tree."""
    ck, fk = group_key(term, n)
    if ck[0] == "T":
        mid = term[closure_block(term)]
        sizes = sorted(len(topo.leaves_of(c)) for c in mid[1:])
        if len(sizes) == 3 and sizes[1] == sizes[2] and sizes[0] < sizes[1]:
            # gggg root with two equally large children: "the big child" is a tie; the odd one out is unique
            small = min(mid[1:], key=lambda c: len(topo.leaves_of(c)))
            return "Tk1", tuple(sorted(topo.leaves_of(small)))
        return "T" + fk[0], fk[1]
    return ck[0], ck[1]


def amp_sort_key(lchain, rchain, mid, acc_max, n):
    term = lchain + (mid,) + rchain
    gk = group_key(term, n)
    gk = (gk[0][0], gk[0][1], gk[1])
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
def partition_terms(n, max_terms=170, max_phase=32):
    """Splits the terms of g g -> t t~ + (n-2) g into kernels and phases: returns a list of kernels, each a list
    of phases, each a list of terms.  Coarse keys (group_key) make kernels — small ones are bin-packed up to
    `max_terms` —, fine keys make phases, bin-packed up to `max_phase` terms."""
    terms = topo.diagram_terms(n)
    coarse = {}
    for term in terms:
        ck, fk = group_key(term, n)
        coarse.setdefault(ck, {}).setdefault(fk, []).append(term)

    def phases_of(fine):
        out, cur = [], []
        for fk in sorted(fine, key=repr):
            b = fine[fk]
            cls = fk[0][0] if isinstance(fk[0], tuple) else fk[0]
            limit = max_phase.get(cls, max_phase.get("*", 32)) if isinstance(max_phase, dict) else max_phase
            if cur and len(cur) + len(b) > limit:
                out.append(cur)
                cur = []
            cur = cur + b
        if cur:
            out.append(cur)
        return out

    kernels, cur, cur_n = [], {}, 0
    for ck in sorted(coarse, key=repr):
        fine = {(ck, fk): v for fk, v in coarse[ck].items()}
        nt = sum(len(v) for v in fine.values())
        if ck[0] in ("A", "T") or nt >= max_terms:
            kernels.append(phases_of(fine))
            continue
        if cur and cur_n + nt > max_terms:
            kernels.append(phases_of(cur))
            cur, cur_n = {}, 0
        cur.update(fine)
        cur_n += nt
    if cur:
        kernels.append(phases_of(cur))
    assert sum(len(p) for k in kernels for p in k) == len(terms)
    return kernels
