"""Per-event helicity tables of the low-multiplicity currents (helicity recycling).

A current depends only on the helicities of its own legs: an off-shell gluon current over k external gluons has
2^k variants, a quark-line current that has absorbed k gluons 2^(k+1) — not 2^npar.  The event-CTA kernel shape
(emit_coop.py) therefore computes every current up to a multiplicity threshold *once per event* for all of its
variants, cooperatively (one thread per (current, variant)), into a shared-memory table; the diagram-group bodies
read the variant that matches their thread's helicity.  These are exactly the currents the diagram groups would
otherwise recompute (they are shared by many groups), so the tables remove the recomputation between groups and
most of the per-helicity cost of the low-multiplicity sub-diagrams.

Table layout (element type T): item at offset `off`, `nv` = 2^nbits variants, component c (0..3 = Re, 4..7 = Im of
the four complex components) of variant v at  off + c * nv + v.  Variant index: bit j of v is the helicity bit
(1 <=> lambda = +1) of particle bits[j]; bits = the item's gluon leaves in ascending order, preceded by the antitop for
antitop-side chains.  The top-quark helicity is NOT a variant bit: the kernel works on slots = (event, lambda_t), so
it is fixed while a table is alive (half the top-side chain tables, and a run that uses the helicity-flip symmetry
|M(-h)|^2 = |M(h)|^2 only ever builds lambda_t = +1).
"""
from . import topology as topo

KIND = {"eg": 0, "q": 1, "v3": 2, "k": 3, "lq": 4, "rq": 5, "kz": 6}


def gluon_particle(i):
    """Process order g g t t~ g ...: gluon i is particle i (beams) or i + 2 (final state)."""
    return i if i < 2 else i + 2


class Tables:
    def __init__(self, n, gtab, qtab):
        """gtab: gluon currents over <= gtab leaves are tabled (externals always are); qtab: quark-line currents
        that have absorbed <= qtab gluons are tabled (the external spinors always are)."""
        self.n, self.gtab, self.qtab = n, max(gtab, 1), max(qtab, 0)
        self.items = {}       # key -> item dict
        self.order = []       # keys in dependency order
        self.ext = {}

    # ---- registration ----
    def _add(self, key, kind, bits, inputs, inv, level, name):
        it = dict(key=key, kind=kind, bits=tuple(bits), inputs=tuple(inputs), inv=tuple(inv), level=level, name=name,
                  nv=1 << len(bits), off=None)
        self.items[key] = it
        self.order.append(key)
        return it

    def ext_gluon(self, i):
        key = ("e", i)
        if key not in self.items:
            self._add(key, "eg", [gluon_particle(i)], [], ["eg%d" % i], 0, "e%d" % i)
        return self.items[key]

    def ext_quark(self, which):
        key = ("q", which)           # "ub" = ubar(p_t), "vv" = v(p_tb)
        if key not in self.items:
            self._add(key, "q", [] if which == "ub" else [3], [], [which], 0, which)
        return self.items[key]

    def has_gluon(self, tree):
        return len(topo.leaves_of(tree)) <= self.gtab

    def gluon(self, tree):
        if tree[0] == "g":
            return self.ext_gluon(tree[1])
        key = ("g", tree)
        if key in self.items:
            return self.items[key]
        leaves = sorted(topo.leaves_of(tree))
        mask = topo.leafmask(tree)
        if tree[0] == "kz":
            # the eliminated four-gluon structure K_Z = -K_X - K_Y (parts x, y, z by smallest leaf), kept in the
            # event-wide tables so that every relabelled entry is a plain copy of one item
            x, y, z = tree[1:]
            kids = [self.gluon(("k", y, x, z)), self.gluon(("k", x, y, z))]
            return self._add(key, "kz", [gluon_particle(i) for i in leaves], [k["key"] for k in kids], [], len(leaves),
                             "tg%d" % len(self.items))
        kids = [self.gluon(c) for c in tree[1:]]
        if tree[0] == "v3":
            inv = ["pm%d" % topo.leafmask(tree[1]), "pm%d" % topo.leafmask(tree[2]), "sg%d" % mask]
        else:
            inv = ["sg%d" % mask]
        return self._add(key, tree[0], [gluon_particle(i) for i in leaves], [k["key"] for k in kids], inv,
                         len(leaves), "tg%d" % len(self.items))

    @staticmethod
    def _chain_gluons(chain):
        out = []
        for t in chain:
            out += list(topo.leaves_of(t))
        return out

    def has_chain(self, chain):
        return len(self._chain_gluons(chain)) <= self.qtab and all(self.has_gluon(t) for t in chain)

    def lchain(self, chain):
        if not chain:
            return self.ext_quark("ub")
        key = ("l", chain)
        if key in self.items:
            return self.items[key]
        prev, g = self.lchain(chain[:-1]), self.gluon(chain[-1])
        gl = sorted(self._chain_gluons(chain))
        mask = sum(1 << i for i in gl)
        return self._add(key, "lq", [gluon_particle(i) for i in gl], [prev["key"], g["key"]], ["tl%d" % mask],
                         len(gl), "tl%d" % len(self.items))

    def rchain(self, chain):
        if not chain:
            return self.ext_quark("vv")
        key = ("r", chain)
        if key in self.items:
            return self.items[key]
        nxt, g = self.rchain(chain[1:]), self.gluon(chain[0])
        gl = sorted(self._chain_gluons(chain))
        mask = sum(1 << i for i in gl)
        return self._add(key, "rq", [3] + [gluon_particle(i) for i in gl], [nxt["key"], g["key"]], ["tr%d" % mask],
                         len(gl), "tr%d" % len(self.items))

    # ---- layout / build schedule ----
    def layout(self):
        """Assigns offsets; returns the table length in elements (even)."""
        off = 0
        for key in self.order:
            it = self.items[key]
            it["off"] = off
            off += 8 * it["nv"]
        self.size = off + (off & 1)
        self.by_name = {it["name"]: it for it in self.items.values()}
        return self.size

    def groups(self):
        """Build groups in dependency order: items of one group have the same kind and number of variants (one
        uniform loop in the kernel) and depend only on earlier rounds.  Returns [(kind, nbits, [items], sync_after)]:
        sync_after marks the last group of a round (the CTA synchronises before it reads what the round wrote)."""
        done, out = set(), []
        todo = [self.items[k] for k in self.order]
        while todo:
            ready = [it for it in todo if all(k in done for k in it["inputs"])]
            assert ready
            sig = {}
            for it in ready:
                sig.setdefault((it["kind"], len(it["bits"])), []).append(it)
            rnd = sorted(sig.items(), key=lambda kv: (KIND[kv[0][0]], kv[0][1]))
            for i, ((kind, nb), its) in enumerate(rnd):
                out.append((kind, nb, its, i == len(rnd) - 1))
            done.update(it["key"] for it in ready)
            todo = [it for it in todo if it["key"] not in done]
        return out

    def flops(self):
        """Static FLOPs of building all tables once (per event)."""
        from .plan import FLOPS
        cost = {"v3": FLOPS["v3"], "k": FLOPS["k"], "lq": FLOPS["lq"], "rq": FLOPS["rq"], "eg": 0, "q": 0, "kz": 8}
        return sum(cost[it["kind"]] * it["nv"] for it in self.items.values())

    def inv_names(self):
        s = set()
        for it in self.items.values():
            s.update(it["inv"])
        return s

    def register_all(self):
        """Registers every current the thresholds allow: all trees over <= gtab gluons, all chains that have absorbed
        <= qtab gluons (the event-wide tables the relabelled views of the bodies are gathered from)."""
        from itertools import combinations
        gl = range(self.n)
        for i in gl:
            self.ext_gluon(i)
        self.ext_quark("ub")
        self.ext_quark("vv")
        for k in range(2, self.gtab + 1):
            for S in combinations(gl, k):
                for t in topo.gluon_tree_terms(S):
                    self.gluon(t)
                    if t[0] == "k" and min(topo.leaves_of(t[1])) < min(topo.leaves_of(t[2])):     # the K_Y term: parts in order
                        self.gluon(("kz", t[1], t[2], t[3]))
        for k in range(1, self.qtab + 1):
            for S in combinations(gl, k):
                for blocks in topo.ordered_block_partitions(S):
                    def rec(i, acc):
                        if i == len(blocks):
                            self.lchain(tuple(acc))
                            self.rchain(tuple(acc))
                            return
                        for t in topo.gluon_tree_terms(tuple(sorted(blocks[i]))):
                            if self.has_gluon(t):
                                rec(i + 1, acc + [t])
                    rec(0, [])
        return self

    # ---- relabelling: the current that plays the role of item `key` when canonical gluon i is gluon pi[i] ----
    def relabel(self, key, pi):
        """[(sign, key')]: the relabelled current as a signed sum of registered (canonical-embedding) items."""
        kind = key[0]
        if kind == "e":
            return [(1, ("e", pi[key[1]]))]
        if kind == "q":
            return [(1, key)]
        if kind == "g":
            return [(s, ("g", t)) for s, t in relabel_tree(key[1], pi)]
        out = [(1, ())]
        for t in key[1]:
            out = [(s * st, ch + (tt,)) for s, ch in out for st, tt in relabel_tree(t, pi)]
        return [(s, (kind, ch)) for s, ch in out]

    def selector(self, parent, child):
        """Packed 4-bit positions: bit j of the child's variant index is bit sel_j of the parent's."""
        sel = 0
        for j, q in enumerate(child["bits"]):
            sel |= parent["bits"].index(q) << (4 * j)
        return sel


def relabel_tree(tree, pi):
    """Tree with every leaf i replaced by pi[i], brought to the canonical embedding of topology.gluon_tree_terms
    (children of a ggg vertex ordered by smallest leaf: a swap costs a sign; a gggg structure whose middle part is the
    one with the largest smallest-leaf is the "kz" item K_Z = -K_X - K_Y).  Returns [(sign, canonical tree)]."""
    if tree[0] == "g":
        return [(1, ("g", pi[tree[1]]))]
    kids = [relabel_tree(c, pi) for c in tree[1:]]
    out = []
    if tree[0] == "v3":
        for sa, a in kids[0]:
            for sb, b in kids[1]:
                if min(topo.leaves_of(a)) < min(topo.leaves_of(b)):
                    out.append((sa * sb, ("v3", a, b)))
                else:
                    out.append((-sa * sb, ("v3", b, a)))
        return out
    for sa, a in kids[0]:
        for sm, m in kids[1]:
            for sc, c in kids[2]:
                s = sa * sm * sc
                x, y, z = sorted((a, m, c), key=lambda t: min(topo.leaves_of(t)))
                if m is x:
                    out.append((s, ("k", y, x, z)))
                elif m is y:
                    out.append((s, ("k", x, y, z)))
                else:
                    out.append((s, ("kz", x, y, z)))
    return out
