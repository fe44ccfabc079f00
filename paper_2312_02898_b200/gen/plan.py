"""Current scheduling for g g -> t t~ + (n-2) g  (K0 -> K4/K5 of SURVEY.md §8a).

Every diagram term (topology.py) is a sequence of gluon-tree blocks tau_1..tau_m along the quark line.  It is
evaluated by closing the line on one block c:
     A = Lbar(tau_1..tau_{c-1}) . Gslash(tau_c) . R(tau_{c+1}..tau_m) = B_mu(L, R) G^mu(tau_c)
with  Lbar(chain) the row-spinor current grown from ubar(p_t),  R(chain) the column-spinor current grown from
v(p_t~), G(tree) the off-shell gluon current of a block, and B the fermion bilinear shared by all terms with
the same (L, R).  Currents are memoised by structure, so sub-diagrams are computed once per helicity pass
(the "wavefunction recycling" of the diagram-based method, PAPER.md:45/:97 `matrix1_`).

The plan is a flat list of ops in evaluation order:
   ("v3", out, A, B, maskA, maskB)      gluon current from a ggg vertex
   ("k",  out, A, M, C, mask)           gluon current from one gggg kinematic structure
   ("lq", out, Lprev, G, mask)          quark line, top side;    mask = gluons absorbed so far (incl. G)
   ("rq", out, Rnext, G, mask)          quark line, antitop side
   ("bil", out, L, R)                   B_mu = L gamma_mu R
   ("amp", B, G, flows)                 A = B.G ; JAMP[f] += sign*A for (f, sign) in flows
Names: external gluons "e<i>", "ub" (ubar(p_t)), "vv" (v(p_t~)); internal "w<k>".
"""
from . import topology as topo

# static FLOP counts per routine (DFMA = 2, DMUL/DADD = 1), counted from mg_wave.cuh by hand; used only
# for mg_process_info()'s algorithmic FLOP figure — measured FLOPs come from ncu.
FLOPS = {"v3": 4 * 7 + 2 * 7 * 2 + 12 + 6 + 4 * (1 + 9 * 2 + 1), "k": 3 * 4 * 7 + 8 + 4 * 2 * 11,
         "lq": 8 + 2 * 28 + 8 + 8 * 9, "rq": 8 + 2 * 28 + 8 + 8 * 9, "bil": 16 * 3 + 24, "amp": 4 * 7,
         "ext_g": 30, "ext_q": 50, "jamp_add": 2}


class Plan:
    def __init__(self, n, closure="largest"):
        self.n = n
        self.flow_index = topo.flow_index_table(n)
        self.ncol = len(self.flow_index)
        self.terms = topo.diagram_terms(n)
        self.ndiagrams = topo.n_feynman_diagrams(self.terms)
        self.ops = []
        self._g = {}
        self._l = {(): "ub"}
        self._r = {(): "vv"}
        self._b = {}
        self._next = 0
        self.gmasks = set()      # gluon-propagator subsets
        self.lmasks = set()      # top-side quark propagators
        self.rmasks = set()      # antitop-side quark propagators
        self.closure = closure
        self._build()

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

    def _closure_block(self, term):
        sizes = [len(topo.leaves_of(t)) for t in term]
        m = len(term)
        if self.closure == "largest":
            best = max(range(m), key=lambda i: (sizes[i], -abs(i - (m - 1) / 2.0)))
        else:
            best = (m - 1) // 2
        return best

    def _build(self):
        # order terms so that terms sharing (L chain, R chain) are adjacent
        keyed = []
        for term in self.terms:
            c = self._closure_block(term)
            keyed.append((term[:c], term[c + 1:], term[c], term))
        keyed.sort(key=lambda k: (len(k[0]) + len(k[1]), repr(k[0]), repr(k[1]), repr(k[2])))
        self.namps = 0
        for lchain, rchain, mid, term in keyed:
            ln = self.l(lchain)
            rn = self.r(rchain)
            bn = self.b(ln, rn)
            gn = self.g(mid)
            flows = topo.term_flows(term, self.flow_index)
            self.ops.append(("amp", bn, gn, flows))
            self.namps += 1

    # ---- statistics ----
    def counts(self):
        c = {}
        for op in self.ops:
            c[op[0]] = c.get(op[0], 0) + 1
        c["jamp_add"] = sum(len(op[3]) for op in self.ops if op[0] == "amp")
        return c

    def flops_per_helicity(self, colour=True):
        c = self.counts()
        f = sum(FLOPS[k] * v for k, v in c.items())
        f += self.n * FLOPS["ext_g"] + 2 * FLOPS["ext_q"]
        if colour:
            # symmetric quadratic form: per i: 2 FMA per j>i, plus 2 FMA + 2 FMA
            f += 2 * (self.ncol * (self.ncol - 1) // 2) * 2 + self.ncol * 8
        return f

    def max_live(self):
        """Peak number of simultaneously live internal currents in program order (register-pressure proxy)."""
        last = {}
        for i, op in enumerate(self.ops):
            for nm in _inputs(op):
                last[nm] = i
        live, peak = set(), 0
        for i, op in enumerate(self.ops):
            if op[0] != "amp":
                live.add(op[1])
            peak = max(peak, len(live))
            for nm in _inputs(op):
                if last.get(nm) == i and nm in live:
                    live.discard(nm)
        return peak


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
