"""Event-CTA kernel shape (n >= 4 gluons): invariants kernel + ONE persistent sigma kernel per process.

Run-time picture: csrc/mg_coop.cuh.  What this module decides at build time:

* Families.  The diagram terms are classified by a permutation-equivariant key (plan.family_key: e.g. "the (n-1)-gluon
  set of the closing tree", "the gluon set on the top side of the closing block").  All classes of one kind and set
  size are relabelings of each other (the diagram set of g g -> t t~ + gluons is symmetric under permutations of the
  gluons once every gluon carries an incoming momentum and its own polarisation table), so only the class of the
  lexicographically first set is turned into code — split into *bodies* of <= max_phase terms — and every body is
  executed once per member of its family with relabelled inputs.  That is what keeps the instruction stream warm: a
  body's code runs 4..10 times in a row per visit instead of once (measured: straight-line code that is executed once
  per visit is instruction-fetch bound at ~20 % FP64-pipe activity; the second and later passes run 2.4x faster).
* Relabelling needs no special code in the bodies: the event's helicity tables (gen/tables.py: every current up to the
  multiplicity thresholds, all helicity variants) are built once per event group into the CTA's L2-resident scratch;
  for member pi the kernel gathers the body's operands into shared memory through index maps computed here —
  invariants (mask -> pi(mask)) and table entries (the relabelled current in its canonical embedding, with the sign of
  the child swaps, K_Z = -K_X - K_Y for a four-gluon structure whose eliminated part moved into the middle, and the
  permutation of the variant bits) —, permutes the thread's helicity bits, and maps the body's colour flows through
  pi when it adds the partial JAMPs.
* Bodies are separate translation units: __noinline__ device functions (relocatable device code) that compile in
  parallel and link into the one kernel.

Workspace (element type T): inv[E][NINVP] per event tile + jamp[nCTA][NCOL][2][BLK] (nCTA = resident CTAs of the chip).
"""
from math import comb, factorial

from . import topology as topo
from .colour import colour_matrix, common_denominator
from .plan import Plan, family_key, group_key
from .tables import Tables, KIND, gluon_particle

BLK = 256      # default threads per CTA (cfg["block"])
# body sizes, table thresholds (gluon currents over <= gtab leaves and quark-line currents with <= qtab absorbed gluons
# come from the per-visit helicity tables) and the shared-memory budget, per multiplicity
# (measured on B200: gg -> tt~gg 37.9 ms with (2, 1) tables and 40-term bodies against 40.6 ms with (3, 2)
# and 24; gg -> tt~ggg with (3, 2) and 16-term bodies: 424 ms against 500 / 562 ms with 32 / 48 at that stage; l2_window: the
# scratch as a persisting L2 window, 387 -> 373 ms; gather16: 16-byte copies of groups of four table operands, 366 -> 355 ms,
# but 37.7 -> 38.3 ms at n = 4; merge_complement: classes over k- and (n - k)-subsets share bodies, 15 -> 11 visits at n = 4,
# 37.7 -> 36.6 ms (fp32 24.9 -> 22.6), no change at n = 5 (135 -> 115 visits, 355 -> 356 ms))
TUNED = {4: dict(max_phase=40, gtab=2, qtab=1, smem_kb=110, block=128, sync_every=0, merge_complement=True),
         5: dict(max_phase=16, gtab=3, qtab=2, smem_kb=110, block=128, sync_every=0, min_class=5, l2_window=True, gather16=True)}
INV_SIZE = {"sg": 1, "pm": 4, "tl": 5, "tr": 5, "eg": 5, "ub": 16, "vv": 16}
_ORDER = {"s": 0, "p": 1, "t": 2, "e": 3, "u": 4, "v": 5}


def _inv_sort(x):
    return (_ORDER[x[0]], x[:2], int(x[2:]) if x[2:].isdigit() else 0)


def _mul(s, expr):
    return expr if abs(s) == 1 else "T(%d) * %s" % (abs(s), expr)


def _perm_mask(mask, pi):
    out = 0
    for i in range(len(pi)):
        if mask >> i & 1:
            out |= 1 << pi[i]
    return out


def _perm_name(name, pi):
    """Invariant `name` of the canonical labelling -> the invariant that plays its role for relabelling pi."""
    for pre in ("sg", "pm", "tl", "tr"):
        if name.startswith(pre):
            return "%s%d" % (pre, _perm_mask(int(name[2:]), pi))
    if name.startswith("eg"):
        return "eg%d" % pi[int(name[2:])]
    return name          # ub, vv


def _pack(groups, limit):
    """First-fit-decreasing packing of term groups (kept whole when they fit) into bodies of <= limit terms."""
    bodies = []
    for g in sorted(groups, key=lambda g: -len(g)):
        while len(g) > limit:
            bodies.append(g[:limit])
            g = g[limit:]
        for b in bodies:
            if len(b) + len(g) <= limit:
                b.extend(g)
                break
        else:
            bodies.append(list(g))
    return [b for b in bodies if b]


def families(n, max_phase, min_class=6, merge_complement=False):
    """[dict(kind, size, members=[pi, ...], bodies=[[term, ...], ...])]: the canonical class of every family, cut into
    bodies, and the relabellings pi (tuples: canonical gluon i -> actual gluon pi[i]) of its members.  Classes with
    fewer than `min_class` terms are not worth a visit per member: small classes over the same gluon subsets (same
    relabellings) are merged into one family if that makes them big enough, the rest is emitted as it is, together, in a
    last family with the identity as its only member.  merge_complement: classes over k-subsets and over (n - k)-subsets
    (k != n - k) become one family too — keyed by the complement, the smaller classes have the same relabellings — so
    that their terms share bodies (fewer visits per event group)."""
    classes = {}
    for term in topo.diagram_terms(n):
        kind, S = family_key(term, n)
        classes.setdefault((kind, len(S)), {}).setdefault(S, []).append(term)
    out, misc, small = [], [], {}
    normal = []
    for (kind, size), cls in sorted(classes.items()):
        sizes = {len(v) for v in cls.values()}
        if not (len(sizes) == 1 and len(cls) == comb(n, size)):
            misc += [t for S in sorted(cls) for t in cls[S]]      # key not equivariant (ties)
        elif min(sizes) < min_class:
            small.setdefault(size, []).append((kind, cls))        # class too small for a visit of its own
        else:
            normal.append((kind, size, cls))
    # small classes over the same gluon subsets share their relabellings: together they may be worth a visit per member
    for size, lst in sorted(small.items()):
        merged = {}
        for _, cls in lst:
            for S, ts in cls.items():
                merged.setdefault(S, []).extend(ts)
        if len(lst) > 1 and len(merged[min(merged)]) >= min_class:
            normal.append(("+".join(k for k, _ in lst), size, merged))
        else:
            misc += [t for _, cls in lst for S in sorted(cls) for t in cls[S]]
    if merge_complement:
        byk = {}
        for kind, size, cls in normal:
            big = max(size, n - size)
            if size != big:                   # re-key by the complement: same subsets as the (n - size)-classes
                cls = {tuple(i for i in range(n) if i not in S): ts for S, ts in cls.items()}
            grp = byk.setdefault(big, dict(kinds=[], cls={}))
            grp["kinds"].append(kind + ("c" if size != big else ""))
            for S, ts in cls.items():
                grp["cls"].setdefault(S, []).extend(ts)
        normal = [("+".join(g["kinds"]), big, g["cls"]) for big, g in sorted(byk.items())]
    for kind, size, cls in normal:
        S0 = min(cls)
        rest0 = [i for i in range(n) if i not in S0]
        members = []
        for S in sorted(cls):
            rest = [i for i in range(n) if i not in S]
            pi = [0] * n
            for a, b in zip(S0, S):
                pi[a] = b
            for a, b in zip(rest0, rest):
                pi[a] = b
            members.append(tuple(pi))
        # bodies: terms that share their fine key (the big sub-tree they hang on) stay together
        fine = {}
        for t in cls[S0]:
            fine.setdefault(repr(group_key(t, n)[1]), []).append(t)
        out.append(dict(kind=kind, size=size, members=members, bodies=_pack([fine[k] for k in sorted(fine)], max_phase)))
    if misc:
        fine = {}
        for t in misc:
            fine.setdefault(repr(group_key(t, n)), []).append(t)
        out.append(dict(kind="X", size=0, members=[tuple(range(n))], bodies=_pack([fine[k] for k in sorted(fine)], max_phase)))
    return out


class _Body:
    """One body: its plan, its private table registry and its local operand layout."""

    def __init__(self, n, terms, acc_max, gtab, qtab):
        self.tables = Tables(n, gtab, qtab)
        self.plan = Plan(n, terms=terms, acc_max=acc_max, tables=self.tables)
        self.ntab = self.tables.layout()
        p = self.plan
        names = {"sg%d" % m for m in p.gmasks} | {"tl%d" % m for m in p.lmasks} | {"tr%d" % m for m in p.rmasks}
        for op in p.ops:
            if op[0] == "v3":
                names.update(("pm%d" % op[4], "pm%d" % op[5]))
        self.inv, self.sizes, pos = {}, {}, 0
        for nm in sorted(names, key=_inv_sort):
            sz = INV_SIZE[nm[:2]]
            self.inv[nm], self.sizes[nm] = pos, sz
            pos += sz
        self.ninv = pos
        self.flows = sorted(p.flows_touched())
        self.slot = {f: k for k, f in enumerate(self.flows)}

    def S(self, name):
        return "ld1<T>(sinv + %du * SZ)" % self.inv[name]

    def V(self, name):
        return "ldp4<T>(sinv + %du * SZ)" % self.inv[name]

    def C(self, name, m):
        return "ld1<T>(sinv + %du * SZ)" % (self.inv[name] + m)


def _emit_ops(body, w, sink, sync_every):
    """Currents, amplitudes, accumulators of one body; returns the variant-address variables used."""
    tabs = body.tables.by_name
    tmp = [0]
    vaddr = {}

    def operand(name):
        it = tabs.get(name)
        if it is None:
            return name
        va = vaddr.setdefault(it["bits"], "va" + "_".join(map(str, it["bits"])) if it["bits"] else "tab")
        tmp[0] += 1
        nm = "t%d" % tmp[0]
        w("    W4<T> %s; ldw(%s + %du * SZ, %d, %s);\n" % (nm, va, it["off"], it["nv"], nm))
        return nm

    namp, nops, declared = 0, 0, set()
    for op in body.plan.ops:
        kind = op[0]
        if sync_every and kind not in ("flush", "amp"):
            nops += 1
            if nops % sync_every == 0:
                w("    __syncthreads();   // keeps the CTA's warps on the same instruction-cache lines\n")
        if kind == "v3":
            _, o, a, b_, ma, mb = op
            a, b_ = operand(a), operand(b_)
            w("    W4<T> %s; cur_v3(%s, %s, %s, %s, %s, %s);\n" % (o, body.V("pm%d" % ma), a, body.V("pm%d" % mb), b_, body.S("sg%d" % (ma | mb)), o))
        elif kind == "k":
            _, o, a, m_, c, mask = op
            a, m_, c = operand(a), operand(m_), operand(c)
            w("    W4<T> %s; cur_k(%s, %s, %s, %s, %s);\n" % (o, a, m_, c, body.S("sg%d" % mask), o))
        elif kind in ("lq", "rq"):
            _, o, prev, g, mask = op
            prev, g = operand(prev), operand(g)
            nm = ("tl%d" if kind == "lq" else "tr%d") % mask
            c5 = ", ".join(body.C(nm, q) for q in range(5))
            w("    W4<T> %s; cur_%sp(%s, %s, %s, %s);\n" % (o, kind, prev, g, c5, o))
        elif kind == "bil":
            _, o, l, r = op
            l, r = operand(l), operand(r)
            w("    W4<T> %s; bilinear(%s, %s, %s);\n" % (o, l, r, o))
        elif kind == "amp":
            _, b_, g, accs = op
            g = operand(g)
            # the relabelling's sign of this amplitude (+-1, staged per visit) rides on the accumulation: FMA instead of ADD
            w("    const C1<T> a%d = contract(%s, %s); const T s%d = ld1<T>(sgn + %du * SZ);" % (namp, b_, g, namp, namp))
            for blk, a, s in accs:
                nm = "%d_%d" % (blk, a)
                if nm not in declared:
                    declared.add(nm)
                    w(" T ar%s = %ss%d * a%d.r, ai%s = %ss%d * a%d.i;" % (nm, "" if s > 0 else "-", namp, namp, nm, "" if s > 0 else "-", namp, namp))
                else:
                    sg = "+=" if s > 0 else "-="
                    w(" ar%s %s s%d * a%d.r; ai%s %s s%d * a%d.i;" % (nm, sg, namp, namp, nm, sg, namp, namp))
            w("\n")
            namp += 1
        elif kind == "flush":
            _, blk, a, flows = op
            for f, s in flows:
                sink(f, s, "ar%d_%d" % (blk, a), "ai%d_%d" % (blk, a))
    return vaddr


def _table_maps(local, full, pi):
    """For relabelling pi: per element of a body's local table layout the index of the relabelled entry in the
    event-wide tables, and per local item the sign of the relabelled current (child swaps of ggg vertices)."""
    m1 = [0] * local.size
    signs = {}
    for key, it in local.items.items():
        (sign, skey), = full.relabel(key, pi)
        signs[it["name"]] = sign
        # actual particle behind each variant bit of the local item
        act = []
        for q in it["bits"]:
            act.append(3 if q == 3 else gluon_particle(pi[q if q < 2 else q - 2]))
        src = full.items[skey]
        assert sorted(src["bits"]) == sorted(act), (key, skey)
        pos = [src["bits"].index(a) for a in act]
        nv = it["nv"]
        for c in range(8):
            for v in range(nv):
                vs = 0
                for j, pj in enumerate(pos):
                    vs |= ((v >> j) & 1) << pj
                m1[it["off"] + c * nv + v] = src["off"] + c * nv + vs
    return m1, signs


def _amp_signs(plan, item_sign):
    """Sign of every amplitude of `plan` when its tabled operands carry the signs `item_sign` (every in-body current is a
    single vertex, i.e. multilinear in its inputs, so signs simply multiply)."""
    sg = dict(item_sign)
    out = []
    for op in plan.ops:
        k = op[0]
        if k == "v3":
            sg[op[1]] = sg.get(op[2], 1) * sg.get(op[3], 1)
        elif k == "k":
            sg[op[1]] = sg.get(op[2], 1) * sg.get(op[3], 1) * sg.get(op[4], 1)
        elif k in ("lq", "rq", "bil"):
            sg[op[1]] = sg.get(op[2], 1) * sg.get(op[3], 1)
        elif k == "amp":
            out.append(sg.get(op[1], 1) * sg.get(op[2], 1))
    return out


HEADER = """// GENERATED by paper_2312_02898_b200/gen (process generator, K0) — do not edit.%(nvcc)s
// process: %(proc)s   gluons: %(n)d   Feynman diagrams: %(ndiag)d (whole process)
// this unit: %(what)s
// diagram terms here: %(nterms)d   colour flows: %(ncol)d   helicities: %(nhel)d   static flops / helicity here: %(flops)d
#include "mg_coop.cuh"
namespace %(ns)s {
using namespace mgw;
using namespace mgq;
constexpr int NPAR = %(npar)d, NGLU = %(n)d, NCOL = %(ncol)d, NHEL = %(nhel)d, NLANE = %(nlane)d, BLK = %(blk)d, SLOTS = BLK / NLANE;
"""

BODY_ARGS = "unsigned sinv, unsigned tab, unsigned sgn, unsigned sj, %s* jamp, int h, int live, unsigned fm"


def emit_coop(n, fp32=True, acc_max=24, **over):
    from . import emit as E
    global BLK
    cfg = dict(TUNED.get(n, TUNED[5]))
    cfg.update({k: v for k, v in over.items() if v is not None})
    BLK = cfg.get("block", 256)
    sync_every = cfg.get("sync_every", 2)
    npar, nhel = n + 2, 1 << (n + 2)
    nlane = 1 << (npar - 1)
    assert BLK % (2 * nlane) == 0, "slot layout: an even number of slots of 2^(npar-1) lanes per CTA"
    slots = BLK // nlane
    ns = "mg_ggtt" + "g" * (n - 2)
    proc = "g g > t t~" + " g" * (n - 2)
    cf = colour_matrix(n)
    cfden = common_denominator(cf)
    ncol = len(cf)
    cfi = [[int(v * cfden) for v in row] for row in cf]
    flow_index = topo.flow_index_table(n)
    flow_order = {i: p for p, i in flow_index.items()}
    fams = families(n, cfg["max_phase"], cfg.get("min_class", 6), cfg.get("merge_complement", False))
    # bodies are compiled for the register budget of the kernel's occupancy target (build.py reads the "nvcc:" line)
    maxreg = min(255, 65536 // (BLK * cfg.get("ctas_per_sm", 256 // BLK)) // 8 * 8)
    hdr = dict(proc=proc, n=n, ncol=ncol, nhel=nhel, ns=ns, npar=npar, nlane=nlane, blk=BLK,
               nvcc="\n// nvcc: -maxrregcount=%d" % maxreg if maxreg < 255 else "")
    bodies = []                  # (family index, _Body)
    for fi, fam in enumerate(fams):
        for terms in fam["bodies"]:
            bodies.append((fi, _Body(n, terms, acc_max, cfg["gtab"], cfg["qtab"])))
    ndiag = bodies[0][1].plan.ndiagrams
    nbody = len(bodies)
    hdr["ndiag"] = ndiag
    # event-wide helicity tables: every current the thresholds allow
    ftab = Tables(n, cfg["gtab"], cfg["qtab"]).register_all()
    ntabf = ftab.layout()
    # the event's full set of helicity-independent items: everything the tables and any member of any body read
    full = set(ftab.inv_names())
    for fi, b in bodies:
        for pi in fams[fi]["members"]:
            full.update(_perm_name(nm, pi) for nm in b.inv)
    inv, pos = {}, 0
    for nm in sorted(full, key=_inv_sort):
        inv[nm] = pos
        pos += INV_SIZE[nm[:2]]
    ninv = pos
    ninvp = ninv + (ninv & 1)
    ninvs = max(1, max(b.ninv for _, b in bodies))
    assert ninvs <= BLK, "visit_gather copies one helicity-independent operand per thread"
    ninvs += ninvs & 1
    ntabs = (max(b.ntab for _, b in bodies) + 3) // 4 * 4        # 16-byte aligned slot stride in both precisions
    namps = max(b.plan.namps for _, b in bodies)
    assert namps <= BLK
    namps += namps & 1
    nflows = max(len(b.flows) for _, b in bodies)
    nflows += nflows & 1
    assert nflows <= BLK
    quad = bool(cfg.get("gather16"))      # 16-byte copies of groups of four table operands instead of one copy per operand
    nmap = ntabs // 4 if quad else ntabs
    fixed = slots * (ninvp + ninvs) * 8 + 2 * namps * 8 + 2 * slots * ntabs * 8 + 3 * nmap * 4 + 2 * nflows * 4
    nst_max = max(0, (cfg["smem_kb"] * 1024 - fixed) // (2 * BLK * 8))
    files, binfo = [], []
    exec_hel, exec_slot = 0, 0
    nst_used = 0
    invmap, flowmap, tabmap, ampsign, visits, bmeta = [], [], [], [], [], []      # flat tables + per body offsets into them
    for bi, (fi, b) in enumerate(bodies):
        fam = fams[fi]
        nm_ = len(fam["members"])
        # executed: the relabelling sign costs one complex scaling (2 multiplications) per amplitude
        flops = b.plan.flops_per_helicity(colour=False, externals=False) + 2 * b.plan.namps
        exec_hel += flops * nm_
        touches = {}
        for op in b.plan.ops:
            if op[0] == "flush":
                for f, _ in op[3]:
                    touches[f] = touches.get(f, 0) + 1
        order_f = sorted(touches, key=lambda f: (-touches[f], f))
        staged = {f: i for i, f in enumerate([f for f in order_f if touches[f] > 1][:nst_max])}
        nst_used = max(nst_used, len(staged))
        lines = []
        w = lines.append
        seen = set()

        def sink(f, s, re, im, staged=staged, seen=seen, w=w, b=b):
            neg = "" if s > 0 else "-"
            if f in staged:
                a = "sj + %du * COL" % (2 * staged[f])
                b_ = "sj + %du * COL" % (2 * staged[f] + 1)
                if f in seen:
                    sg = "+" if s > 0 else "-"
                    w("    ssh(%s, ld1<T>(%s) %s %s); ssh(%s, ld1<T>(%s) %s %s);\n" % (a, a, sg, _mul(s, re), b_, b_, sg, _mul(s, im)))
                else:
                    seen.add(f)
                    w("    ssh(%s, %s%s); ssh(%s, %s%s);\n" % (a, neg, _mul(s, re), b_, neg, _mul(s, im)))
            else:
                w("    if (live) { T* jp = jamp + ldsi(fm + %du); red_add(jp, %s%s); red_add(jp + BLK, %s%s); }\n"
                  % (4 * b.slot[f], neg, _mul(s, re), neg, _mul(s, im)))

        vaddr = _emit_ops(b, w, sink, sync_every)
        out = [HEADER % dict(hdr, nterms=len(b.plan.terms), flops=flops,
                             what="body %d of %d (family %s%d, executed for %d relabellings per visit)"
                                  % (bi, nbody, fam["kind"], fam["size"], nm_))]
        o = out.append
        o("template <class T>\nMG_DEV void body%d_impl(const unsigned sinv, const unsigned tab, const unsigned sgn, const unsigned sj,\n"
          "                      T* __restrict__ jamp, const int h, const int live, const unsigned fm) {\n" % bi)
        o("  constexpr unsigned SZ = (unsigned)sizeof(T), COL = (unsigned)BLK * SZ;\n")
        for bits, nm in sorted(vaddr.items()):
            if bits:
                expr = " | ".join("(((h >> %d) & 1) << %d)" % (npar - 1 - q, j) for j, q in enumerate(bits))
                o("  const unsigned %s = tab + (unsigned)(%s) * SZ;\n" % (nm, expr))
        o("  {\n")
        out += lines
        o("  }\n")
        if staged:
            o("  if (live) {\n")
            for f, sl in sorted(staged.items()):
                o("    { T* jp = jamp + ldsi(fm + %du); red_add(jp, ld1<T>(sj + %du * COL)); red_add(jp + BLK, ld1<T>(sj + %du * COL)); }\n"
                  % (4 * b.slot[f], 2 * sl, 2 * sl + 1))
            o("  }\n")
        o("}\n")
        o("__device__ __noinline__ void body%d(%s) {\n  body%d_impl<double>(sinv, tab, sgn, sj, jamp, h, live, fm);\n}\n"
          % (bi, BODY_ARGS % "double", bi))
        if fp32:
            o("__device__ __noinline__ void body%d(%s) {\n  body%d_impl<float>(sinv, tab, sgn, sj, jamp, h, live, fm);\n}\n"
              % (bi, BODY_ARGS % "float", bi))
        o("}  // namespace\n")
        files.append(("%s_b%02d.cu" % (ns, bi), "".join(out)))
        # per member: gather map of the helicity-independent operands, colour-flow map
        bmeta.append((len(flowmap), len(visits)))
        for pi in fam["members"]:
            assert b.ntab % 4 == 0
            visits.append((len(tabmap), b.ntab // 4 if quad else b.ntab, len(invmap), b.ninv, len(ampsign), b.plan.namps, len(flowmap), len(b.flows)))
            for nm, off in sorted(b.inv.items(), key=lambda kv: kv[1]):
                src = inv[_perm_name(nm, pi)]
                invmap += [src + j for j in range(b.sizes[nm])]
            for f in b.flows:
                o_ = tuple(pi[g] for g in flow_order[f])
                flowmap.append(2 * flow_index[o_] * BLK)
            m1, isign = _table_maps(b.tables, ftab, pi)
            # the relabelling maps whole tabled currents (8 x nv contiguous elements): one map entry per group of four
            assert all(m1[k] % 4 == 0 and m1[k + 1:k + 4] == [m1[k] + 1, m1[k] + 2, m1[k] + 3] for k in range(0, len(m1), 4))
            tabmap += m1[0::4] if quad else m1
            ampsign += _amp_signs(b.plan, isign)
        binfo.append(dict(family="%s%d" % (fam["kind"], fam["size"]), members=nm_, terms=len(b.plan.terms), flops=flops,
                          flows=len(touches), staged=len(staged), max_live=b.plan.max_live(), ninv=b.ninv, ntab=b.ntab))
    colour_flops = 2 * (ncol * (ncol - 1) // 2) * 2 + ncol * 8
    gt = Tables(n, cfg["gtab"], cfg["qtab"])
    algo = Plan(n, acc_max=acc_max, tables=gt).flops_per_helicity(colour=False, externals=False)
    algo_slot = gt.flops()           # the tabled currents the diagrams actually use, once per slot
    exec_slot = ftab.flops()         # the kernel builds every current the thresholds allow
    smem = fixed + 2 * nst_used * BLK * 8
    files.append(_main_unit(E, n, ns, hdr, cfi, cfden, fams, bodies, bmeta, invmap, flowmap, (tabmap, ampsign, visits, namps, nflows), ftab,
                            ntabf, inv, ninv, ninvp, ninvs, ntabs, nst_used, fp32, exec_hel + colour_flops, algo + colour_flops,
                            exec_slot, algo_slot, cfg))
    info = dict(proc=proc, ns=ns, npar=npar, ncol=ncol, nhel=nhel, ndiagrams=ndiag,
                nterms=sum(len(b.plan.terms) * len(fams[fi]["members"]) for fi, b in bodies),
                flops_per_helicity=exec_hel + colour_flops, flops_algorithmic=algo + colour_flops, flops_per_slot=exec_slot,
                flops_algorithmic_per_slot=algo_slot, shape="coop", ngroups=nbody, ninv=ninv, ninv_body=ninvs, ntab_body=ntabs, ntab_full=ntabf,
                nst=nst_used, smem_bytes=smem, slots=slots, gtab=cfg["gtab"], qtab=cfg["qtab"],
                visits=sum(len(fams[fi]["members"]) for fi, _ in bodies), groups=binfo)
    return files, info


def _main_unit(E, n, ns, hdr, cfi, cfden, fams, bodies, bmeta, invmap, flowmap, tabmaps, ftab, ntabf, inv, ninv, ninvp, ninvs,
               ntabs, nst, fp32, flops_hel, algo_hel, flops_slot, algo_slot, cfg):
    npar, nhel, ncol = n + 2, 1 << (n + 2), len(cfi)
    nbody = len(bodies)
    denom = 4 * 64 * factorial(n - 2)
    rows = E._colour_rows(cfi, ncol)
    dmma = ncol > 32 or cfg.get("colour") == "dmma"      # FP64 tensor cores for the colour sum (fp64 kernels only)
    reg = not dmma or fp32
    out = [HEADER % dict(hdr, nterms=0, flops=flops_hel,
                         what="operand maps, table descriptors, invariants kernel, persistent sigma kernel (%d bodies x their "
                              "relabellings, colour sum K6, helicity sum K7), launcher" % nbody)]
    w = out.append
    quad = bool(cfg.get("gather16"))
    w("constexpr int NMAP = %d;      // index-map entries per visit: one per table operand, or per group of four (16-byte copies)\n"
      % (ntabs // 4 if quad else ntabs))
    w("constexpr bool QUAD = %s;\n" % ("true" if quad else "false"))
    w("constexpr int NINV = %d, NINVP = %d, NINVS = %d, NTABS = %d, NTABF = %d, NST = %d, NBODY = %d, TPOS = %d;\n"
      % (ninv, ninvp, ninvs, ntabs, ntabf, nst, nbody, npar - 3))

    def table(name, ctype, vals, per=24):
        w("__device__ const %s %s[%d] = {\n" % (ctype, name, max(1, len(vals))))
        for k_ in range(0, len(vals), per):
            w("  " + ", ".join(map(str, vals[k_:k_ + per])) + ",\n")
        if not vals:
            w("  0\n")
        w("};\n")

    table("inv_map", "short", invmap)
    table("flow_map", "int", flowmap, 16)
    tabmap, ampsign, visits, namps, nflows = tabmaps
    table("tab_map", "int", tabmap, 24)
    w("__device__ const double amp_sign64[%d] = {\n" % max(1, len(ampsign)))
    for k_ in range(0, len(ampsign), 40):
        w("  " + ", ".join("%d." % v for v in ampsign[k_:k_ + 40]) + ",\n")
    w("};\n")
    if fp32:
        w("__device__ const float amp_sign32[%d] = {\n" % max(1, len(ampsign)))
        for k_ in range(0, len(ampsign), 40):
            w("  " + ", ".join("%d.f" % v for v in ampsign[k_:k_ + 40]) + ",\n")
        w("};\n")
        w("MG_DEV const float* amp_sign_of(float*) { return amp_sign32; }\n")
    w("MG_DEV const double* amp_sign_of(double*) { return amp_sign64; }\n")
    w("constexpr int NVISIT = %d, NAMPS = %d, NFLOWS = %d;\n" % (len(visits), namps, nflows))
    w("__constant__ VisitDesc visit_desc[NVISIT + 2] = {\n")
    for v_ in visits:
        w("  {%d, %d, %d, %d, %d, %d, %d, %d},\n" % v_)
    w("  {0, 0, 0, 0, 0, 0, 0, 0}, {0, 0, 0, 0, 0, 0, 0, 0}};\n")
    # helicity-bit shifts per family member: canonical gluon i takes the helicity of gluon pi[i]
    hsh, foff_of = [], {}
    for fi, fam in enumerate(fams):
        foff_of[fi] = len(hsh)
        for pi in fam["members"]:
            hsh += [npar - 1 - gluon_particle(pi[i]) for i in range(n)]
    table("hel_shift", "signed char", hsh, 40)
    # ---- descriptors of the event-wide tables ----
    gl, dl = [], []
    for kind, nb, its, sync in ftab.groups():
        gl.append("{%d, %d, %d, %d, %d, 0, 0, 0}" % (KIND[kind], nb, len(its), len(dl), 1 if sync else 0))
        for it in its:
            ins = [ftab.items[k] for k in it["inputs"]]
            in_off = [c["off"] for c in ins] + [0] * (3 - len(ins))
            in_nb = [len(c["bits"]) for c in ins] + [0] * (3 - len(ins))
            in_sel = [ftab.selector(it, c) for c in ins] + [0] * (3 - len(ins))
            iv = [inv[nm] for nm in it["inv"]]
            if kind == "q":
                iv = [iv[0], 0 if it["name"] == "ub" else 1]
            iv += [0] * (3 - len(iv))
            dl.append("{%d, {%s}, {%s}, {%s}, {%s}, {0, 0, 0}}" % (it["off"], ", ".join(map(str, in_off)), ", ".join(map(str, in_nb)),
                                                                   ", ".join(map(str, in_sel)), ", ".join(map(str, iv))))
    w("constexpr int NGROUPS = %d;\n" % len(gl))
    w("__device__ const TabGroup tab_groups[%d] = {\n  " % len(gl) + ",\n  ".join(gl) + "};\n")
    w("__device__ const TabDesc tab_desc[%d] = {\n  " % len(dl) + ",\n  ".join(dl) + "};\n")
    # ---- colour data ----
    if dmma:
        w("// dense colour table for the DMMA contraction: CF on the diagonal 8x8 blocks, 2 CF above, 0 below; the common\n"
          "// denominator %d is folded into the normalisation\n" % cfden)
        w("__device__ __align__(16) const double cf_dense[%d] = {\n" % (ncol * ncol))
        for i in range(ncol):
            w("  " + ", ".join("%d." % (cfi[i][j] if j // 8 == i // 8 else 2 * cfi[i][j] if j // 8 > i // 8 else 0)
                               for j in range(ncol)) + ",\n")
        w("};\n")
    w("// symmetric colour form: me = sum_i J_i^* (CF_ii J_i + 2 sum_{j>i} CF_ij J_j) / %d, integer coefficients as immediates\n" % cfden)
    w("template <class T> MG_DEV T colour_reg(const T* __restrict__ jb) {\n")
    if reg:
        for f in range(ncol):
            w("  const T jr%d = __ldcg(jb + %d * BLK), ji%d = __ldcg(jb + %d * BLK);\n" % (f, 2 * f, f, 2 * f + 1))
        w("  T me = T(0);\n")
        for i in range(ncol):
            zr = " + ".join("T(%d) * jr%d" % (rows[i][j], j) for j in range(i, ncol) if rows[i][j])
            zi = " + ".join("T(%d) * ji%d" % (rows[i][j], j) for j in range(i, ncol) if rows[i][j])
            w("  me += jr%d * (%s);\n  me += ji%d * (%s);\n" % (i, zr, i, zi))
        w("  return me;\n}\n")
    else:
        w("  return T(0);\n}\n")
    for bi in range(nbody):
        w("__device__ void body%d(%s);\n" % (bi, BODY_ARGS % "double"))
        if fp32:
            w("__device__ void body%d(%s);\n" % (bi, BODY_ARGS % "float"))
    # ---- invariants kernel ----
    gm = {int(k[2:]) for k in inv if k.startswith("sg")}
    lm = {int(k[2:]) for k in inv if k.startswith("tl")}
    rm = {int(k[2:]) for k in inv if k.startswith("tr")}
    v3m = {int(k[2:]) for k in inv if k.startswith("pm")}
    w("template <class T>\n__global__ void __launch_bounds__(128) invariants_kernel(const double* __restrict__ mom, long long nevt,\n"
      "                  T* __restrict__ invbuf, double mt_d) {\n")
    w("  const long long ievt = (long long)blockIdx.x * blockDim.x + threadIdx.x;\n  if (ievt >= nevt) return;\n")
    E._prologue(_Masks(n, gm, lm, rm, v3m), w)
    w("  T* __restrict__ o = invbuf + ievt * NINVP;\n")
    for name, i in sorted(inv.items(), key=lambda kv: kv[1]):
        if name[0] == "s":
            w("  o[%d] = %s;\n" % (i, name))
        elif name.startswith("eg"):
            g = int(name[2:])
            w("  { W4<double> e; ext_gluon(kd[%d], +1, %s, e);   // lambda = +1: e.r = -R, e.i = I\n" % (g, "false" if g < 2 else "true"))
            w("    o[%d] = T(-e.r[1]); o[%d] = T(-e.r[2]); o[%d] = T(-e.r[3]); o[%d] = T(e.i[1]); o[%d] = T(e.i[2]); }\n"
              % (i, i + 1, i + 2, i + 3, i + 4))
        elif name.startswith("tl") or name.startswith("tr"):
            side, m_ = name[1], int(name[2:])
            sv, qv = "ds%s%d" % (side, m_), "dq%s%d" % (side, m_)
            w("  o[%d] = T(%s * (%s.c[0] + %s.c[3])); o[%d] = T(%s * (%s.c[0] - %s.c[3])); o[%d] = T(%s * %s.c[1]); "
              "o[%d] = T(%s * %s.c[2]); o[%d] = T(%s * mt_d);\n"
              % (i, sv, qv, qv, i + 1, sv, qv, qv, i + 2, sv, qv, i + 3, sv, qv, i + 4, sv))
        elif name in ("ub", "vv"):
            fn, mom = ("ext_ubar", "ptd") if name == "ub" else ("ext_v", "ptbd")
            for hi, lam in ((0, "+1"), (8, "-1")):
                w("  { W4<double> q; %s(%s, mt_d, %s, q);\n" % (fn, mom, lam))
                w("    " + " ".join("o[%d] = T(q.r[%d]); o[%d] = T(q.i[%d]);" % (i + hi + 2 * m, m, i + hi + 2 * m + 1, m)
                                    for m in range(4)) + " }\n")
        else:
            w("  stp(o + %d, 1, %s);\n" % (i, name))
    w("}\n")
    # ---- the persistent sigma kernel ----
    calls = []
    for bi, (fi, b) in enumerate(bodies):
        nm_ = len(fams[fi]["members"])
        fo, v0 = bmeta[bi]
        calls.append(
            "    // body %d: family %s%d, %d terms, %d relabellings\n"
            "#pragma unroll 1\n    for (int m = 0; m < %d; ++m) {\n"
            "      const int v = %d + m;\n"
            "      visit_step<T, SLOTS, QUAD>(visit_desc, v, tab_map, inv_map, gtab, asgn, flow_map, sinv0, sinvp0, smap0, stab0, ssgn0, sfm0, NINVP, NINVS,\n"
            "                                 NTABS, NMAP, NTABF, NAMPS, NFLOWS);\n"
            "      const int hp = permute_helicity<NPAR, NGLU>(h, hel_shift + %d + m * NGLU);\n"
            "      body%d(sinvp, stab0 + (unsigned)(((v & 1) * SLOTS + slot) * NTABS) * SZ, ssgn0 + (unsigned)((v & 1) * NAMPS) * SZ, sj, jamp, hp, live,\n"
            "             sfm0 + (unsigned)((v & 1) * NFLOWS) * 4u);\n    }\n"
            % (bi, fams[fi]["kind"], fams[fi]["size"], len(b.plan.terms), nm_, nm_, v0, foff_of[fi], bi))
    w(KERNEL % dict(calls="".join(calls), minb=cfg.get("ctas_per_sm", 256 // BLK),
                    colour=("T meh;\n    if constexpr (sizeof(T) == 8) {\n"
                            "      colour_dmma_cta<NCOL, BLK>(cf_dense, (const double*)jamp_cta, reinterpret_cast<double*>(smem_raw + SINV_BYTES), (double*)s_meh);\n"
                            "      meh = s_meh[tid];\n    } else meh = colour_reg<T>(jamp);" if dmma else
                            "T meh = colour_reg<T>(jamp);"),
                    coloursm=((2 * ncol * 34 + (BLK // 32) * 32) * 8 + ((BLK // hdr["nlane"]) * ninvp * 8 + 15) // 16 * 16) if dmma else 0))
    w(LAUNCH % dict(cfden=cfden, denom=denom, minb=cfg.get("ctas_per_sm", 256 // BLK), l2win=1 if cfg.get("l2_window") else 0,
                    run32=("  return run<float>(mom, (float*)me_out, nevt, (const float*)lane_w, ntb, tb_first, (float*)perhel_out, par, ws, ws_bytes, st);"
                           if fp32 else "  return -1;")))
    w("}  // namespace\n")
    w("extern const mg_procdesc_t mg_desc_%s = {\"%s\", %d, %d, %d, %d, %d, %d,\n"
      "  %dLL, {0, 0, 1, 1%s}, nullptr, %s::launch, {0, 0}, 2, %d, {%d, %d}, %dLL, %dLL, %dLL, {%d, %d}, %d, %d};\n"
      % (ns[3:], hdr["proc"], npar, n, hdr["ndiag"], nhel, ncol, denom, flops_hel, ", 0" * (n - 2), ns, 1 if fp32 else 0,
         ninvp * 8, ninvp * 4, algo_hel, flops_slot, algo_slot, (2 * ncol * BLK + (BLK // hdr["nlane"]) * ntabf) * 8,
         (2 * ncol * BLK + (BLK // hdr["nlane"]) * ntabf) * 4, hdr["nlane"], cfg.get("ctas_per_sm", 256 // BLK)))
    return (ns + ".cu", "".join(out))


class _Masks:
    """What emit._prologue needs: the propagator / vertex masks of the event's full operand set."""

    def __init__(self, n, gm, lm, rm, v3m):
        self.n, self.gmasks, self.lmasks, self.rmasks = n, gm, lm, rm
        self.ops = [("v3", None, None, None, m, m) for m in v3m]


KERNEL = """
// One CTA = SLOTS slots = SLOTS (event, top helicity) pairs; thread = (slot, lane): lane = the helicity bits of the other
// particles.  ntb = number of top helicities run (2: both, slots 2k / 2k+1 are lambda_t = -1 / +1 of event k;
// 1: only tb_first — the helicity-flip symmetry |M(-h)|^2 = |M(h)|^2 is in the lane weights, mg_api.cu).
template <class T>
__global__ void __launch_bounds__(BLK, %(minb)d)
sigma_kernel(long long nevt, int ntb, int tb_first, const T* __restrict__ lane_w, const T* __restrict__ invbuf,
             T* __restrict__ scratch, T* __restrict__ gtab_all, T* __restrict__ me_out, T* __restrict__ perhel_out,
             long long perhel_stride, T norm) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int s_tbit[SLOTS];
  __shared__ T s_meh[BLK];
  constexpr unsigned SZ = (unsigned)sizeof(T);
  const unsigned sbase = (unsigned)__cvta_generic_to_shared(smem_raw);
  const int tid = threadIdx.x, slot = tid / NLANE, lane = tid %% NLANE;
  // shared memory: full per-event operand set | the running visit's helicity-independent operands | amplitude signs [2] |
  // table operands [2] | index maps [3] | staged JAMPs
  const unsigned sinv0 = sbase, sinvp0 = sinv0 + SLOTS * NINVP * SZ, ssgn0 = sinvp0 + SLOTS * NINVS * SZ;
  const unsigned stab0 = ssgn0 + 2 * NAMPS * SZ, smap0 = stab0 + 2 * SLOTS * NTABS * SZ, sfm0 = smap0 + 3 * NMAP * 4;
  const unsigned sj = sfm0 + 2 * NFLOWS * 4 + ((NMAP & 1) ? 4 : 0) + tid * SZ;
  const unsigned sinvp = sinvp0 + slot * NINVS * SZ;
  const T* __restrict__ asgn = amp_sign_of((T*)nullptr);
  constexpr unsigned SINV_BYTES = (SLOTS * NINVP * SZ + 15u) / 16u * 16u;      // the colour sum's tile staging starts behind it
  // scratch = [JAMPs of every resident CTA][event-wide helicity tables of every resident CTA]: the JAMP part is what the
  // launcher's persisting L2 window covers
  T* __restrict__ jamp_cta = scratch + (size_t)blockIdx.x * (2 * NCOL * BLK);
  T* __restrict__ jamp = jamp_cta + tid;
  T* __restrict__ gtab = gtab_all + (size_t)blockIdx.x * (SLOTS * NTABF);      // event-wide helicity tables of the CTA's slots
  const long long nslot = nevt * ntb;
  prefetch_invariants<T>(invbuf, sinv0, (long long)blockIdx.x * SLOTS, nslot, nevt, ntb, NINVP, SLOTS);
  for (long long g0 = (long long)blockIdx.x * SLOTS; g0 < nslot; g0 += (long long)gridDim.x * SLOTS) {
    const long long gs = g0 + slot;
    const bool slot_live = gs < nslot;
    const long long ievt = slot_live ? (ntb == 2 ? gs >> 1 : gs) : nevt - 1;
    const int tb = ntb == 2 ? (int)(gs & 1) : tb_first;
    visit_drain();                         // this group's invariants (prefetched) have landed ..
    __syncthreads();                       // .. for every thread, and the previous iteration's shared memory is dead
    if (lane == 0) s_tbit[slot] = tb;
    {   // the bodies only ever add (L2 reductions): zero the CTA's JAMPs, two columns per store
      struct __align__(2 * sizeof(T)) T2 { T x, y; };
      T2* __restrict__ z = reinterpret_cast<T2*>(jamp_cta) + tid;        // 2 NCOL BLK values = NCOL BLK pairs
#pragma unroll 8
      for (int q = 0; q < NCOL; ++q) z[q * BLK] = T2{T(0), T(0)};
    }
    // full helicity index: bit (NPAR-1-i) <=> particle i; the top quark (particle 2) sits at bit TPOS
    const int h = ((lane >> TPOS) << (TPOS + 1)) | (tb << TPOS) | (lane & ((1 << TPOS) - 1));
    const T wgt = lane_w[tb * NLANE + lane];
    const int live = slot_live && wgt != T(0);
    __syncthreads();
    build_tables_global<T>(tab_groups, NGROUPS, tab_desc, sinv0, gtab, NINVP, NTABF, SLOTS, s_tbit);
    visit_prologue<T, SLOTS, QUAD>(visit_desc, tab_map, gtab, asgn, flow_map, smap0, stab0, ssgn0, sfm0, NTABS, NMAP, NTABF, NAMPS, NFLOWS);
%(calls)s
    visit_drain();
    // nothing reads the invariant block after the last visit: the next group's invariants travel during the colour sum
    prefetch_invariants<T>(invbuf, sinv0, g0 + (long long)gridDim.x * SLOTS, nslot, nevt, ntb, NINVP, SLOTS);
    __threadfence();                       // the JAMP reductions are performed at L2 before anyone reads them back
    __syncthreads();
    %(colour)s
    if (perhel_out && slot_live) perhel_out[(long long)h * perhel_stride + ievt] = meh * norm;
    __syncthreads();
    s_meh[tid] = live ? wgt * meh : T(0);
    __syncthreads();
    for (int off = NLANE / 2; off > 0; off >>= 1) {       // fixed-order tree: deterministic helicity sum
      if (lane < off) s_meh[tid] += s_meh[tid + off];
      __syncthreads();
    }
    if (lane == 0 && slot_live) {
      if (ntb == 2) { if ((slot & 1) == 0) me_out[ievt] = (s_meh[tid] + s_meh[tid + NLANE]) * norm; }
      else me_out[ievt] = s_meh[tid] * norm;
    }
  }
}
constexpr size_t COLOUR_SMEM = %(coloursm)d;
"""

LAUNCH = """
template <class T>
static int run(const double* mom, T* me_out, long long nevt, const T* lane_w, int ntb, int tb_first, T* perhel_out,
               const double* par, void* ws, size_t ws_bytes, cudaStream_t st) {
  double norm = 1.0;
  for (int i = 0; i < NGLU; ++i) norm *= par[0];          // par[0] = g_s^2, par[1] = mt
  norm /= (double)%(cfden)d * (double)%(denom)d;
  int dev = 0, nsm = 0, per_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
  size_t smem = (size_t)(SLOTS * (NINVP + NINVS) + 2 * NAMPS + 2 * SLOTS * NTABS + 2 * NST * BLK) * sizeof(T) + 3 * NMAP * 4 + 2 * NFLOWS * 4 + 8;
  if (sizeof(T) == 8 && smem < COLOUR_SMEM) smem = COLOUR_SMEM;
  auto kern = sigma_kernel<T>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, BLK, smem) != cudaSuccess || per_sm < 1) return -1;
  if (per_sm > %(minb)d) per_sm = %(minb)d;                             // mg_api.cu sizes the scratch for this many CTAs per SM
  const long long ncta_max = (long long)per_sm * nsm;
  const size_t per_cta = (size_t)2 * NCOL * BLK + (size_t)SLOTS * NTABF;
  const size_t scratch_bytes = (size_t)ncta_max * per_cta * sizeof(T);
  if (ws_bytes < scratch_bytes + (size_t)NINVP * sizeof(T) * 32) return -2;
  T* scratch = (T*)ws;
  T* inv = scratch + (size_t)ncta_max * per_cta;
  long long E = (long long)((ws_bytes - scratch_bytes) / ((size_t)NINVP * sizeof(T))) / 32 * 32;   // whole momentum pages
  if (E > nevt) E = (nevt + 31) / 32 * 32;
  else { const long long nt = (nevt + E - 1) / E; E = ((nevt + nt - 1) / nt + 31) / 32 * 32; }   // equal tiles
  int nlaunch = 0;
  // The CTA-private JAMPs are the kernel's read-modify-write working set (gg -> t t~ g g g: 73 MB, next to 35 MB of tables, in
  // a 126 MB L2): without help dirty JAMP lines are evicted and fetched again all the time (measured: 395 GB of DRAM writes
  // per call).  An access-policy window makes the JAMP part of the scratch persisting, up to the device's limit.
  const size_t jamp_bytes = (size_t)ncta_max * 2 * NCOL * BLK * sizeof(T);
  const bool l2win = %(l2win)d && jamp_bytes > ((size_t)32 << 20);
  if (l2win) {
    int maxp = 0, maxw = 0;
    cudaDeviceGetAttribute(&maxp, cudaDevAttrMaxPersistingL2CacheSize, dev);
    cudaDeviceGetAttribute(&maxw, cudaDevAttrMaxAccessPolicyWindowSize, dev);
    if (maxp > 0 && maxw > 0) {
      const size_t setaside = jamp_bytes < (size_t)maxp ? jamp_bytes : (size_t)maxp;
      cudaStreamAttrValue av;
      av.accessPolicyWindow.base_ptr = (void*)scratch;
      av.accessPolicyWindow.num_bytes = jamp_bytes < (size_t)maxw ? jamp_bytes : (size_t)maxw;
      const double ratio = (double)setaside / (double)av.accessPolicyWindow.num_bytes;
      av.accessPolicyWindow.hitRatio = ratio < 1.0 ? (float)ratio : 1.f;
      av.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
      av.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
      if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, setaside) != cudaSuccess ||
          cudaStreamSetAttribute(st, cudaStreamAttributeAccessPolicyWindow, &av) != cudaSuccess) (void)cudaGetLastError();
    }
  }
  for (long long e0 = 0; e0 < nevt; e0 += E) {
    const long long ne = nevt - e0 < E ? nevt - e0 : E;
    invariants_kernel<T><<<(unsigned)((ne + 127) / 128), 128, 0, st>>>(mom + e0 * NPAR * 4, ne, inv, par[1]);
    const long long nslot = ne * ntb, ngroup = (nslot + SLOTS - 1) / SLOTS;
    const unsigned grid = (unsigned)(ngroup < ncta_max ? ngroup : ncta_max);
    kern<<<grid, BLK, smem, st>>>(ne, ntb, tb_first, lane_w, inv, scratch, scratch + (size_t)ncta_max * 2 * NCOL * BLK, me_out + e0,
                                  perhel_out ? perhel_out + e0 : (T*)nullptr, nevt, T(norm));
    nlaunch += 2;
  }
  if (l2win) {                              // the caller's stream leaves without a window
    cudaStreamAttrValue av;
    av.accessPolicyWindow.base_ptr = nullptr;
    av.accessPolicyWindow.num_bytes = 0;
    av.accessPolicyWindow.hitRatio = 0.f;
    av.accessPolicyWindow.hitProp = cudaAccessPropertyNormal;
    av.accessPolicyWindow.missProp = cudaAccessPropertyNormal;
    if (cudaStreamSetAttribute(st, cudaStreamAttributeAccessPolicyWindow, &av) != cudaSuccess) (void)cudaGetLastError();
  }
  return nlaunch;
}
static int launch(int prec, const double* mom, void* me_out, long long nevt, const void* lane_w, int ntb, int tb_first,
                  void* perhel_out, const double* par, void* ws, size_t ws_bytes, cudaStream_t st) {
  if (prec == 0) return run<double>(mom, (double*)me_out, nevt, (const double*)lane_w, ntb, tb_first, (double*)perhel_out, par, ws, ws_bytes, st);
%(run32)s
}
"""
