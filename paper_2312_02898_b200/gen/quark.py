"""Quark channels of p p -> t t~ + 0..2 jets: the top line, ONE massless quark line of
another flavour and k <= 2 gluons, in every crossing.  Process generation (K0) for this family: diagram enumeration,
colour-flow expansion, colour matrix, and a fused kernel (thread = event, JAMPs in registers) emitted as straight-line
code over the same device routines as g g -> t t~ + gluons (csrc/mg_wave.cuh).

Diagrams.  The light line is connected to the rest by exactly one off-shell gluon x.  Along its fermion flow it
absorbs a sequence of gluon trees before x (blocks A, counted from the end of the flow) and after x (blocks B): a
*light configuration* (A, B) over a gluon subset Sq.  Its current J_P^mu = -Vbar(A) gamma^mu U(B) / P^2 is a
pseudo-gluon P: the rest of the diagram is a one-quark-line diagram term of topology.py over the leaves
(gluons not in Sq) + {P}.  Counts: 1, 5, 36 Feynman diagrams for k = 0, 1, 2.

Colour.  A term's colour factor is (alpha T^x beta)_{i l} (A T^x B)_{o n}  (i, l: top, antitop; o, n: end and start
of the light line's fermion flow; alpha, beta, A, B: T-strings of the gluon orderings, commutators expanded as in
topology.orderings).  Fierz:  = 1/2 (alpha B)_{i n} (A beta)_{o l} - 1/(2N) (alpha beta)_{i l} (A B)_{o n}.
Basis: L(S1|S2) = 1/2 (T^S1)_{in} (T^S2)_{ol} and S(S1|S2) = -1/(2N) (T^S1)_{il} (T^S2)_{on} over all ordered splits of
the gluons: 2 (k+1)! flows, every term adds its amplitude with unit coefficients.  The colour matrix is evaluated
exactly with colour._traces (Fierz again), the common factor 1/4 goes into the denominator.
"""
from fractions import Fraction
from itertools import permutations, product
from math import factorial, lcm

from . import topology as topo
from .colour import NC, _canon, _traces

FLOPS = {"v3": 156, "k": 141, "lq": 120, "rq": 120, "bil": 72, "amp": 30, "pair": 80, "ext_g": 30, "ext_q": 50, "jamp_add": 2}
NAMES = {"q": "q", "Q": "q~", "g": "g", "t": "t", "T": "t~"}
TAGS = {"q": "q", "Q": "qx", "g": "g", "t": "t", "T": "tx"}

# the subprocesses of p p -> t t~ + 0, 1, 2 jets with one light-quark line
SPECS = ("qQtT", "QqtT",
         "qQtTg", "QqtTg", "qgtTq", "gqtTq", "QgtTQ", "gQtTQ",
         "qQtTgg", "QqtTgg", "qgtTqg", "gqtTqg", "QgtTQg", "gQtTQg", "ggtTqQ")


class QProcess:
    """Particles and crossing of one subprocess.  spec: one character per particle in process order ('q' light quark,
    'Q' light antiquark, 'g' gluon, "tT" at positions 2, 3; the first two are the beams)."""

    def __init__(self, spec):
        assert len(spec) >= 4 and spec[2:4] == "tT", spec
        self.spec, self.npar = spec, len(spec)
        self.gpart = [i for i, c in enumerate(spec) if c == "g"]
        self.k = len(self.gpart)
        starts = [i for i, c in enumerate(spec) if c in "qQ" and ((c == "q") == (i < 2))]     # incoming q / outgoing q~
        ends = [i for i, c in enumerate(spec) if c in "qQ" and ((c == "q") != (i < 2))]       # outgoing q / incoming q~
        assert len(starts) == 1 and len(ends) == 1, spec
        self.pin, self.pout = starts[0], ends[0]
        self.in_is_u, self.out_is_ubar = self.pin < 2, self.pout >= 2
        d = 1
        for i in (0, 1):
            d *= 16 if spec[i] == "g" else 6
        self.denominator = d * factorial(sum(1 for i in self.gpart if i >= 2))
        self.proc = " ".join(NAMES[c] for c in spec[:2]) + " > " + " ".join(NAMES[c] for c in spec[2:])
        self.tag = "".join(TAGS[c] for c in spec)
        self.massive = [1 if c in "tT" else 0 for c in spec]


def light_configs(sq):
    """[(A, B)]: tuples of gluon-tree terms absorbed before / after the off-shell gluon, over the gluon labels sq."""
    out = []
    for blocks in topo.ordered_block_partitions(sq):
        for trees in product(*[topo.gluon_tree_terms(b) for b in blocks]):
            for c in range(len(trees) + 1):
                out.append((tuple(trees[:c]), tuple(trees[c:])))
    return out


def diagram_terms(k):
    """[(A, B, blocks)]: light configuration + one-line term over the remaining gluons and the pseudo-gluon (leaf k)."""
    out = []
    for mask in range(1 << k):
        sq = tuple(i for i in range(k) if mask >> i & 1)
        rest = tuple(i for i in range(k) if not mask >> i & 1) + (k,)
        for a, b in light_configs(sq):
            for blocks in topo.ordered_block_partitions(rest):
                for trees in product(*[topo.gluon_tree_terms(bl) for bl in blocks]):
                    out.append((a, b, tuple(trees)))
    return out


def n_feynman_diagrams(terms):
    tot = Fraction(0)
    for a, b, blocks in terms:
        q = sum(topo.n_four_vertices(t) for t in a + b + blocks)
        tot += Fraction(1, 1 << q)
    assert tot.denominator == 1
    return int(tot)


def flows(k):
    """Colour-flow basis: [('L' | 'S', S1, S2)] over all ordered splits of the gluons."""
    out = []
    for kind in "LS":
        for perm in permutations(range(k)):
            for cut in range(k + 1):
                out.append((kind, perm[:cut], perm[cut:]))
    return out


def _orderings_seq(trees):
    acc = [((), 1)]
    for t in trees:
        acc = [(o + ot, s * st) for o, s in acc for ot, st in topo.orderings(t)]
    return acc


def term_flows(term, k, index):
    """[(flow index, sign)] of one term."""
    a, b, blocks = term
    d = {}
    for otop, s1 in _orderings_seq(blocks):
        ip = otop.index(k)
        alpha, beta = otop[:ip], otop[ip + 1:]
        for oa, s2 in _orderings_seq(a):
            for ob, s3 in _orderings_seq(b):
                s = s1 * s2 * s3
                for key in (("L", alpha + ob, oa + beta), ("S", alpha + beta, oa + ob)):
                    d[index[key]] = d.get(index[key], 0) + s
    return tuple(sorted((f, s) for f, s in d.items() if s != 0))


def colour_matrix(k):
    """Exact CF (Fractions) in the basis of flows(k), without the common factor 1/4."""
    fl = flows(k)
    w = {"L": Fraction(1), "S": Fraction(-1, NC)}

    def rev(s):
        return tuple(reversed(s))

    cf = [[None] * len(fl) for _ in fl]
    for i, (k1, a1, a2) in enumerate(fl):
        for j, (k2, b1, b2) in enumerate(fl):
            if k1 == k2:       # Tr(S1' rev S1) Tr(S2' rev S2)
                state = (b1 + rev(a1), b2 + rev(a2))
            else:              # Tr(rev S1 . S1' . rev S2 . S2')
                state = (rev(a1) + b1 + rev(a2) + b2,)
            ok = all(sum(t.count(g) for t in state) == 2 for g in range(k))
            cf[i][j] = w[k1] * w[k2] * _traces(_canon(state)) if ok else Fraction(0)
    for i in range(len(fl)):
        for j in range(len(fl)):
            assert cf[i][j] == cf[j][i]
    return cf


# ------------------------------------------------------------------------------------------------------------------
# CUDA emission: one fused kernel per subprocess.  Constituent momenta (all massless, incoming): c_0..c_{k-1} the
# gluons, c_k = f_in (momentum carried along the fermion arrow at the start of the light line), c_{k+1} = -f_out
# (minus the one at its end); the pair is the constituent set {k, k+1}.  Every current is computed once (common
# sub-expressions by key).
# ------------------------------------------------------------------------------------------------------------------
HEADER = """// GENERATED by paper_2312_02898_b200/gen/quark.py (process generator, K0) — do not edit.
// process: %(proc)s   gluons: %(k)d   Feynman diagrams: %(ndiag)d
// this unit: whole process, fused (thread = event, JAMPs in registers); one light-quark line + the top line
// diagram terms: %(nterms)d   colour flows: %(ncol)d   helicities: %(nhel)d   static flops / helicity pass: %(flops)d
#include "mg_kernel.cuh"
namespace %(ns)s {
using namespace mgw;
constexpr int NPAR = %(npar)d, NGLU = %(k)d, NCOL = %(ncol)d, NHEL = %(nhel)d;
"""


def _bits(mask):
    return [i for i in range(32) if mask >> i & 1]


class _Emit:
    def __init__(self, qp):
        self.qp, self.k = qp, qp.k
        self.pairmask = 3 << qp.k
        self.memo, self.ops = {}, []
        self.gmasks, self.pmasks, self.umasks, self.vmasks, self.lmasks = set(), set(), set(), set(), set()
        self.counts = {}

    def _new(self, key, prefix, op):
        name = "%s%d" % (prefix, len(self.memo))
        self.memo[key] = name
        self.ops.append((name,) + op)
        self.counts[op[0]] = self.counts.get(op[0], 0) + 1
        return name

    def mask(self, tree, cfg):
        m = 0
        for leaf in topo.leaves_of(tree):
            if leaf == self.k:
                m |= self.pairmask
                for t in cfg[0] + cfg[1]:
                    m |= topo.leafmask(t)
            else:
                m |= 1 << leaf
        return m

    def seqmask(self, trees):
        m = 0
        for t in trees:
            m |= topo.leafmask(t)
        return m

    def gcur(self, tree, cfg):
        """Variable holding the off-shell current of a gluon tree (cfg: the light configuration behind leaf k)."""
        has_p = self.k in topo.leaves_of(tree)
        key = ("g", tree, cfg if has_p else None)
        if key in self.memo:
            return self.memo[key]
        if tree[0] == "g":
            if tree[1] != self.k:
                self.memo[key] = "e%d" % tree[1]
                return self.memo[key]
            a, b = cfg
            m = self.mask(tree, cfg)
            self.gmasks.add(m)
            return self._new(key, "jp", ("pair", self.vbar(a), self.ucol(b), m))
        m = self.mask(tree, cfg)
        self.gmasks.add(m)
        if tree[0] == "v3":
            ma, mb = self.mask(tree[1], cfg), self.mask(tree[2], cfg)
            self.pmasks.update((ma, mb))
            return self._new(key, "j", ("v3", self.gcur(tree[1], cfg), self.gcur(tree[2], cfg), ma, mb, m))
        return self._new(key, "j", ("k", self.gcur(tree[1], cfg), self.gcur(tree[2], cfg), self.gcur(tree[3], cfg), m))

    def vbar(self, seq):
        """Row spinor at the end of the light line's fermion flow after absorbing the blocks seq (string order)."""
        if not seq:
            return "lout"
        key = ("vb", seq)
        if key not in self.memo:
            m = self.seqmask(seq)
            self.vmasks.add(m)
            self._new(key, "vb", ("lqv", self.vbar(seq[:-1]), self.gcur(seq[-1], None), m))
        return self.memo[key]

    def ucol(self, seq):
        """Column spinor at the start of the flow; seq in string order: its first block is absorbed last."""
        if not seq:
            return "lin"
        key = ("uc", seq)
        if key not in self.memo:
            m = self.seqmask(seq)
            self.umasks.add(m)
            self._new(key, "uc", ("rqu", self.ucol(seq[1:]), self.gcur(seq[0], None), m))
        return self.memo[key]

    def lrow(self, blocks, cfg):
        """Top line from ubar(t) after absorbing the blocks (from the top quark's end)."""
        if not blocks:
            return "ub"
        has_p = any(self.k in topo.leaves_of(t) for t in blocks)
        key = ("lt", blocks, cfg if has_p else None)
        if key not in self.memo:
            m = 0
            for t in blocks:
                m |= self.mask(t, cfg)
            self.lmasks.add(m)
            self._new(key, "lt", ("lqt", self.lrow(blocks[:-1], cfg), self.gcur(blocks[-1], cfg), m))
        return self.memo[key]

    def amplitude(self, term):
        a, b, blocks = term
        cfg = (a, b)
        left = self.lrow(blocks[:-1], cfg)
        last = self.gcur(blocks[-1], cfg)
        key = ("bil", left)
        if key not in self.memo:
            self._new(key, "bl", ("bil", left, "vv"))
        name = "a%d" % len([o for o in self.ops if o[1] == "amp"])
        self.ops.append((name, "amp", self.memo[key], last))
        self.counts["amp"] = self.counts.get("amp", 0) + 1
        return name


def _colour_rows(cfi, ncol):
    return [[cfi[i][j] if j == i else (2 * cfi[i][j] if j > i else 0) for j in range(ncol)] for i in range(ncol)]


def emit_quark(spec, block=128, fp32=True):
    """One fused kernel for the subprocess `spec`.  Returns ([(filename, source)], info)."""
    qp = QProcess(spec)
    k, npar = qp.k, qp.npar
    terms = diagram_terms(k)
    fl = flows(k)
    index = {f: i for i, f in enumerate(fl)}
    ncol, nhel = len(fl), 1 << npar
    cf = colour_matrix(k)
    cfden = 1
    for row in cf:
        for v in row:
            cfden = lcm(cfden, v.denominator)
    cfi = [[int(v * cfden) for v in row] for row in cf]
    em = _Emit(qp)
    amps = [(em.amplitude(t), term_flows(t, k, index)) for t in terms]
    ampflows = dict(amps)
    flops = sum(FLOPS[{"lqv": "lq", "lqt": "lq", "rqu": "rq"}.get(kind, kind)] * n for kind, n in em.counts.items())
    flops += k * FLOPS["ext_g"] + 4 * FLOPS["ext_q"] + sum(FLOPS["jamp_add"] * len(f) for _, f in amps) + 2 * ncol * (ncol + 1)
    ns = "mg_" + qp.tag
    ndiag = n_feynman_diagrams(terms)
    out = [HEADER % dict(proc=qp.proc, k=k, ndiag=ndiag, nterms=len(terms), ncol=ncol, nhel=nhel, flops=flops, ns=ns, npar=npar)]
    w = out.append
    w("template <class T>\nMG_DEV void sigma_event(const double* __restrict__ mom, T* __restrict__ me_out, long long nevt,\n"
      "             long long ievt, const int* __restrict__ hel_list, const double* __restrict__ hel_w, int nhel_run,\n"
      "             T* __restrict__ perhel_out, double mt_d, double norm_d) {\n")
    # ---- helicity-independent part, in double ----
    w("  typedef P4<double> PD;\n  PD pp[NPAR];\n#pragma unroll\n  for (int i = 0; i < NPAR; ++i) load_momentum<double, NPAR>(mom, ievt, i, pp[i]);\n")
    w("  const PD ptd = pp[2];\n")

    def signed(part, plus):
        return "pp[%d]" % part if plus else "{{-pp[%d].c[0], -pp[%d].c[1], -pp[%d].c[2], -pp[%d].c[3]}}" % ((part,) * 4)

    w("  // massless incoming constituents: gluons, f_in (start of the light line's fermion flow), -f_out (its end)\n")
    for i, part in enumerate(qp.gpart):
        w("  const PD dm%d = %s;\n" % (1 << i, signed(part, part < 2)))
    w("  const PD dm%d = %s;\n" % (1 << k, signed(qp.pin, qp.in_is_u)))
    w("  const PD dm%d = %s;\n" % (1 << (k + 1), signed(qp.pout, not qp.out_is_ubar)))
    ubit, vbit = 1 << k, 1 << (k + 1)
    inv_masks = set(em.gmasks) | set(em.lmasks) | {g | ubit for g in em.umasks} | {g | vbit for g in em.vmasks}
    need = set(inv_masks) | set(em.pmasks)
    work = list(need)
    while work:
        m = work.pop()
        low = m & (m - 1)
        if low and low not in need:
            need.add(low)
            work.append(low)
    for m in sorted(need, key=lambda m: (bin(m).count("1"), m)):
        if len(_bits(m)) >= 2:
            w("  const PD dm%d = padd(dm%d, dm%d);\n" % (m, m & (m - 1), m & -m))
    pairs = set()
    for m in inv_masks:
        b = _bits(m)
        pairs.update((b[i], b[j]) for i in range(len(b)) for j in range(i + 1, len(b)))
    for a, b_ in sorted(pairs):
        w("  const double d%d_%d = 2.0 * pdot(dm%d, dm%d);\n" % (a, b_, 1 << a, 1 << b_))

    def psq(m):
        b = _bits(m)
        if len(b) < 2:
            return "0.0"
        return "(" + " + ".join("d%d_%d" % (b[i], b[j]) for i in range(len(b)) for j in range(i + 1, len(b))) + ")"

    w("  // propagator factors: sg = -1/P^2 (gluon currents), su / sv = -1/q^2 (light line), sl = -1/(q^2 - mt^2) (top line)\n")
    for m in sorted(em.gmasks):
        w("  const T sg%d = T(-1.0 / %s);\n" % (m, psq(m)))
    for g in sorted(em.umasks):
        w("  const T su%d = T(-1.0 / %s);\n  const P4<T> qu%d = pcast<T>(dm%d);\n" % (g, psq(g | ubit), g, g | ubit))
    for g in sorted(em.vmasks):
        w("  const T sv%d = T(-1.0 / %s);\n  const P4<T> qv%d = pcast<T>(psub(PD{{0.0, 0.0, 0.0, 0.0}}, dm%d));\n" % (g, psq(g | vbit), g, g | vbit))
    for m in sorted(em.lmasks):
        w("  const T sl%d = T(-1.0 / (%s - 2.0 * pdot(ptd, dm%d)));\n  const P4<T> ql%d = pcast<T>(psub(ptd, dm%d));\n" % (m, psq(m), m, m, m))
    for m in sorted(em.pmasks):
        w("  const P4<T> pm%d = pcast<T>(dm%d);\n" % (m, m))
    w("  P4<T> pq[NPAR];\n#pragma unroll\n  for (int i = 0; i < NPAR; ++i) pq[i] = pcast<T>(pp[i]);\n")
    w("  const T mt = T(mt_d);\n  T me = T(0);\n")
    # ---- helicity loop ----
    w("#pragma unroll 1\n  for (int ih = 0; ih < nhel_run; ++ih) {\n    const int h = hel_list[ih];\n")
    for i, part in enumerate(qp.gpart):
        w("    W4<T> e%d; ext_gluon(pq[%d], hel_of<NPAR>(h, %d), %s, e%d);\n" % (i, part, part, "false" if part < 2 else "true", i))
    w("    W4<T> lin, lout, ub, vv;\n")
    w("    %s(pq[%d], T(0), hel_of<NPAR>(h, %d), lin);\n" % ("ext_u" if qp.in_is_u else "ext_v", qp.pin, qp.pin))
    w("    %s(pq[%d], T(0), hel_of<NPAR>(h, %d), lout);\n" % ("ext_ubar" if qp.out_is_ubar else "ext_vbar", qp.pout, qp.pout))
    w("    ext_ubar(pq[2], mt, hel_of<NPAR>(h, 2), ub);\n    ext_v(pq[3], mt, hel_of<NPAR>(h, 3), vv);\n")
    w("    T " + ", ".join("jr%d = T(0), ji%d = T(0)" % (f, f) for f in range(ncol)) + ";\n")
    for op in em.ops:
        name, kind = op[0], op[1]
        if kind == "pair":
            w("    W4<T> %s; cur_pair(%s, %s, sg%d, %s);\n" % (name, op[2], op[3], op[4], name))
        elif kind == "v3":
            w("    W4<T> %s; cur_v3(pm%d, %s, pm%d, %s, sg%d, %s);\n" % (name, op[4], op[2], op[5], op[3], op[6], name))
        elif kind == "k":
            w("    W4<T> %s; cur_k(%s, %s, %s, sg%d, %s);\n" % (name, op[2], op[3], op[4], op[5], name))
        elif kind == "lqv":
            w("    W4<T> %s; cur_lq(%s, %s, qv%d, T(0), sv%d, %s);\n" % (name, op[2], op[3], op[4], op[4], name))
        elif kind == "rqu":
            w("    W4<T> %s; cur_rq(%s, %s, qu%d, T(0), su%d, %s);\n" % (name, op[2], op[3], op[4], op[4], name))
        elif kind == "lqt":
            w("    W4<T> %s; cur_lq(%s, %s, ql%d, mt, sl%d, %s);\n" % (name, op[2], op[3], op[4], op[4], name))
        elif kind == "bil":
            w("    W4<T> %s; bilinear(%s, %s, %s);\n" % (name, op[2], op[3], name))
        elif kind == "amp":
            w("    const C1<T> %s = contract(%s, %s);" % (name, op[2], op[3]))
            for f, s in ampflows[name]:
                sg = "+=" if s > 0 else "-="
                w(" jr%d %s %s.r; ji%d %s %s.i;" % (f, sg, name, f, sg, name))
            w("\n")
    rows = _colour_rows(cfi, ncol)
    w("    T meh = T(0);\n")
    for i in range(ncol):
        zr = " + ".join("T(%d) * jr%d" % (rows[i][j], j) for j in range(i, ncol) if rows[i][j])
        zi = " + ".join("T(%d) * ji%d" % (rows[i][j], j) for j in range(i, ncol) if rows[i][j])
        w("    meh += jr%d * (%s);\n    meh += ji%d * (%s);\n" % (i, zr, i, zi))
    w("    if (perhel_out) perhel_out[(long long)ih * nevt + ievt] = meh * T(norm_d);\n")
    w("    me += T(hel_w[ih]) * meh;\n  }\n  me_out[ievt] = me * T(norm_d);\n}\n")
    # ---- kernel, launcher, descriptor ----
    w("#ifdef __CUDACC__\ntemplate <class T>\n__global__ void __launch_bounds__(%d)\n" % block)
    w("sigma_kernel(const double* __restrict__ mom, T* __restrict__ me_out, long long nevt,\n"
      "             const int* __restrict__ hel_list, const double* __restrict__ hel_w, int nhel_run,\n"
      "             T* __restrict__ perhel_out, double mt_d, double norm_d) {\n"
      "  const long long ievt = (long long)blockIdx.x * blockDim.x + threadIdx.x;\n  if (ievt >= nevt) return;\n"
      "  sigma_event<T>(mom, me_out, nevt, ievt, hel_list, hel_w, nhel_run, perhel_out, mt_d, norm_d);\n}\n")
    fp32line = ("  else sigma_kernel<float><<<grid, block, 0, st>>>(mom, (float*)me_out, nevt, hel_list, hel_w, nhel_run, "
                "(float*)perhel_out, par[1], norm);") if fp32 else "  else return -1;"
    w("""
static int launch(int prec, const double* mom, void* me_out, long long nevt, const int* hel_list, const double* hel_w,
                  int nhel_run, void* perhel_out, const double* par, cudaStream_t st) {
  // par[0] = g_s^2, par[1] = mt; |M|^2 ~ g_s^(2 (k + 2)); 4 = the 1/2 of each Fierz term, squared
  double norm = 1.0;
  for (int i = 0; i < NGLU + 2; ++i) norm *= par[0];
  norm /= (double)%d * 4.0 * (double)%d;
  const int block = %d;
  const unsigned grid = (unsigned)((nevt + block - 1) / block);
  if (grid == 0) return 0;
  if (prec == 0) sigma_kernel<double><<<grid, block, 0, st>>>(mom, (double*)me_out, nevt, hel_list, hel_w, nhel_run, (double*)perhel_out, par[1], norm);
%s
  return 1;
}
#endif  // __CUDACC__
}  // namespace
""" % (cfden, qp.denominator, block, fp32line))
    mass = ", ".join(str(x) for x in qp.massive)
    w("""#ifdef __CUDACC__
extern const mg_procdesc_t mg_desc_%(tag)s = {"%(proc)s", %(npar)d, %(k)d, %(ndiag)d, %(nhel)d, %(ncol)d, %(denom)d,
  %(flops)dLL, {%(mass)s}, %(ns)s::launch, nullptr, {0, 0}, 1, %(fp32)d, {0, 0}, %(flops)dLL, 0LL, 0LL, {0, 0}, 0, 0};
#endif  // __CUDACC__
""" % dict(tag=qp.tag, proc=qp.proc, npar=npar, k=k, ndiag=ndiag, nhel=nhel, ncol=ncol, denom=qp.denominator,
           flops=flops, mass=mass, ns=ns, fp32=1 if fp32 else 0))
    info = dict(proc=qp.proc, ns=ns, spec=spec, npar=npar, ncol=ncol, nhel=nhel, ndiagrams=ndiag, nterms=len(terms),
                flops_per_helicity=flops, counts=dict(em.counts), shape="fused", ngroups=1, cfden=cfden,
                denominator=qp.denominator)
    return [(ns + ".cu", "".join(out))], info
