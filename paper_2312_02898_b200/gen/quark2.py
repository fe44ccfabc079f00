"""Quark channels of p p -> t t~ + 2 jets with TWO light-quark lines and no gluon:
    q q~ -> t t~ r r~,  q r -> t t~ q r,  q r~ -> t t~ q r~, ...   (two flavours: 7 Feynman diagrams)
    q q~ -> t t~ q q~,  q q -> t t~ q q,  q~ q~ -> t t~ q~ q~      (one flavour: 14 diagrams, two pairings, Fermi sign)
Companion of quark.py (one light line); same device routines, same fused kernel shape.

Diagrams.  As in quark.py the pair of light line l with everything it absorbed is a pseudo-gluon P_l.  With no gluon
there are seven ways of tying the three quark lines together, for a given pairing of line starts with line ends:
    the top line absorbs P_0 then P_1, or P_1 then P_0                              (top line in the middle)
    the top line absorbs the three-gluon vertex v3(P_0, P_1)
    line 0 absorbs P_1 before or after its own off-shell gluon; the top absorbs that  (line 0 in the middle)
    the same with the lines exchanged                                                (line 1 in the middle)
Colour.  Strings of pseudo-gluon labels on the three open lines (row index = top / end of a light line, column index =
antitop / start of a light line), the commutator of the three-gluon vertex expanded as in topology.orderings; every
pseudo label is removed with the Fierz identity
    (X T^x Y)_{r1 c1} (Z T^x W)_{r2 c2} = 1/2 (X W)_{r1 c2} (Z Y)_{r2 c1} - 1/(2N) (X Y)_{r1 c1} (Z W)_{r2 c2},
which leaves products of three Kronecker deltas: the 3! = 6 colour flows (bijections rows -> columns), with rational
coefficients (common denominator 4 N^2 = 36).  The colour matrix of two flows is N^(number of closed loops).
Same flavour twice: the second pairing connects the same particles the other way and enters with a minus sign.
"""
from fractions import Fraction
from itertools import permutations
from math import factorial, lcm

from .colour import NC

FLOPS = {"v3": 156, "lq": 120, "rq": 120, "bil": 72, "amp": 30, "pair": 80, "ext_q": 50}
NAMES = {"q": "q", "Q": "q~", "r": "r", "R": "r~", "g": "g", "t": "t", "T": "t~"}
TAGS = {"q": "q", "Q": "qx", "r": "r", "R": "rx", "g": "g", "t": "t", "T": "tx"}

# two flavours, then one flavour; beams first, "tT", then the two jets
SPECS = ("qQtTrR", "QqtTrR", "qrtTqr", "qRtTqR", "QrtTQr", "QRtTQR",
         "qQtTqQ", "QqtTqQ", "qqtTqq", "QQtTQQ")


class QProcess2:
    def __init__(self, spec):
        assert len(spec) == 6 and spec[2:4] == "tT" and all(c in "qQrR" for c in spec[:2] + spec[4:]), spec
        self.spec, self.npar = spec, 6
        self.light = [0, 1, 4, 5]                                  # particle index of light particle j (= constituent bit j)
        is_q = lambda c: c in "qr"
        self.start = {i: is_q(spec[i]) == (i < 2) for i in self.light}   # incoming quark / outgoing antiquark start a flow
        st = {f: [i for i in self.light if self.start[i] and spec[i].lower() == f] for f in "qr"}
        en = {f: [i for i in self.light if not self.start[i] and spec[i].lower() == f] for f in "qr"}
        assert len(st["q"]) == len(en["q"]) and len(st["r"]) == len(en["r"]), spec
        if len(st["q"]) == 1 and len(st["r"]) == 1:
            self.pairings = [(((st["q"][0], en["q"][0]), (st["r"][0], en["r"][0])), 1)]
        else:
            assert len(st["q"]) == 2 and not st["r"], spec
            (s0, s1), (e0, e1) = st["q"], en["q"]
            self.pairings = [(((s0, e0), (s1, e1)), 1), (((s0, e1), (s1, e0)), -1)]
        d = 36
        for c in set(spec[4:]):
            d *= factorial(spec[4:].count(c))
        self.denominator = d
        self.proc = " ".join(NAMES[c] for c in spec[:2]) + " > " + " ".join(NAMES[c] for c in spec[2:])
        self.tag = "".join(TAGS[c] for c in spec)
        self.massive = [1 if c in "tT" else 0 for c in spec]


# ---------------------------------------------------------------------------------------------------------------- terms
# a term: (name, top string, string of line 0, string of line 1) with signs; strings hold the pseudo labels "P0", "P1"
def terms():
    """[(kind, [(sign, top, line0, line1)])]: the seven terms of one pairing with their colour strings."""
    P0, P1 = "P0", "P1"
    return [
        ("top01", [(1, (P0, P1), (P0,), (P1,))]),
        ("top10", [(1, (P1, P0), (P0,), (P1,))]),
        ("v3", [(1, (P0, P1), (P0,), (P1,)), (-1, (P1, P0), (P0,), (P1,))]),
        ("l0A", [(1, (P0,), (P1, P0), (P1,))]),          # line 0 absorbs P1 before its own gluon (towards the end of its flow)
        ("l0B", [(1, (P0,), (P0, P1), (P1,))]),
        ("l1A", [(1, (P1,), (P0,), (P0, P1))]),
        ("l1B", [(1, (P1,), (P0,), (P1, P0))]),
    ]


def _fierz(lines, label):
    """lines: {row: (col, string)}; removes `label` (which sits on two different lines); returns [(coef, lines')]."""
    hits = [(r, c, s) for r, (c, s) in lines.items() if label in s]
    assert len(hits) == 2, (lines, label)
    (r1, c1, s1), (r2, c2, s2) = hits
    i1, i2 = s1.index(label), s2.index(label)
    x, y, z, w = s1[:i1], s1[i1 + 1:], s2[:i2], s2[i2 + 1:]
    a = dict(lines); a[r1] = (c2, x + w); a[r2] = (c1, z + y)
    b = dict(lines); b[r1] = (c1, x + y); b[r2] = (c2, z + w)
    return [(Fraction(1, 2), a), (Fraction(-1, 2 * NC), b)]


def term_colour(strings, rows, cols, canon_rows):
    """{flow: coefficient}: rows / cols = (top, end of line 0, end of line 1) / (antitop, start of line 0, start of line 1)
    of this pairing; flow = tuple over `canon_rows` (the same for every pairing) of the column each row is connected to."""
    out = {}
    for sign, top, l0, l1 in strings:
        work = [(Fraction(sign), {rows[0]: (cols[0], top), rows[1]: (cols[1], l0), rows[2]: (cols[2], l1)})]
        for label in ("P0", "P1"):
            work = [(c * cf, ln) for c, lines in work for cf, ln in _fierz(lines, label)]
        for c, lines in work:
            assert all(not s for _, s in lines.values())
            key = tuple(lines[r][0] for r in canon_rows)
            out[key] = out.get(key, 0) + c
    return {k_: v for k_, v in out.items() if v != 0}


def flow_matrix(flows, rows):
    """CF[f][g] = sum over colours of f^* g = N^(loops) for two delta products."""
    cf = []
    for f in flows:
        inv = {c: r for r, c in zip(rows, f)}              # f^*: from a column back to its row
        row = []
        for g in flows:
            gm = dict(zip(rows, g))
            seen, loops = set(), 0
            for r in rows:
                if r in seen:
                    continue
                loops += 1
                x = r
                while x not in seen:
                    seen.add(x)
                    x = inv[gm[x]]
            row.append(NC ** loops)
        cf.append(row)
    return cf


# ------------------------------------------------------------------------------------------------------------- emission
HEADER = """// GENERATED by paper_2312_02898_b200/gen/quark2.py (process generator, K0) — do not edit.
// process: %(proc)s   gluons: 0   Feynman diagrams: %(ndiag)d
// this unit: whole process, fused (thread = event, JAMPs in registers); two light-quark lines + the top line
// diagram terms: %(ndiag)d   colour flows: %(ncol)d   helicities: %(nhel)d   static flops / helicity pass: %(flops)d
#include "mg_kernel.cuh"
namespace %(ns)s {
using namespace mgw;
constexpr int NPAR = %(npar)d, NGLU = 0, NCOL = %(ncol)d, NHEL = %(nhel)d;
"""


def _bits(mask):
    return [i for i in range(8) if mask >> i & 1]


def emit_quark2(spec, block=128, fp32=True):
    """One fused kernel for the two-light-line subprocess `spec`.  Returns ([(filename, source)], info)."""
    qp = QProcess2(spec)
    npar, nhel = 6, 64
    bit = {part: 1 << j for j, part in enumerate(qp.light)}      # massless incoming constituents: +p incoming, -p outgoing
    (base_lines, _) = qp.pairings[0]
    canon_rows = ("t", base_lines[0][1], base_lines[1][1])
    canon_cols = ("T", base_lines[0][0], base_lines[1][0])
    flows = list(permutations(canon_cols))
    findex = {f: i for i, f in enumerate(flows)}
    ncol = len(flows)
    cf = flow_matrix(flows, canon_rows)

    # ---- ops of every pairing: (name, kind, args...) with common sub-expressions shared, and the JAMP coefficients
    ops, names, masks = [], {}, dict(sg=set(), su=set(), sv=set(), sl=set(), pm=set())
    counts = {}

    def new(key, prefix, op):
        if key not in names:
            names[key] = "%s%d" % (prefix, len(names))
            ops.append((names[key],) + op)
            counts[op[0]] = counts.get(op[0], 0) + 1
        return names[key]

    amps = []                                                       # (name, {flow index: Fraction})
    for ip, (lines, fermi) in enumerate(qp.pairings):
        (s0, e0), (s1, e1) = lines
        m = [bit[s0] | bit[e0], bit[s1] | bit[e1]]
        se = [(s0, e0), (s1, e1)]
        rows, cols = ("t", e0, e1), ("T", s0, s1)
        J = []
        for l in (0, 1):
            masks["sg"].add(m[l])
            J.append(new(("pair", se[l]), "jp", ("pair", "x%d" % se[l][1], "x%d" % se[l][0], m[l])))
        allm = m[0] | m[1]
        masks["sg"].add(allm)
        blub = new(("bil", "ub"), "bl", ("bil", "ub", "vv"))

        def closing(kind, l):
            """The pseudo-gluon of line l with the other line's pair absorbed before (A) / after (B) its own gluon."""
            o = 1 - l
            s, e = se[l]
            if kind == "A":
                g = m[o] | bit[e]
                masks["sv"].add(g)
                v = new(("vb", se[l], se[o]), "vb", ("lqv", "x%d" % e, J[o], g))
                return new(("pairA", se[l], se[o]), "jp", ("pair", v, "x%d" % s, allm))
            g = m[o] | bit[s]
            masks["su"].add(g)
            u = new(("uc", se[l], se[o]), "uc", ("rqu", "x%d" % s, J[o], g))
            return new(("pairB", se[l], se[o]), "jp", ("pair", "x%d" % e, u, allm))

        for kind, strings in terms():
            if kind in ("top01", "top10"):
                a, b_ = (0, 1) if kind == "top01" else (1, 0)
                masks["sl"].add(m[a])
                lt = new(("lt", se[a]), "lt", ("lqt", "ub", J[a], m[a]))
                bl = new(("bil", lt), "bl", ("bil", lt, "vv"))
                last = J[b_]
            elif kind == "v3":
                masks["pm"].update(m)
                bl, last = blub, new(("v3", lines), "j", ("v3", J[0], J[1], m[0], m[1], allm))
            else:
                bl, last = blub, closing(kind[2], int(kind[1]))
            name = "a%d" % len(amps)
            ops.append((name, "amp", bl, last))
            counts["amp"] = counts.get("amp", 0) + 1
            col = term_colour(strings, rows, cols, canon_rows)
            amps.append((name, {findex[f]: fermi * c for f, c in col.items()}))
    den = 1
    for _, col in amps:
        for c in col.values():
            den = lcm(den, c.denominator)
    ampflows = {name: sorted((f, int(c * den)) for f, c in col.items()) for name, col in amps}
    ndiag = 7 * len(qp.pairings)
    flops = sum(FLOPS[{"lqv": "lq", "lqt": "lq", "rqu": "rq"}.get(kind, kind)] * n for kind, n in counts.items())
    flops += 6 * FLOPS["ext_q"] + sum(4 * len(f) for f in ampflows.values()) + 2 * ncol * (ncol + 1)
    ns = "mg_" + qp.tag
    out = [HEADER % dict(proc=qp.proc, ndiag=ndiag, ncol=ncol, nhel=nhel, flops=flops, ns=ns, npar=npar)]
    w = out.append
    w("template <class T>\nMG_DEV void sigma_event(const double* __restrict__ mom, T* __restrict__ me_out, long long nevt,\n"
      "             long long ievt, const int* __restrict__ hel_list, const double* __restrict__ hel_w, int nhel_run,\n"
      "             T* __restrict__ perhel_out, double mt_d, double norm_d) {\n")
    w("  typedef P4<double> PD;\n  PD pp[NPAR];\n#pragma unroll\n  for (int i = 0; i < NPAR; ++i) load_momentum<double, NPAR>(mom, ievt, i, pp[i]);\n")
    w("  const PD ptd = pp[2];\n  // massless incoming constituents: +p for the beams, -p for the jets\n")
    for part in qp.light:
        w("  const PD dm%d = %s;\n" % (bit[part], "pp[%d]" % part if part < 2 else
                                       "{{-pp[%d].c[0], -pp[%d].c[1], -pp[%d].c[2], -pp[%d].c[3]}}" % ((part,) * 4)))
    need = set()
    for k_ in masks:
        need |= masks[k_]
    work = list(need)
    while work:
        mm = work.pop()
        low = mm & (mm - 1)
        if low and low not in need:
            need.add(low)
            work.append(low)
    for mm in sorted(need, key=lambda x: (bin(x).count("1"), x)):
        if len(_bits(mm)) >= 2:
            w("  const PD dm%d = padd(dm%d, dm%d);\n" % (mm, mm & (mm - 1), mm & -mm))
    for a in range(4):
        for b_ in range(a + 1, 4):
            w("  const double d%d_%d = 2.0 * pdot(dm%d, dm%d);\n" % (a, b_, 1 << a, 1 << b_))

    def psq(mm):
        b = _bits(mm)
        return "(" + " + ".join("d%d_%d" % (b[i], b[j]) for i in range(len(b)) for j in range(i + 1, len(b))) + ")"

    w("  // propagator factors: sg = -1/P^2 (gluon currents), su / sv = -1/q^2 (light lines), sl = -1/(q^2 - mt^2) (top line)\n")
    for mm in sorted(masks["sg"]):
        w("  const T sg%d = T(-1.0 / %s);\n" % (mm, psq(mm)))
    for mm in sorted(masks["su"]):
        w("  const T su%d = T(-1.0 / %s);\n  const P4<T> qu%d = pcast<T>(dm%d);\n" % (mm, psq(mm), mm, mm))
    for mm in sorted(masks["sv"]):
        w("  const T sv%d = T(-1.0 / %s);\n  const P4<T> qv%d = pcast<T>(psub(PD{{0.0, 0.0, 0.0, 0.0}}, dm%d));\n" % (mm, psq(mm), mm, mm))
    for mm in sorted(masks["sl"]):
        w("  const T sl%d = T(-1.0 / (%s - 2.0 * pdot(ptd, dm%d)));\n  const P4<T> ql%d = pcast<T>(psub(ptd, dm%d));\n" % (mm, psq(mm), mm, mm, mm))
    for mm in sorted(masks["pm"]):
        w("  const P4<T> pm%d = pcast<T>(dm%d);\n" % (mm, mm))
    w("  P4<T> pq[NPAR];\n#pragma unroll\n  for (int i = 0; i < NPAR; ++i) pq[i] = pcast<T>(pp[i]);\n")
    w("  const T mt = T(mt_d);\n  T me = T(0);\n")
    w("#pragma unroll 1\n  for (int ih = 0; ih < nhel_run; ++ih) {\n    const int h = hel_list[ih];\n")
    w("    W4<T> " + ", ".join("x%d" % part for part in qp.light) + ", ub, vv;\n")
    for part in qp.light:
        quark = spec[part] in "qr"
        fn = ("ext_u" if quark else "ext_v") if qp.start[part] else ("ext_ubar" if quark else "ext_vbar")
        w("    %s(pq[%d], T(0), hel_of<NPAR>(h, %d), x%d);\n" % (fn, part, part, part))
    w("    ext_ubar(pq[2], mt, hel_of<NPAR>(h, 2), ub);\n    ext_v(pq[3], mt, hel_of<NPAR>(h, 3), vv);\n")
    w("    T " + ", ".join("jr%d = T(0), ji%d = T(0)" % (f, f) for f in range(ncol)) + ";\n")
    for op in ops:
        name, kind = op[0], op[1]
        if kind == "pair":
            w("    W4<T> %s; cur_pair(%s, %s, sg%d, %s);\n" % (name, op[2], op[3], op[4], name))
        elif kind == "v3":
            w("    W4<T> %s; cur_v3(pm%d, %s, pm%d, %s, sg%d, %s);\n" % (name, op[4], op[2], op[5], op[3], op[6], name))
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
            for f, c in ampflows[name]:
                sg = "+=" if c > 0 else "-="
                mul = "" if abs(c) == 1 else "T(%d) * " % abs(c)
                w(" jr%d %s %s%s.r; ji%d %s %s%s.i;" % (f, sg, mul, name, f, sg, mul, name))
            w("\n")
    w("    T meh = T(0);\n")
    for i in range(ncol):
        row = [cf[i][j] if j == i else 2 * cf[i][j] for j in range(ncol)]
        zr = " + ".join("T(%d) * jr%d" % (row[j], j) for j in range(i, ncol))
        zi = " + ".join("T(%d) * ji%d" % (row[j], j) for j in range(i, ncol))
        w("    meh += jr%d * (%s);\n    meh += ji%d * (%s);\n" % (i, zr, i, zi))
    w("    if (perhel_out) perhel_out[(long long)ih * nevt + ievt] = meh * T(norm_d);\n")
    w("    me += T(hel_w[ih]) * meh;\n  }\n  me_out[ievt] = me * T(norm_d);\n}\n")
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
  // par[0] = g_s^2, par[1] = mt; |M|^2 ~ g_s^8; %d = the common denominator of the Fierz coefficients, squared below
  double norm = par[0] * par[0] * par[0] * par[0];
  norm /= (double)%d * (double)%d * (double)%d;
  const int block = %d;
  const unsigned grid = (unsigned)((nevt + block - 1) / block);
  if (grid == 0) return 0;
  if (prec == 0) sigma_kernel<double><<<grid, block, 0, st>>>(mom, (double*)me_out, nevt, hel_list, hel_w, nhel_run, (double*)perhel_out, par[1], norm);
%s
  return 1;
}
#endif  // __CUDACC__
}  // namespace
""" % (den, den, den, qp.denominator, block, fp32line))
    mass = ", ".join(str(x) for x in qp.massive)
    w("""#ifdef __CUDACC__
extern const mg_procdesc_t mg_desc_%(tag)s = {"%(proc)s", %(npar)d, 0, %(ndiag)d, %(nhel)d, %(ncol)d, %(denom)d,
  %(flops)dLL, {%(mass)s}, %(ns)s::launch, nullptr, {0, 0}, 1, %(fp32)d, {0, 0}, %(flops)dLL, 0LL, 0LL, {0, 0}, 0, 0};
#endif  // __CUDACC__
""" % dict(tag=qp.tag, proc=qp.proc, npar=npar, ndiag=ndiag, nhel=nhel, ncol=ncol, denom=qp.denominator,
           flops=flops, mass=mass, ns=ns, fp32=1 if fp32 else 0))
    info = dict(proc=qp.proc, ns=ns, spec=spec, npar=npar, ncol=ncol, nhel=nhel, ndiagrams=ndiag, nterms=ndiag,
                flops_per_helicity=flops, counts=dict(counts), shape="fused", ngroups=1, cfden=den * den,
                denominator=qp.denominator)
    return [(ns + ".cu", "".join(out))], info
