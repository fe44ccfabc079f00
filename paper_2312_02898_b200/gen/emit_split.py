"""Split kernel shape (n >= 4 gluons): invariants + diagram-group + colour + helicity-sum kernels.

Workspace for one tile of E events and H helicities (element type T, event index fastest):
    jamp[H][NCOL][2][E]    JAMPs, accumulated in place by the diagram-group kernels: the first kernel (in launch
                           order) that touches a flow stores, later kernels add with L2 reductions (reduce_mode
                           "red"; "slots" = the earlier scheme with private partial slots + a gather kernel);
    meh[H][E]              J^dagger CF J per (event, helicity) (colour kernel);
    inv[NINV][E]           helicity-independent per-event tables (invariants kernel).
The launcher loops over event tiles (and helicity chunks if the workspace the API layer allocated is smaller than
one tile with all helicities: mg_api.cu, MG5B200_WS_GB).
"""
from math import factorial

from .colour import colour_matrix, common_denominator
from .plan import Plan, partition_terms


def choose_kernels(n, max_terms, live_max, acc_max, flat_phase=0):
    """Kernels (coarse diagram groups) and their phases: every kernel is split into as few phases as keep the
    number of simultaneously live currents of each phase <= live_max (register pressure), because every extra
    phase recomputes the low-multiplicity currents it shares with its neighbours."""
    import os
    flat = int(os.environ.get("MG_FLATPHASE", "0")) or flat_phase
    if isinstance(flat, dict):
        flat = dict(flat)
    if flat and os.environ.get("MG_FLAT_LR"):
        flat = {"*": flat, "L": int(os.environ["MG_FLAT_LR"]), "R": int(os.environ["MG_FLAT_LR"])}
    if flat and os.environ.get("MG_FLAT_A"):
        flat = dict(flat) if isinstance(flat, dict) else {"*": flat}
        flat["A"] = int(os.environ["MG_FLAT_A"])
    if flat and os.environ.get("MG_FLAT_T"):
        flat = dict(flat) if isinstance(flat, dict) else {"*": flat}
        flat["T"] = int(os.environ["MG_FLAT_T"])
    if flat:
        # every phase its own kernel: short straight-line bodies that stay resident in the instruction caches
        return [[Plan(n, terms=ph, acc_max=acc_max)] for k in partition_terms(n, max_terms=max_terms, max_phase=flat)
                for ph in k]
    cands = [10 ** 6, 128, 96, 64, 48, 32, 24, 16, 8]
    parts = {mp: partition_terms(n, max_terms=max_terms, max_phase=mp) for mp in cands}
    out = []
    for i in range(len(parts[cands[0]])):
        for mp in cands:
            plans = [Plan(n, terms=ph, acc_max=acc_max) for ph in parts[mp][i]]
            if max(p.max_live() for p in plans) <= live_max or mp == cands[-1]:
                out.append(plans)
                break
    return out


# measured on B200: short kernels win — their straight-line bodies stay in the instruction caches and
# their live state fits the register file — even though every extra kernel recomputes a few shared currents and
# adds partial-JAMP slots.  n = 4: 7 kernels of <= 40 terms; n = 5: 86 kernels of <= 24 terms (<= 12 for the
# single-block 5-gluon trees, whose amplitudes touch the most colour flows).
TUNED = {4: dict(max_terms=40, live_max=1000, flat_phase=0, prefetch=0),
         5: dict(max_terms=170, live_max=12, flat_phase={"*": 24, "T": 12}, prefetch=1)}


def emit_split(n, block=128, fp32=True, acc_max=24, max_terms=None, sync_every=2, minblocks=2, live_max=None, flat_phase=None, noinline=False,
               stage_kb=110, reduce_mode="red", prefetch=None):
    from . import emit as E
    tuned = TUNED.get(n, TUNED[5])
    max_terms = max_terms or tuned["max_terms"]
    live_max = live_max or tuned["live_max"]
    flat_phase = tuned["flat_phase"] if flat_phase is None else flat_phase
    prefetch = tuned["prefetch"] if prefetch is None else prefetch      # n = 5: +1.2 %; n = 4: -1.5 % (measured)
    kernels = choose_kernels(n, max_terms, live_max, acc_max, flat_phase)
    npar, nhel = n + 2, 1 << (n + 2)
    ns = "mg_ggtt" + "g" * (n - 2)
    proc = "g g > t t~" + " g" * (n - 2)
    cf = colour_matrix(n)
    cfden = common_denominator(cf)
    ncol = len(cf)
    cfi = [[int(v * cfden) for v in row] for row in cf]
    plans = [p for k in kernels for p in k]
    union = E._Union(n, plans)
    inv = union.items()
    ninv = union.nitems
    ndiag = plans[0].ndiagrams
    files, ginfo = [], []
    total_flops = 0
    part_of_flow = {f: [] for f in range(ncol)}     # flow -> global partial slots
    written_flows = set()                            # reduce_mode "red": flows some earlier kernel has stored
    base = 0
    nkern = len(kernels)
    ext_flops = 0      # external wavefunctions come from per-event tables (invariants kernel): no FLOPs per helicity
    for gi, phases in enumerate(kernels):
        flops = sum(p.flops_per_helicity(colour=False, externals=False) for p in phases) + ext_flops
        total_flops += flops
        touched = sorted(set().union(*[p.flows_touched() for p in phases]))
        nterms = sum(len(p.terms) for p in phases)
        live = max(p.max_live() for p in phases)
        slot = {f: i for i, f in enumerate(touched)}
        for f in touched:
            part_of_flow[f].append(base + slot[f])
        first_writer = [f for f in touched if f not in written_flows]
        written_flows.update(touched)
        gblock = block
        while 2 * len(touched) * gblock * 8 > 225 * 1024:
            gblock -= 32
        smem64 = 2 * len(touched) * gblock * 8
        # invariants staged in shared memory: as many of the most used items as fit next to the partial JAMPs while
        # two CTAs still share an SM (stage_kb per CTA); the rest stays in the global buffer
        probe = E.InvAccess(inv, union.sizes)
        E._externals(_AllExternals(n), lambda x: None, probe)
        for plan in phases:
            E._body(plan, lambda x: None, lambda *a: None, probe)
        budget = max(0, (stage_kb * 1024 - smem64) // (8 * gblock)) if stage_kb else 0
        staged, nstage = {}, 0
        for name in sorted(probe.count, key=lambda k_: (-probe.count[k_], k_)):
            size = union.sizes[name]
            if nstage + size <= budget:
                staged[name] = nstage
                nstage += size
        acc = E.InvAccess(inv, union.sizes, staged)
        smem64 += nstage * gblock * 8
        gmin = max(1, min(minblocks, (227 * 1024) // (smem64 + 1024)))
        out = [E.HEADER % dict(proc=proc, n=n, ndiag=ndiag, nterms=nterms, ncol=ncol, nhel=nhel, flops=flops, ns=ns,
                               npar=npar, what="diagram group %d of %d, %d phase(s) (partial JAMP slots %d..%d)"
                               % (gi, nkern, len(phases), base, base + len(touched) - 1))]
        w = out.append
        if noinline:
            out[0] = "#define MG_NOINLINE_ROUTINES 1\n" + out[0]
        w("constexpr int BLK = %d, NTOUCH = %d, PBASE = %d, NSTAGE = %d;\n" % (gblock, len(touched), base, nstage))
        w("template <class T>\n__global__ void __launch_bounds__(%d, %d)\n" % (gblock, gmin))
        w("group%d_kernel(long long nevt, const int* __restrict__ hel_list, int hcount, int per_thread, int npart,\n"
          "              T* __restrict__ part, const T* __restrict__ invbuf, long long stride, double mt_d) {\n" % gi)
        w("  extern __shared__ __align__(16) unsigned char smem_raw[];\n")
        w("  T* __restrict__ sj = reinterpret_cast<T*>(smem_raw) + threadIdx.x;\n")
        w("  const long long ievt0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;\n")
        w("  const bool live = ievt0 < nevt;\n  const long long ievt = live ? ievt0 : nevt - 1;\n")
        w("  const T* __restrict__ inv = invbuf + ievt;\n  const T mt = T(mt_d);\n")
        w("  T* __restrict__ sinv = sj + 2 * NTOUCH * BLK;    // staged invariants, sinv[slot][thread]\n")
        for name, sl in sorted(staged.items(), key=lambda kv: kv[1]):
            for m in range(union.sizes[name]):
                w("  sinv[%d * BLK] = inv[%d * stride];\n" % (sl + m, inv[name] + m))
        w("  const int ih0 = blockIdx.y * per_thread, ih1 = min(hcount, ih0 + per_thread);\n")
        w("#pragma unroll 1\n  for (int ih = ih0; ih < ih1; ++ih) {\n")
        w("    const int h = hel_list[ih];\n")
        E._externals(_AllExternals(n), w, acc)
        local_written = set()

        def sink(f, s, re, im, slot=slot, local_written=local_written, w=w):
            a, b_ = 2 * slot[f], 2 * slot[f] + 1
            if f in local_written:
                sg = "+=" if s > 0 else "-="
                w("    sj[%d * BLK] %s %s; sj[%d * BLK] %s %s;\n" % (a, sg, E._mul(s, re), b_, sg, E._mul(s, im)))
            else:
                local_written.add(f)
                neg = "" if s > 0 else "-"
                w("    sj[%d * BLK] = %s%s; sj[%d * BLK] = %s%s;\n" % (a, neg, E._mul(s, re), b_, neg, E._mul(s, im)))

        for pi, plan in enumerate(phases):
            w("    {   // phase %d: %d terms, <= %d live currents\n" % (pi, len(plan.terms), plan.max_live()))
            E._body(plan, w, sink, acc, sync_every=sync_every, noinline=noinline, prefetch=prefetch)
            w("    }\n")
        w("    if (live) {\n")
        if reduce_mode == "red":
            # JAMP[f] accumulated in place across the kernels of the stream: the first kernel (in launch order) that
            # touches a flow stores, the later ones add with fire-and-forget L2 reductions (red.global.add): no
            # partial slots, no gather pass, and still a fixed summation order (one add per kernel, stream order)
            w("      T* __restrict__ pb = part + (long long)ih * npart * 2 * stride + ievt;\n")
            for f in touched:
                for c_ in (0, 1):
                    if f in first_writer:
                        w("      pb[%d * stride] = sj[%d * BLK];\n" % (2 * f + c_, 2 * slot[f] + c_))
                    else:
                        w("      atomicAdd(pb + %d * stride, sj[%d * BLK]);\n" % (2 * f + c_, 2 * slot[f] + c_))
        else:
            w("      T* __restrict__ pb = part + ((long long)ih * npart + PBASE) * 2 * stride + ievt;\n")
            w("#pragma unroll\n      for (int q = 0; q < 2 * NTOUCH; ++q) pb[q * stride] = sj[q * BLK];\n")
        w("    }\n  }\n}\n")
        w("void launch_group%d(int prec, long long nevt, const int* hel_list, int hcount, int per_thread, int npart, void* part,\n"
          "                    const void* inv, long long stride, double mt, cudaStream_t st) {\n" % gi)
        w("  const dim3 grid((unsigned)((nevt + BLK - 1) / BLK), (unsigned)((hcount + per_thread - 1) / per_thread));\n")
        w("  static bool attr_set = false;\n  if (!attr_set) {\n")
        w("    cudaFuncSetAttribute(group%d_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (2 * NTOUCH + NSTAGE) * BLK * 8);\n" % gi)
        if fp32:
            w("    cudaFuncSetAttribute(group%d_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (2 * NTOUCH + NSTAGE) * BLK * 4);\n" % gi)
        w("    attr_set = true;\n  }\n")
        w("  if (prec == 0) group%d_kernel<double><<<grid, BLK, (2 * NTOUCH + NSTAGE) * BLK * 8, st>>>(nevt, hel_list, hcount, per_thread, npart, (double*)part, (const double*)inv, stride, mt);\n" % gi)
        if fp32:
            w("  else group%d_kernel<float><<<grid, BLK, (2 * NTOUCH + NSTAGE) * BLK * 4, st>>>(nevt, hel_list, hcount, per_thread, npart, (float*)part, (const float*)inv, stride, mt);\n" % gi)
        w("}\n}  // namespace\n")
        files.append(("%s_g%02d.cu" % (ns, gi), "".join(out)))
        ginfo.append(dict(terms=nterms, phases=[len(p.terms) for p in phases], max_live=live, flops=flops,
                          flows=len(touched), block=gblock, minblocks=gmin, smem64=smem64, staged=nstage,
                          inv_items=sum(union.sizes[k_] for k_ in probe.count)))
        base += len(touched)
    npart = base if reduce_mode != "red" else ncol
    assert all(part_of_flow[f] for f in range(ncol)), "every colour flow must be written by some group"
    files.append(_main_unit(E, n, ns, proc, npar, nhel, ncol, ndiag, cfi, cfden, union, inv, ninv, npart, part_of_flow,
                            nkern, total_flops, fp32, reduce_mode))
    colour_flops = 2 * (ncol * (ncol - 1) // 2) * 2 + ncol * 8
    info = dict(proc=proc, ns=ns, npar=npar, ncol=ncol, nhel=nhel, ndiagrams=ndiag, nterms=sum(len(p.terms) for p in plans),
                flops_per_helicity=total_flops + colour_flops, shape="split", ngroups=nkern, npart=npart, ninv=ninv,
                groups=ginfo)
    return files, info


class _AllExternals:
    """Stand-in plan for _externals(): every external wavefunction is used somewhere in a multi-phase kernel."""

    def __init__(self, n):
        self.n = n
        self.ops = [("x",) + tuple("e%d" % i for i in range(n))]


def _main_unit(E, n, ns, proc, npar, nhel, ncol, ndiag, cfi, cfden, union, inv, ninv, npart, part_of_flow, ngroups,
               group_flops, fp32, reduce_mode="slots"):
    colour_flops = 2 * (ncol * (ncol - 1) // 2) * 2 + ncol * 8
    denom = 4 * 64 * factorial(n - 2)
    rows = E._colour_rows(cfi, ncol)
    out = [E.HEADER % dict(proc=proc, n=n, ndiag=ndiag, nterms=0, ncol=ncol, nhel=nhel, flops=colour_flops, ns=ns, npar=npar,
                           what="invariants kernel, JAMP gather, colour sum (K6), helicity sum (K7), tile loop over the "
                                "%d diagram-group kernels" % ngroups)]
    w = out.append
    w("// symmetric colour form: me = sum_i J_i^* (CF_ii J_i + 2 sum_{j>i} CF_ij J_j) / %d ; rows blocked by 8\n" % cfden)
    tab = []
    for i0 in range(0, ncol, 8):
        for j in range(i0, ncol):
            for i in range(i0, i0 + 8):
                tab.append(rows[i][j] if i < ncol else 0)
    w("__device__ __align__(16) const double cf_table[%d] = {\n" % len(tab))
    for k_ in range(0, len(tab), 24):
        w("  " + ", ".join("%d." % v for v in tab[k_:k_ + 24]) + ",\n")
    w("};\n")
    import os
    if os.environ.get("MG_CF_CONST") == "1" and len(tab) * 8 <= 62 * 1024:
        # measured slower (261k vs 271k ME/s, gg->tt~ggg): the 61 KB table thrashes the constant cache; off
        w("__constant__ double cf_const[%d] = {\n" % len(tab))
        for k_ in range(0, len(tab), 24):
            w("  " + ", ".join("%d." % v for v in tab[k_:k_ + 24]) + ",\n")
        w("};\n#define MG_CF_CONST %s::cf_const\n" % ns)
    # dense table for the DMMA variant of the colour sum (CF integers; the denominator is folded into `norm`)
    w("__device__ __align__(16) const double cf_dense[%d] = {\n" % (ncol * ncol))
    for i in range(ncol):      # diagonal 8x8 blocks: CF; blocks above: 2 CF; blocks below: unused (0)
        w("  " + ", ".join("%d." % (cfi[i][j] if j // 8 == i // 8 else 2 * cfi[i][j] if j // 8 > i // 8 else 0)
                           for j in range(ncol)) + ",\n")
    w("};\n")
    w("}  // namespace\n#include \"mg_colour.cuh\"\nnamespace %s {\n" % ns)
    if ncol <= 32 and reduce_mode == "red":
        # small colour basis: all JAMPs of a (event, helicity) in registers, the symmetric form fully unrolled with the
        # integer coefficients as immediates — no table loads, every JAMP read once
        w("#define MG_HAVE_COLOUR_REG 1\n")
        w("template <class T>\n__global__ void __launch_bounds__(128) colour_reg_kernel(const T* __restrict__ jamp, T* __restrict__ meh,\n"
          "                                                                    long long stride, long long nevt) {\n")
        w("  const long long ievt = (long long)blockIdx.x * blockDim.x + threadIdx.x;\n  const int ih = blockIdx.y;\n")
        w("  if (ievt >= nevt) return;\n")
        w("  const T* __restrict__ jb = jamp + (long long)ih * (2 * NCOL) * stride + ievt;\n")
        for f in range(ncol):
            w("  const T jr%d = jb[%d * stride], ji%d = jb[%d * stride];\n" % (f, 2 * f, f, 2 * f + 1))
        w("  T me = T(0);\n")
        for i in range(ncol):
            zr = " + ".join("T(%d) * jr%d" % (rows[i][j], j) for j in range(i, ncol) if rows[i][j])
            zi = " + ".join("T(%d) * ji%d" % (rows[i][j], j) for j in range(i, ncol) if rows[i][j])
            w("  me += jr%d * (%s);\n  me += ji%d * (%s);\n" % (i, zr, i, zi))
        w("  meh[(long long)ih * stride + ievt] = me;\n}\n")
    # gather table (CSR): flow f <- partial slots part_idx[part_ptr[f] .. part_ptr[f+1])
    ptr, idx = [0], []
    for f in range(ncol):
        idx += part_of_flow[f]
        ptr.append(len(idx))
    w("constexpr int NPART = %d, NINV = %d;\n" % (npart, ninv))
    w("__device__ const short part_ptr[%d] = {%s};\n" % (len(ptr), ", ".join(map(str, ptr))))
    w("__device__ const short part_idx[%d] = {\n" % len(idx))
    for k_ in range(0, len(idx), 32):
        w("  " + ", ".join(map(str, idx[k_:k_ + 32])) + ",\n")
    w("};\n")
    for gi in range(ngroups):
        w("void launch_group%d(int prec, long long nevt, const int* hel_list, int hcount, int per_thread, int npart, void* part,\n"
          "                    const void* inv, long long stride, double mt, cudaStream_t st);\n" % gi)
    w("template <class T>\n__global__ void __launch_bounds__(128) invariants_kernel(const double* __restrict__ mom, long long nevt,\n"
      "                  T* __restrict__ invbuf, long long stride, double mt_d) {\n")
    w("  const long long ievt = (long long)blockIdx.x * blockDim.x + threadIdx.x;\n  if (ievt >= nevt) return;\n")
    E._prologue(union, w)
    w("  T* __restrict__ o = invbuf + ievt;\n")
    for name, i in sorted(inv.items(), key=lambda kv: kv[1]):
        if name[0] == "s":
            w("  o[%d * stride] = %s;\n" % (i, name))
        elif name.startswith("eg"):
            g = int(name[2:])
            w("  { W4<double> e; ext_gluon(kd[%d], +1, %s, e);   // lambda = +1: e.r = -R, e.i = I\n" % (g, "false" if g < 2 else "true"))
            w("    o[%d * stride] = T(-e.r[1]); o[%d * stride] = T(-e.r[2]); o[%d * stride] = T(-e.r[3]);\n" % (i, i + 1, i + 2))
            w("    o[%d * stride] = T(e.i[1]); o[%d * stride] = T(e.i[2]); }\n" % (i + 3, i + 4))
        elif name.startswith("v3_"):
            ma, mb = (int(x) for x in name[3:].split("_"))
            sgn = "dsg%d" % (ma | mb)
            for m in range(4):
                w("  o[%d * stride] = T(%s * (dm%d.c[%d] - dm%d.c[%d])); o[%d * stride] = T(%s * (2.0 * dm%d.c[%d] + dm%d.c[%d])); "
                  "o[%d * stride] = T(-%s * (2.0 * dm%d.c[%d] + dm%d.c[%d]));\n"
                  % (i + m, sgn, ma, m, mb, m, i + 4 + m, sgn, mb, m, ma, m, i + 8 + m, sgn, ma, m, mb, m))
        elif name.startswith("tl") or name.startswith("tr"):
            side, m_ = name[1], int(name[2:])
            sv, qv = "ds%s%d" % (side, m_), "dq%s%d" % (side, m_)
            w("  o[%d * stride] = T(%s * (%s.c[0] + %s.c[3])); o[%d * stride] = T(%s * (%s.c[0] - %s.c[3])); o[%d * stride] = T(%s * %s.c[1]); "
              "o[%d * stride] = T(%s * %s.c[2]); o[%d * stride] = T(%s * mt_d);\n"
              % (i, sv, qv, qv, i + 1, sv, qv, qv, i + 2, sv, qv, i + 3, sv, qv, i + 4, sv))
        elif name in ("ub", "vv"):
            fn, mom = ("ext_ubar", "ptd") if name == "ub" else ("ext_v", "ptbd")
            for hi, lam in ((0, "+1"), (8, "-1")):
                w("  { W4<double> q; %s(%s, mt_d, %s, q);\n" % (fn, mom, lam))
                w("    " + " ".join("o[%d * stride] = T(q.r[%d]); o[%d * stride] = T(q.i[%d]);"
                                    % (i + hi + 2 * m, m, i + hi + 2 * m + 1, m) for m in range(4)) + " }\n")
        else:
            w("  stp(o + %d * stride, stride, %s);\n" % (i, name))
    w("}\n")
    w("""
#ifndef MG_TILE_MAX
#define MG_TILE_MAX (1 << 20)
#endif
template <class T>
static int run(const double* mom, T* me_out, long long nevt, const int* hel_list, int nhel_run, T* perhel_out,
                const double* par, void* ws, size_t ws_bytes, cudaStream_t st, int prec) {
  double norm = 1.0;
  for (int i = 0; i < NGLU; ++i) norm *= par[0];          // par[0] = g_s^2, par[1] = mt
  norm /= (double)%(cfden)d * (double)%(denom)d;
  const size_t es = sizeof(T);
  const size_t per_eh = (size_t)(%(slots)s + 2 * NCOL + 1) * es;     // bytes per (event, helicity)
  const size_t per_e = (size_t)NINV * es;                            // bytes per event
  // Event tile E and helicity chunk H.  Prefer the whole batch in one tile (one launch per kernel covers many waves
  // of CTAs: with 2 CTAs of 128 threads per SM a 131072-event tile is 3.46 waves, i.e. the last wave is half empty)
  // and chunk the helicities if the workspace is too small; only shrink the tile when fewer than MINH helicities fit.
  const long long EMAX = (long long)MG_TILE_MAX;
  long long E = (nevt + 31) / 32 * 32;
  if (E > EMAX) E = EMAX;
  const long long MINH = nhel_run < 16 ? nhel_run : 16;
  while (E > 1024 && (size_t)E * (per_e + MINH * per_eh) > ws_bytes) E = (E / 2 + 1023) / 1024 * 1024;
  if ((size_t)E * (per_e + per_eh) > ws_bytes) return 0;            // mg_api.cu sizes the workspace; cannot happen
  int nlaunch = 0;
  long long H = (long long)((ws_bytes / (size_t)E - per_e) / per_eh);
  if (H > nhel_run) H = nhel_run;
  if (H < nhel_run) {                                               // equal chunks
    const long long nchunk = (nhel_run + H - 1) / H;
    H = (nhel_run + nchunk - 1) / nchunk;
  }
  const double* cft = nullptr; const short* pptr = nullptr; const short* pidx = nullptr;
  cudaGetSymbolAddress((void**)&cft, cf_table);
  const double* cfd = nullptr;
  cudaGetSymbolAddress((void**)&cfd, cf_dense);
  cudaGetSymbolAddress((void**)&pptr, part_ptr);
  cudaGetSymbolAddress((void**)&pidx, part_idx);
  T* part = (T*)ws;
  T* jsum = part + (size_t)H * %(slots)s * E;
  T* meh = jsum + (size_t)H * 2 * NCOL * E;
  T* inv = meh + (size_t)H * E;
  for (long long e0 = 0; e0 < nevt; e0 += E) {
    const long long ne = nevt - e0 < E ? nevt - e0 : E;
    const double* m0 = mom + e0 * NPAR * 4;       // tile starts on a page boundary
    invariants_kernel<T><<<(unsigned)((ne + 127) / 128), 128, 0, st>>>(m0, ne, inv, E, par[1]);
    ++nlaunch;
    for (int h0 = 0; h0 < nhel_run; h0 += (int)H) {
      const int hc = nhel_run - h0 < H ? nhel_run - h0 : (int)H;
      // helicities per thread: consecutive helicities of an event reuse its invariants from L1, so give each thread
      // as many as leaves >= ~3 waves of threads in flight, in equal shares
      long long slices = (148LL * 256 * 3 + ne - 1) / ne;
      if (slices > hc) slices = hc;
      if (slices < 1) slices = 1;
      while (hc %% slices) ++slices;          // equal shares
      const int per_thread = (int)(hc / slices);
%(calls)s
#ifdef MG_HAVE_COLOUR_REG
      colour_reg_kernel<T><<<dim3((unsigned)((ne + 127) / 128), (unsigned)hc), 128, 0, st>>>(part, meh, E, ne);
      mgc::helsum_kernel<T><<<(unsigned)((ne + 255) / 256), 256, 0, st>>>(meh, E, ne, hc, T(norm), me_out + e0,
          perhel_out ? perhel_out + (long long)h0 * nevt + e0 : (T*)nullptr, nevt, h0 == 0);
#else
      mgc::gather_colour_sum<T, NCOL>(cft, pptr, pidx, NPART, part, %(jsrc)s, meh, E, ne, hc, T(norm), me_out + e0,
                                      perhel_out ? perhel_out + (long long)h0 * nevt + e0 : (T*)nullptr, nevt, h0 == 0, %(gather)s, st, cfd);
#endif
      nlaunch += %(ngroups)d + %(extra)d;
    }
  }
  return nlaunch;
}
static int launch(int prec, const double* mom, void* me_out, long long nevt, const int* hel_list, int nhel_run,
                  void* perhel_out, const double* par, void* ws, size_t ws_bytes, cudaStream_t st) {
  if (prec == 0) return run<double>(mom, (double*)me_out, nevt, hel_list, nhel_run, (double*)perhel_out, par, ws, ws_bytes, st, prec);
%(run32)s
  return 0;
}
}  // namespace
extern const mg_procdesc_t mg_desc_%(tag)s = {"%(proc)s", %(npar)d, %(nfinal)d, %(ndiag)d, %(nhel)d, %(ncol)d, %(denom)d,
  %(flops)dLL, {0, 0, 1, 1%(gm)s}, %(ns)s::launch, {%(ws64)d, %(ws32)d}, %(nk)d, %(hasfp32)d, {%(wse64)d, %(wse32)d}, %(algo)dLL};
""" % dict(ngroups=ngroups, algo=Plan(n, acc_max=24).flops_per_helicity(externals=False), cfden=cfden, denom=denom, tag=ns[3:], proc=proc, npar=npar, nfinal=n, ndiag=ndiag, nhel=nhel, ncol=ncol,
           flops=group_flops + colour_flops, gm=", 0" * (n - 2), ns=ns,
           ws64=((0 if reduce_mode == "red" else 2 * npart) + 2 * ncol + 1) * 8,
           ws32=((0 if reduce_mode == "red" else 2 * npart) + 2 * ncol + 1) * 4,
           slots="0" if reduce_mode == "red" else "2 * NPART", jsrc="part" if reduce_mode == "red" else "jsum",
           gather="false" if reduce_mode == "red" else "true", extra=2 if reduce_mode == "red" else 3,
           nk=ngroups + (3 if reduce_mode == "red" else 4), hasfp32=1 if fp32 else 0, wse64=ninv * 8, wse32=ninv * 4,
           calls="\n".join("      launch_group%d(prec, ne, hel_list + h0, hc, per_thread, NPART, part, inv, E, par[1], st);" % gi
                           for gi in range(ngroups)),
           run32=("  return run<float>(mom, (float*)me_out, nevt, hel_list, nhel_run, (float*)perhel_out, par, ws, ws_bytes, st, prec);"
                  if fp32 else "")))
    return (ns + ".cu", "".join(out))
