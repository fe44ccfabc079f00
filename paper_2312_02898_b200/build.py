"""Build step: run the process generator (K0) and compile libmg5b200.so for sm_100a, in-tree.

    python -m paper_2312_02898_b200.build [--force]

Generated sources go to csrc/generated/ (git-ignored: they are a pure function of gen/); objects and the per-unit
`ptxas -v` logs to csrc/build/; the shared library next to this file.  Everything is compiled as relocatable device
code (-rdc=true): the diagram-group bodies of the event-CTA kernels are separate translation units linked into one
kernel.  nvcc cross-compiles without a GPU.  `python -m paper_2312_02898_b200.build --resources` prints the
registers / spill / stack table of the compiled units (from the ptxas logs).
"""
import hashlib
import os
import re
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
GEN = os.path.join(CSRC, "generated")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libmg5b200.so")
PEAK_LIB = os.path.join(HERE, "libmg5b200_peak.so")     # measurement helper for bench.py (csrc/peak), not the product
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-rdc=true", "-Xcompiler", "-fPIC", "-I", CSRC]
HAND = ("mg_api.cu", "mg_rambo.cu", "mg_reduce.cu", "mg_noalloc.cu")


def generate(overrides=None):
    """Runs the process generator; returns (list of generated .cu paths, list of info dicts).  `overrides`
    (tuning runs only): {n_gluons: dict of emit_coop keyword overrides}."""
    import json
    from .gen.emit import emit_eemumu, emit_ggttng
    from .gen.quark import SPECS, emit_quark
    from .gen.quark2 import SPECS as SPECS2, emit_quark2
    os.makedirs(GEN, exist_ok=True)
    infos, paths = [], []
    jobs = [emit_eemumu()]
    for n in (2, 3, 4, 5):
        kw = dict(fp32=(n < 5))
        kw.update((overrides or {}).get(n, {}))
        jobs.append(emit_ggttng(n, **kw))
    for spec in SPECS:                       # quark channels of p p -> t t~ + 0..2 jets
        jobs.append(emit_quark(spec))
    for spec in SPECS2:                      # ... with two light-quark lines (2 jets, no gluon)
        jobs.append(emit_quark2(spec))
    keep = set()
    for files, info in jobs:
        for fname, src in files:
            path = os.path.join(GEN, fname)
            old = open(path).read() if os.path.exists(path) else None
            if old != src:
                with open(path, "w") as fh:
                    fh.write(src)
            paths.append(path)
            keep.add(fname)
        infos.append(info)
    tags = [i["ns"][3:] for i in infos]
    reg = "// GENERATED: table of generated processes\n#include \"mg_kernel.cuh\"\n"
    reg += "".join("extern const mg_procdesc_t mg_desc_%s;\n" % t for t in tags)
    reg += "extern const mg_procdesc_t* const mg_registry[] = {%s};\n" % ", ".join("&mg_desc_" + t for t in tags)
    reg += "extern const int mg_registry_n = %d;\n" % len(tags)
    path = os.path.join(GEN, "mg_registry.cu")
    if not os.path.exists(path) or open(path).read() != reg:
        with open(path, "w") as fh:
            fh.write(reg)
    paths.append(path)
    keep.add("mg_registry.cu")
    for f in os.listdir(GEN):            # stale units of an earlier partition
        if f.endswith(".cu") and f not in keep:
            os.remove(os.path.join(GEN, f))
    with open(os.path.join(GEN, "generator_info.json"), "w") as fh:
        json.dump(infos, fh, indent=1, default=str)
    return paths, infos


def _stamp(path):
    h = hashlib.sha1()
    for p in [path] + [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cuh", ".h"))]:
        with open(p, "rb") as fh:
            h.update(fh.read())
    with open(os.path.join(HERE, "..", "include", "mg5b200.h"), "rb") as fh:
        h.update(fh.read())
    h.update(" ".join(ARCH + FLAGS).encode())
    return h.hexdigest()


def _compile(path, force, log):
    os.makedirs(OBJ, exist_ok=True)
    base = os.path.splitext(os.path.basename(path))[0]
    obj = os.path.join(OBJ, base + ".o")
    stamp_file = obj + ".stamp"
    stamp = _stamp(path)
    if not force and os.path.exists(obj) and os.path.exists(stamp_file) and open(stamp_file).read() == stamp:
        return obj
    extra = []
    with open(path) as fh:                      # per-unit flags requested by the generator ("// nvcc: ..." in the header)
        for line in fh.readlines()[:4]:
            if line.startswith("// nvcc:"):
                extra = line[len("// nvcc:"):].split()
    cmd = [NVCC] + ARCH + FLAGS + extra + ["-Xptxas", "-v", "-c", path, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(os.path.join(OBJ, base + ".ptxas.log"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s" % (path, r.stderr[-4000:]))
    with open(stamp_file, "w") as fh:
        fh.write(stamp)
    if log:
        print("compiled", base, flush=True)
    return obj


def build(force=False, log=True, overrides=None):
    gen_paths, infos = generate(overrides)
    hand = [os.path.join(CSRC, f) for f in HAND]
    srcs = sorted(gen_paths, key=lambda p: -os.path.getsize(p)) + hand    # largest first
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        objs = list(ex.map(lambda p: _compile(p, force, log), srcs))
    for f in os.listdir(OBJ):            # objects of units that no longer exist
        if f.endswith(".o") and os.path.join(OBJ, f) not in objs:
            for victim in (f, f + ".stamp", f[:-2] + ".ptxas.log"):
                if os.path.exists(os.path.join(OBJ, victim)):
                    os.remove(os.path.join(OBJ, victim))
    newest = max(os.path.getmtime(o) for o in objs)
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        cmd = [NVCC] + ARCH + ["-rdc=true", "-shared", "-o", LIB] + objs + ["-lcudart"]
        subprocess.check_call(cmd)
        if log:
            print("linked", LIB, flush=True)
    peak_src = os.path.join(CSRC, "peak", "mg_peak.cu")
    if force or not os.path.exists(PEAK_LIB) or os.path.getmtime(PEAK_LIB) < os.path.getmtime(peak_src):
        subprocess.check_call([NVCC] + ARCH + ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-shared", "-o", PEAK_LIB,
                                               peak_src, "-lcudart"])
    return LIB


def resources():
    """Registers / stack / spill per compiled entry or device function, parsed from the ptxas -v logs."""
    rows = []
    for f in sorted(os.listdir(OBJ)):
        if not f.endswith(".ptxas.log"):
            continue
        txt = open(os.path.join(OBJ, f)).read()
        for m in re.finditer(r"Compiling entry function '(\S+)'.*?\n(?:ptxas info\s*:.*\n)*?ptxas info\s*: Function properties for \S+\n"
                             r"\s*(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads\n"
                             r"ptxas info\s*: Used (\d+) registers", txt):
            rows.append((f[:-10], m.group(1), int(m.group(5)), int(m.group(2)), int(m.group(3)), int(m.group(4))))
        for m in re.finditer(r"Function properties for (\S+)\n\s*(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads", txt):
            rows.append((f[:-10], m.group(1), None, int(m.group(2)), int(m.group(3)), int(m.group(4))))
    return rows


if __name__ == "__main__":
    if "--resources" in sys.argv:
        for r in resources():
            print("%-22s %-60s regs=%s stack=%d spill_st=%d spill_ld=%d" % r)
    else:
        build(force="--force" in sys.argv)
