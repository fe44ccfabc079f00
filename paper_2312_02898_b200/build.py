"""Build step: run the process generator (K0) and compile libmg5b200.so for sm_100a, in-tree.

    python -m paper_2312_02898_b200.build [--force]

Generated sources go to csrc/generated/ (git-ignored: they are a pure function of gen/); objects to
csrc/build/; the shared library next to this file.  nvcc cross-compiles without a GPU.
"""
import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
GEN = os.path.join(CSRC, "generated")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libmg5b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", CSRC] + os.environ.get("MG_NVCC_EXTRA", "").split()


def generate():
    """Runs the process generator; returns (list of generated .cu paths, list of info dicts)."""
    import json
    from .gen.emit import emit_eemumu, emit_ggttng
    os.makedirs(GEN, exist_ok=True)
    infos, paths = [], []
    ns_gluons = [int(x) for x in os.environ.get("MG_NGLUONS", "2,3,4,5").split(",") if x]
    shapes = dict(kv.split("=") for kv in os.environ.get("MG_SHAPES", "").split(",") if kv)   # e.g. "4=fused"
    maxterms = dict(kv.split("=") for kv in os.environ.get("MG_MAXTERMS", "").split(",") if kv)   # e.g. "4=40"
    block = dict(kv.split("=") for kv in os.environ.get("MG_BLOCK", "").split(",") if kv)
    jobs = [emit_eemumu()]
    for n in ns_gluons:
        kw = dict(fp32=(n < 5))
        if os.environ.get("MG_ACCMAX"):
            kw["acc_max"] = int(os.environ["MG_ACCMAX"])
        if str(n) in block:
            kw["block"] = int(block[str(n)])
        if str(n) in maxterms:
            kw["max_terms"] = int(maxterms[str(n)])
        if os.environ.get("MG_PREFETCH"):
            kw["prefetch"] = int(os.environ["MG_PREFETCH"])
        if os.environ.get("MG_REDUCE"):
            kw["reduce_mode"] = os.environ["MG_REDUCE"]
        if os.environ.get("MG_STAGEKB"):
            kw["stage_kb"] = int(os.environ["MG_STAGEKB"])
        if os.environ.get("MG_NOINLINE"):
            kw["noinline"] = os.environ["MG_NOINLINE"] == "1"
        if os.environ.get("MG_FLAT") and n >= 5:
            kw["flat_phase"] = int(os.environ["MG_FLAT"])
        if os.environ.get("MG_LIVEMAX"):
            kw["live_max"] = int(os.environ["MG_LIVEMAX"])
        if os.environ.get("MG_SYNC"):
            kw["sync_every"] = int(os.environ["MG_SYNC"])
        if os.environ.get("MG_MINBLOCKS"):
            kw["minblocks"] = int(os.environ["MG_MINBLOCKS"])
        jobs.append(emit_ggttng(n, shape=shapes.get(str(n)), **kw))
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
    cmd = [NVCC] + ARCH + FLAGS + ["-Xptxas", "-v", "-c", path, "-o", obj]
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


def build(force=False, log=True):
    gen_paths, infos = generate()
    hand = [os.path.join(CSRC, f) for f in ("mg_api.cu", "mg_rambo.cu", "mg_peak.cu")]
    srcs = sorted(gen_paths, key=lambda p: -os.path.getsize(p)) + hand    # largest first
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        objs = list(ex.map(lambda p: _compile(p, force, log), srcs))
    newest = max(os.path.getmtime(o) for o in objs)
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        cmd = [NVCC] + ARCH + ["-shared", "-o", LIB] + objs + ["-lcudart"]
        subprocess.check_call(cmd)
        if log:
            print("linked", LIB, flush=True)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv)
