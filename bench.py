#!/usr/bin/env python
"""bench.py — throughput of the hot path (matrix elements / second) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload ggttgg|ggttggg|...] [--impl reference]

A *step* is one pass of the whole hot path over one batch of synthetic input:
mg_rambo (device Philox + RAMBO) followed by mg_sigma on BASELINE.json's configuration (default: config 4,
g g > t t~ g g, 524288 events, sqrt(s) = 1500 GeV, seed 4, fp64 — the first process BASELINE.json's metric
is quoted on).  Prints ONE JSON line (contract in the task statement): `value` = ME/s with inputs resident
in HBM; `e2e` = the same through mg_sigma_host with pinned HOST buffers (H2D/D2H inside the timed region);
`roofline` = achieved FP64 FLOP/s of the sigma kernel(s) against the larger of the nominal DFMA peak and the FMA-loop
rate measured in the same run (libmg5b200_peak.so), bound "alu"; `cpu_baseline` = the CPU oracle timed on this box's host cores on a bounded
sample.  `--impl reference` times the oracle alone (it is the reference arm of this tier).
Under torchrun each rank takes its own shard of the Philox event stream (first_event = rank * nevt): weak
scaling, no data-path collective.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
import workloads  # noqa: E402

METRIC = "matrix elements/sec"
UNIT = "ME/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="ggttgg",
                    choices=list(workloads.CONFIGS) + ["quark_" + q for q in workloads.QUARK_SPECS + workloads.QUARK2_SPECS],
                    help="a BASELINE.json config, or quark_<spec>: one quark channel of p p > t t~ + jets (SURVEY 8f-3; not a "
                         "BASELINE.json config: reported for the record, no cpu_baseline leg)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--nevt", type=int, default=0, help="override the batch size (profiling runs only; not a bench value)")
    ap.add_argument("--single", action="store_true", help="only the named workload (no second process under 'also')")
    return ap.parse_args()


def config_dict(name, cfg, world, precision):
    where = "BASELINE.json configs[%d]" % cfg["index"] if cfg["index"] >= 0 else "not a BASELINE.json config"
    return {"workload": "%s: %s, sqrt_s=%g GeV, %d RAMBO events/GPU, Philox seed %d (%s)"
                        % (name, cfg["proc"], cfg["sqrt_s"], cfg["nevt"], cfg["seed"], where),
            "proc": cfg["proc"], "nevt_per_gpu": cfg["nevt"], "global_batch": cfg["nevt"] * world,
            "sqrt_s": cfg["sqrt_s"], "seed": cfg["seed"], "precision": precision,
            "parallelism": "events sharded over %d GPU(s), no collective" % world,
            "l2": "step rewrites the 100 MB momenta batch; 256 MB L2 flush between timed steps"}


# ---------------------------------------------------------------------------------------------- oracle legs
ORACLE_SAMPLE = {"eemumu": 524288, "ggtt": 262144, "ggttg": 131072, "ggttgg": 49152, "ggttggg": 4096}


def oracle_time(name, cfg, nsample, repeats=1):
    """Times the oracle as it stands (double build, OpenMP over events) on `nsample` events of the workload."""
    from oracle import oracle as O
    orc = O.load(False)
    cores = host_cores()
    mom = orc.rambo(cfg["seed"], nsample, cfg["masses_final"], cfg["sqrt_s"])
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        me = orc.me_batch(cfg["proc"], mom, nthreads=cores)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    assert (me > 0).all()
    return nsample / best, best, cores


def host_cores():
    """Threads the oracle legs run on: the cores this process may use (torchrun exports OMP_NUM_THREADS=1 for N > 1, which
    would otherwise make the oracle single-threaded)."""
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


def run_reference(args, name, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    nsample = max(8, ORACLE_SAMPLE[name] // 4)
    from oracle import oracle as O
    orc = O.load(False)
    mom = orc.rambo(cfg["seed"], nsample, cfg["masses_final"], cfg["sqrt_s"])
    cores = host_cores()
    for _ in range(min(args.warmup, 1)):
        orc.me_batch(cfg["proc"], mom[: max(8, nsample // 8)], nthreads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        mom = orc.rambo(cfg["seed"], nsample, cfg["masses_final"], cfg["sqrt_s"])
        orc.me_batch(cfg["proc"], mom, nthreads=cores)
    dt = time.perf_counter() - t0
    val = nsample * args.steps / dt
    sample = "%d events per step (prefix of the workload's seeded RAMBO batch), oracle RAMBO + |M|^2" % nsample
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(name, cfg, 1, "fp64"),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


def dram_traffic(name, precision):
    """DRAM bytes (read + write) moved by all kernels of one mg_sigma call at the full batch size, from the ncu capture
    summarised in profiles/r2_traffic.csv (columns: workload, precision, bytes_per_call, source); None if absent."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    if not os.path.exists(path):
        return None
    for line in open(path):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 4 and f[0] == name and f[1] == precision:
            return float(f[2]), f[3]
    return None


def measured_flops(name, precision):
    """FP64 FLOPs per event of one mg_sigma call as counted by ncu (dadd + dmul + 2 dfma + 512 per DMMA), and the
    generator's static counts, from profiles/r2_flops.csv (columns: workload, precision, measured_flops_per_event,
    static_executed_per_event, static_algorithmic_per_event, source); None if absent."""
    path = os.path.join(ROOT, "profiles", "r2_flops.csv")
    if not os.path.exists(path):
        return None
    for line in open(path):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 6 and f[0] == name and f[1] == precision:
            return dict(measured=float(f[2]), static_executed=float(f[3]), static_algorithmic=float(f[4]), source=f[5])
    return None


# per-event FLOPs of round 1's kernels (its generator's static algorithmic count, BENCH_r01.json / DESIGN.md §7):
# the same |M|^2 costs fewer FLOPs now (helicity-flip symmetry, helicity tables); "frac_r1_flop_model" rates today's
# ME/s with round 1's FLOPs per ME so that the two rounds' roofline fractions can be compared like for like
R1_FLOPS_PER_EVENT = {("ggttgg", "fp64"): 1760640.0, ("ggttggg", "fp64"): 33470976.0}


def measured_peaks(device):
    """DFMA / FFMA / DMMA rates of the device measured now with the helper library libmg5b200_peak.so (FLOP/s)."""
    import ctypes as C
    L = C.CDLL(os.path.join(ROOT, "paper_2312_02898_b200", "libmg5b200_peak.so"))
    out = {}
    v = C.c_double()
    for key, prec in (("dfma", 0), ("ffma", 1)):
        assert L.mgpeak_fma(device, prec, C.byref(v)) == 0
        out[key] = v.value
    assert L.mgpeak_dmma(device, C.byref(v)) == 0
    out["dmma"] = v.value
    return out


# ---------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------- main arm
NOMINAL_FP64 = 148 * 64 * 2 * 1.965e9        # B200: 148 SMs x 64 FP64 lanes x 2 (FMA) x 1.965 GHz = 37.2 TFLOP/s
NOMINAL_FP32 = 148 * 128 * 2 * 1.965e9


def measure(mg, torch, dist, name, cfg, args, steps, rank, world, local, peaks, with_clocks):
    """Times `steps` steps of workload `name` (after >= 3 warm-ups); returns the fields of the JSON line."""
    prec = mg.FP64 if args.precision == "fp64" else mg.FP32
    proc = mg.Process(cfg["proc"], precision=prec, device=local)
    nevt = cfg["nevt"]
    first, _ = mg.shard(nevt, rank, world)
    st = torch.cuda.current_stream()
    mom = proc.alloc_momenta(nevt)
    me = torch.empty(nevt, dtype=torch.float64 if prec == mg.FP64 else torch.float32, device=mom.device)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=mom.device)
    # set-up outside the timed region: helicity probe (K8)
    proc.rambo(cfg["seed"], cfg["sqrt_s"], nevt, first_event=first, out=mom)
    proc.helicity_probe(mom, min(nevt, 4096))

    def step(ev=None):
        if ev:
            ev[0].record(st)
        proc.rambo(cfg["seed"], cfg["sqrt_s"], nevt, first_event=first, out=mom, stream=st)
        if ev:
            ev[1].record(st)
        proc.sigma(mom, nevt, out=me, stream=st)
        if ev:
            ev[2].record(st)

    warm = max(args.warmup, 3)
    for _ in range(warm):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0 and with_clocks:
        sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    for k in range(steps):
        flush.fill_(k & 0xFF)             # L2 flush between timed steps (not timed)
        step(evs[k])
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    t_rambo = sum(e[0].elapsed_time(e[1]) for e in evs) * 1e-3
    t_sigma = sum(e[1].elapsed_time(e[2]) for e in evs) * 1e-3
    t_total = t_rambo + t_sigma

    # e2e: host buffers through the C ABI (mg_sigma_host): H2D of the momenta + D2H of |M|^2 in the timed region
    host_mom = torch.empty(mom.numel(), dtype=torch.float64).pin_memory()
    host_mom.copy_(mom)
    host_me = torch.empty(nevt, dtype=me.dtype).pin_memory()
    ne2e = max(3, min(steps, 5))
    proc.sigma_host(host_mom, nevt, out_host=host_me)
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(ne2e):
        proc.sigma_host(host_mom, nevt, out_host=host_me)      # synchronises internally
    t_e2e = (time.perf_counter() - t0) / ne2e
    clocks = sampler.stop() if (rank == 0 and with_clocks) else None
    assert torch.equal(host_me.cuda(), me), "host and device entry points disagree"

    if dist:
        t = torch.tensor([t_total, t_sigma, t_rambo, t_e2e], dtype=torch.float64, device=mom.device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        t_total, t_sigma, t_rambo, t_e2e = [float(x) for x in t]
    info = proc.info
    launches_per_step = int(info.launches_last_sigma) + 1            # the sigma kernels + the RAMBO kernel
    flops_call = float(info.flops_per_event_goodhel) * nevt          # generator's static (algorithmic) count, FMA = 2
    executed = float(info.flops_executed_per_event_goodhel) * nevt   # including diagram-group recomputation
    mf = None if args.nevt else measured_flops(name, args.precision)
    stale = mf is not None and abs(mf["static_algorithmic"] / float(info.flops_per_event_goodhel) - 1) > 0.02
    if mf is not None and not stale:                                  # ncu counters of this kernel set: the numerator
        flops_call = min(flops_call, mf["measured"] * nevt)
    achieved = flops_call * steps / t_sigma
    fp64 = prec == mg.FP64
    peak_meas = peaks["dfma" if fp64 else "ffma"]
    peak_nom = NOMINAL_FP64 if fp64 else NOMINAL_FP32
    peak = max(peak_meas, peak_nom)                                  # the larger of measured and nominal
    traffic = dram_traffic(name, args.precision)
    mom_bytes = host_mom.numel() * 8
    out = {
        "value": nevt * world * steps / t_total, "ms_per_step": t_total / steps * 1e3, "steps": steps, "warmup": warm,
        "config": config_dict(name, cfg, world, args.precision),
        "sigma_only": {"value": nevt * world * steps / t_sigma, "unit": UNIT, "ms": t_sigma / steps * 1e3},
        "rambo": {"ms": t_rambo / steps * 1e3, "bound": "hbm", "bytes_written": mom_bytes,
                  "achieved_gbs": mom_bytes * steps / t_rambo / 1e9},
        "e2e": {"value": nevt * world / t_e2e, "unit": UNIT, "h2d_bytes_per_step": mom_bytes,
                "d2h_bytes_per_step": host_me.numel() * host_me.element_size(), "ms": t_e2e * 1e3,
                "api": "mg_sigma_host (pinned host momenta in, |M|^2 out)"},
        "gpu_launches": launches_per_step * steps,
        "roofline": {"bound": "alu", "achieved": achieved / 1e12, "peak": peak / 1e12, "unit": "TFLOP/s",
                     "frac": achieved / peak,
                     "peak_measured_fma_loop": peak_meas / 1e12, "peak_nominal": peak_nom / 1e12,
                     "peak_dmma_measured": peaks["dmma"] / 1e12,
                     "peak_source": "max(nominal 148 SM x %d lanes x 2 x 1.965 GHz, %s loop measured in this run with "
                                    "libmg5b200_peak.so); MEASURED_PEAKS.json has no FP64/FP32 ALU entry"
                                    % (64 if fp64 else 128, "DFMA" if fp64 else "FFMA"),
                     "traffic": None if traffic is None or args.nevt else traffic[0],
                     "traffic_unit": "bytes per mg_sigma call (dram read + write, all its kernels)",
                     "traffic_source": None if traffic is None or args.nevt else traffic[1],
                     "algorithmic_bytes": nevt * (32 * info.npar + me.element_size()),
                     "kernel": "mg_sigma: all kernels of one call, timed together with CUDA events (%d launches)"
                               % int(info.launches_last_sigma),
                     "flops_per_event": flops_call / nevt, "flops_per_event_static_algorithmic": int(info.flops_per_event_goodhel),
                     "flops_per_event_ncu": None if mf is None else mf["measured"],
                     "flops_source": ("generator's static algorithmic count (mg_process_info)" if mf is None or stale else
                                      "min(static algorithmic count, ncu dadd+dmul+2*dfma+512*dmma per event from %s)" % mf["source"]),
                     "frac_r1_flop_model": (None if (name, args.precision) not in R1_FLOPS_PER_EVENT else
                                            R1_FLOPS_PER_EVENT[(name, args.precision)] * nevt * steps / t_sigma / peak),
                     "ngoodhel": int(info.ngoodhel),
                     "nhel_evaluated": int(info.nhel_evaluated),
                     "executed_tflops": executed * steps / t_sigma / 1e12,
                     "executed_frac": executed * steps / t_sigma / peak,
                     "executed_flops_per_event": int(info.flops_executed_per_event_goodhel),
                     "workspace_bytes": int(info.workspace_bytes)},
        "clocks": clocks,
    }
    proc.close()
    del mom, me, flush
    torch.cuda.empty_cache()
    return out


def main():
    args = parse()
    name = args.workload
    if name.startswith("quark_"):
        cfg = dict(workloads.QUARK_CHANNELS[name[6:]], nevt=524288, index=-1)
        args.single = args.no_cpu_baseline = True
        if args.impl == "reference":
            print(json.dumps({"impl": "reference", "unavailable": "the reference arm times the BASELINE.json configs only"}))
            return 0
    else:
        cfg = dict(workloads.CONFIGS[name])
    if args.nevt:
        cfg["nevt"] = args.nevt
    if args.impl == "reference":
        return run_reference(args, name, cfg)

    import torch
    import paper_2312_02898_b200 as mg
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = measured_peaks(local)
    res = measure(mg, torch, dist, name, cfg, args, args.steps, rank, world, local, peaks, True)
    also = {}
    if name == "ggttgg" and not args.nevt and not args.single:
        # BASELINE.json's metric is quoted on two processes: the second one, g g > t t~ g g g (configs[4]), is timed
        # in the same invocation and reported under "also"
        also["ggttggg"] = measure(mg, torch, dist, "ggttggg", dict(workloads.CONFIGS["ggttggg"]), args,
                                  max(3, min(args.steps, 5)), rank, world, local, peaks, True)
    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return 0
    line = {"metric": METRIC, "value": res.pop("value"), "unit": UNIT, "n_gpus": world, "steps": res.pop("steps"),
            "warmup": res.pop("warmup"), "ms_per_step": res.pop("ms_per_step"), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if args.precision == "fp64" else "f32", "data": "synthetic"}
    line.update(res)
    if also:
        line["also"] = also
    if not args.no_cpu_baseline and world == 1:                 # reported at N = 1 only
        ns = ORACLE_SAMPLE[name]
        v, dt, cores = oracle_time(name, cfg, ns)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
                                "sample": "first %d events of the workload's seeded RAMBO batch, |M|^2 only" % ns}
        for nm in also:
            ns2 = ORACLE_SAMPLE[nm]
            v2, dt2, cores2 = oracle_time(nm, workloads.CONFIGS[nm], ns2)
            also[nm]["cpu_baseline"] = {"value": v2, "unit": UNIT, "cores": cores2, "kind": "oracle", "seconds": dt2,
                                        "sample": "first %d events of the workload's seeded RAMBO batch, |M|^2 only" % ns2}
    print(json.dumps(line), flush=True)
    if dist:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
