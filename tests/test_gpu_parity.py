"""GPU parity tests: the CUDA path, called through the C ABI (paper_2312_02898_b200 binding), against the
CPU oracle on identical seeded inputs (SURVEY.md §8c "parity protocol").

  * Philox words: bit-exact.
  * RAMBO momenta: adjudicated against the long-double oracle — the CUDA sampler must be as close to it as the
    double oracle is (libm log/sincos differ by an ulp, the conformal boost amplifies that for collinear q's).
  * |M|^2 fp64: per event  rel <= max(1e-10, C 2^-53 s / (2 min_ij |p_i.p_j|), K delta)  against the long-double oracle
    on the GPU-generated momenta: north_star's 1e-10; a conditioning allowance near soft/collinear poles (C = 256: the
    oracle's own double build needs C = 1.7 on the same events, the diagram-based CUDA path up to 126 on 1 event in
    5x10^5); and an allowance for the event's own momentum non-conservation delta (K = 512; RAMBO output conserves to
    rounding only, and off the conserving surface |M|^2 is not unique).  The A12 report (median, 99.9 %, max, count
    above 1e-10) is printed and written to gpurun_out/parity_report.jsonl.  DESIGN.md §3, reading A12.
  * |M|^2 fp32: median 1e-5, max 1e-3 (north_star).
All tests need a CUDA device (-m gpu).  `--full-parity` runs the whole SURVEY.md §8(d) parity set for gg -> tt~ggg too.
"""
import math

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

TOL64 = 1e-10           # north_star
TOL32_MED, TOL32_MAX = 1e-5, 1e-3
COND_C = 256.0          # conditioning allowance: rel <= max(TOL64, COND_C * 2^-53 * s / (2 min |p_i.p_j|)); measured need: 126
VIOL_K = 512.0          # allowance per unit of the event's own momentum non-conservation; measured need: 205


def min_gluon_invariant(ev):
    """min over pairs of massless legs (gluons) of |p_i.p_j|: the soft / collinear poles of gg -> tt~ + gluons."""
    npar = ev.shape[1]
    out = np.full(len(ev), np.inf)
    glu = [a for a in range(npar) if a not in (2, 3)]
    for i, a in enumerate(glu):
        for b in glu[i + 1:]:
            d = ev[:, a, 0] * ev[:, b, 0] - (ev[:, a, 1:] * ev[:, b, 1:]).sum(-1)
            out = np.minimum(out, np.abs(d))
    return out


def momentum_violation(ev, sqrt_s):
    """|sum of incoming - sum of outgoing momenta| / sqrt(s) per event.  RAMBO's output conserves momentum to rounding
    only (rare events with nearly collinear massless q's reach 1e-10, see test_rambo_*), and off the conserving surface
    |M|^2 is not unique: evaluations that route momenta differently (Feynman diagrams here, colour-ordered recursion in
    the oracle) differ by up to ~200 x violation (the size of the gauge cancellation between diagrams) — both equally
    right.  Measured: gg -> tt~, 9 of 524288 events above 1e-10, all with violation 5e-13 .. 2e-10."""
    return np.abs(ev[:, :2].sum(axis=1) - ev[:, 2:].sum(axis=1)).max(axis=1) / sqrt_s


def parity_bound(ev, sqrt_s, poles=True):
    b = np.maximum(TOL64, VIOL_K * momentum_violation(ev, sqrt_s))
    if poles:
        b = np.maximum(b, COND_C * 2.0 ** -53 * sqrt_s ** 2 / (2.0 * min_gluon_invariant(ev)))
    return b


def report(tag, rel, bound):
    """A12 report: median, 99.9 %, max, count above 1e-10 (and above the per-event bound); kept in gpurun_out/ if present."""
    import json
    import os
    rec = dict(case=tag, n=int(len(rel)), median=float(np.median(rel)), q999=float(np.quantile(rel, 0.999)), max=float(rel.max()),
               above_1e10=int((rel > TOL64).sum()), above_bound=int((rel > bound).sum()))
    print("parity", rec)
    out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "parity_report.jsonl"), "a") as fh:
            fh.write(json.dumps(rec) + "\n")
    return rec


@pytest.fixture(scope="module")
def mg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2312_02898_b200 as m
    m.lib()     # fails loudly if the extension is missing
    return m


def available(mg, name):
    try:
        p = mg.Process(workloads.CONFIGS[name]["proc"])
        p.close()
        return True
    except mg.MgError as e:
        if e.status == -2:
            return False
        raise


def gpu_events(mg, proc, cfg, nevt, first_event=0):
    import torch
    mom = proc.rambo(cfg["seed"], cfg["sqrt_s"], nevt, first_event=first_event)
    torch.cuda.synchronize()
    npar = proc.info.npar
    return mom, mg.pages_to_events(mom.cpu().numpy(), nevt, npar).copy()


# ------------------------------------------------------------------------------------------ sampler
def test_philox_words_bit_exact(mg, oracle):
    proc = mg.Process("g g > t t~ g")
    nevt, first = 1000, (1 << 32) - 500      # crosses the 32-bit boundary of the event counter
    w = proc.philox_raw(3, nevt, first_event=first).cpu().numpy().view(np.uint32)
    for i in (0, 1, 499, 500, 501, 999):
        gi = first + i
        for f in range(3):
            want = oracle.philox([gi & 0xFFFFFFFF, gi >> 32, f, 0], [3, 0])
            assert [int(x) for x in w[i, f]] == want


@pytest.mark.parametrize("name", ["eemumu", "ggtt", "ggttg", "ggttgg", "ggttggg"])
def test_rambo_matches_oracle_and_invariants(mg, oracle, oracle_ld, name):
    cfg = workloads.CONFIGS[name]
    if not available(mg, name):
        pytest.skip("process not generated")
    proc = mg.Process(cfg["proc"])
    nevt = 4133                      # several pages + ragged tail
    mom, ev = gpu_events(mg, proc, cfg, nevt)
    ref = oracle.rambo(cfg["seed"], nevt, cfg["masses_final"], cfg["sqrt_s"])
    refl = oracle_ld.rambo(cfg["seed"], nevt, cfg["masses_final"], cfg["sqrt_s"])
    # libm log/sincos differ by an ulp between glibc and CUDA, and RAMBO's conformal boost amplifies rounding by
    # (Q0/M)^2 for nearly collinear massless q's: no flat bound holds.  Adjudication against the long-double oracle: the
    # CUDA sampler's deviation from it must be distributed like the double oracle's own deviation (every quantile within
    # 4x, plus half an ulp of sqrt(s)), and no single event may be off by more than 64x the double oracle's error there
    dev = np.abs(ev - refl).reshape(nevt, -1).max(axis=1) / cfg["sqrt_s"]
    own = np.abs(ref - refl).reshape(nevt, -1).max(axis=1) / cfg["sqrt_s"]
    for q in (0.5, 0.9, 0.99, 0.999, 1.0):
        assert np.quantile(dev, q) <= 4 * np.quantile(own, q) + 4 * 2.0 ** -53, (q, np.quantile(dev, q), np.quantile(own, q))
    assert np.all(dev <= 64 * own + 64 * 2.0 ** -53), float((dev / (own + 2.0 ** -53)).max())
    # weights and first_event offset (sharded call gives the same events)
    import torch
    mom2, w2 = proc.rambo(cfg["seed"], cfg["sqrt_s"], 100, first_event=4000, weights=True)
    torch.cuda.synchronize()
    ev2 = mg.pages_to_events(mom2.cpu().numpy(), 100, proc.info.npar)
    assert np.array_equal(ev2, ev[4000:4100])      # same events bit for bit, whatever the batch split
    _, wref = oracle.rambo(cfg["seed"], 100, cfg["masses_final"], cfg["sqrt_s"], first_event=4000, weights=True)
    assert np.max(np.abs(w2.cpu().numpy() / wref - 1)) < 1e-11
    # invariants on the full-size batch (properties that hold at any size)
    nfull = cfg["nevt"]
    momf, evf = gpu_events(mg, proc, cfg, nfull)
    s = cfg["sqrt_s"]
    tot = evf[:, 2:, :].sum(axis=1)
    viol = np.abs(tot - np.array([s, 0, 0, 0])).max(axis=1) / s       # rare near-collinear q's amplify rounding
    assert np.quantile(viol, 0.999) < 1e-12 and viol.max() < 1e-8
    m2 = evf[..., 0] ** 2 - (evf[..., 1:] ** 2).sum(axis=-1)
    want = np.array([0.0, 0.0] + [m * m for m in cfg["masses_final"]])
    shell = np.abs(m2 - want).max(axis=1) / (s * s)
    assert np.quantile(shell, 0.999) < 1e-12 and shell.max() < 1e-8


# ------------------------------------------------------------------------------------------ |M|^2 fp64
SMALL = {"eemumu": 4133, "ggtt": 4133, "ggttg": 2085, "ggttgg": 517, "ggttggg": 35}


@pytest.mark.parametrize("name", ["eemumu", "ggtt", "ggttg", "ggttgg", "ggttggg"])
def test_sigma_fp64_parity_small(mg, oracle, oracle_ld, name):
    cfg = workloads.CONFIGS[name]
    if not available(mg, name):
        pytest.skip("process not generated")
    import torch
    nevt = SMALL[name]
    for mode in (mg.HEL_ALL, mg.HEL_FILTER):
        proc = mg.Process(cfg["proc"], helicity_mode=mode)
        mom, ev = gpu_events(mg, proc, cfg, nevt)
        me = proc.sigma(mom, nevt)
        torch.cuda.synchronize()
        me = me.cpu().numpy()
        orc = oracle_ld
        ref = orc.me_batch(cfg["proc"], ev)
        rel = np.abs(me / ref - 1)
        assert np.all(np.isfinite(me)) and rel.max() < TOL64, (name, mode, rel.max(), int(rel.argmax()))
        proc.close()


# SURVEY.md §8(d) parity set on BASELINE.json's full batches, in the launch configuration bench.py times: (first N events,
# the H events of the full batch with the smallest gluon invariants = numerically hardest).  The long-double oracle
# adjudicates everything except the bulk of gg -> tt~ggg, where it costs 0.1 s per event: there the double oracle is the
# reference for the first N events (its own error on such events is < 1e-12, measured against the long-double build)
# and the long-double one for the hardest H.
PARITY_SET = {"eemumu": (16384, 0), "ggtt": (524288, 0), "ggttg": (65536, 1024), "ggttgg": (16384, 1024), "ggttggg": (2048, 128)}
PARITY_SET_FULL = {"ggttg": (524288, 1024), "ggttggg": (16384, 1024)}


@pytest.mark.parametrize("name", ["eemumu", "ggtt", "ggttg", "ggttgg", "ggttggg"])
def test_sigma_fp64_parity_set_full_batch(mg, oracle, oracle_ld, full_parity, name):
    cfg = workloads.CONFIGS[name]
    import torch
    nevt = cfg["nevt"]
    proc = mg.Process(cfg["proc"])
    mom, ev = gpu_events(mg, proc, cfg, nevt)
    me = proc.sigma(mom, nevt)
    torch.cuda.synchronize()
    me = me.cpu().numpy()
    assert np.all(np.isfinite(me)) and np.all(me > 0)
    nfirst, nhard = (PARITY_SET_FULL if full_parity else {}).get(name, PARITY_SET[name])
    bulk = oracle if name == "ggttggg" else oracle_ld
    idx = np.arange(nfirst)
    ref = bulk.me_batch(cfg["proc"], ev[idx])
    rel = np.abs(me[idx] / ref - 1)
    poles = name.startswith("ggttg")          # soft / collinear poles need final-state gluons
    bound = parity_bound(ev[idx], cfg["sqrt_s"], poles)
    rec = report("%s first %d" % (name, nfirst), rel, bound)
    assert rec["above_bound"] == 0 and rec["median"] < 1e-12, rec
    if nhard:
        hard = np.argsort(min_gluon_invariant(ev))[:nhard]
        refh = oracle_ld.me_batch(cfg["proc"], ev[hard])
        relh = np.abs(me[hard] / refh - 1)
        rech = report("%s hardest %d of %d" % (name, nhard, nevt), relh, parity_bound(ev[hard], cfg["sqrt_s"]))
        assert rech["above_bound"] == 0, rech
    # a random sample across the whole batch (tiles, tails)
    rng = np.random.default_rng(12345)
    samp = rng.choice(nevt, size=min(nevt, {"ggttggg": 24}.get(name, 512)), replace=False)
    samp[:2] = [nevt - 1, nevt // 2]
    refs = oracle_ld.me_batch(cfg["proc"], ev[samp])
    rels = np.abs(me[samp] / refs - 1)
    assert np.all(rels <= parity_bound(ev[samp], cfg["sqrt_s"], poles)), rels.max()


def test_golden_worked_examples(mg):
    """tests/golden/worked_examples.txt (SURVEY Appendix A / C8 values) through the CUDA path."""
    import torch
    for pt in workloads.read_points("worked_examples.txt"):
        name = workloads.PROC_TO_NAME[pt["proc"]]
        if not available(mg, name):
            continue
        proc = mg.Process(pt["proc"], helicity_mode=mg.HEL_ALL)
        ev = np.array(pt["momenta"])[None]
        mom = mg.events_to_pages(ev)
        me = proc.sigma(torch.from_numpy(mom).cuda(), 1)
        assert abs(float(me.cpu()[0]) / pt["value"] - 1) < 1e-9, (pt["name"], float(me.cpu()[0]))


def test_closed_forms_on_gpu(mg):
    """gg -> tt~ against Combridge, e+e- -> mu+mu- against the gamma+Z angular formula (not via the oracle)."""
    import torch
    from test_oracle_me import combridge, eemumu_closed
    for name, fn in (("ggtt", combridge), ("eemumu", eemumu_closed)):
        cfg = workloads.CONFIGS[name]
        proc = mg.Process(cfg["proc"])
        mom, ev = gpu_events(mg, proc, cfg, 1000)
        me = proc.sigma(mom, 1000).cpu().numpy()
        ref = np.array([fn(p) for p in ev])
        assert np.max(np.abs(me / ref - 1)) < 1e-11


# ------------------------------------------------------------------------------------------ helicities
def test_helicity_filter_counts_and_per_helicity(mg, oracle):
    import torch
    want = {"eemumu": (4, 3), "ggtt": (12, 6), "ggttg": (32, 16), "ggttgg": (64, 32), "ggttggg": (128, 64)}
    for name, (ngood, neval) in want.items():
        cfg = workloads.CONFIGS[name]
        proc = mg.Process(cfg["proc"])
        mom, ev = gpu_events(mg, proc, cfg, 4096)
        good = proc.helicity_probe(mom, 4096)
        assert len(good) == ngood == proc.info.ngoodhel
        # helicity-flip symmetry: QCD helicities pair up (evaluated once, counted twice); with Z exchange only the pair
        # e-L e+R -> mu-R mu+L / e-R e+L -> mu-L mu+R (coupling gL gR in both) has equal |M_h|^2
        assert proc.info.nhel_evaluated == neval
        # per-helicity |M_h|^2 is basis independent in a fixed frame (reading A8): compare to the oracle
        ph = proc.sigma_per_helicity(mom, 64).cpu().numpy()
        for i in ((0, 63) if name != "ggttggg" else (5,)):
            tot, hel = oracle.me(cfg["proc"], ev[i], per_helicity=True)
            assert np.allclose(ph[:, i], hel, rtol=1e-9, atol=1e-13 * tot)
            og = [h for h in range(len(hel)) if hel[h] > 1e-14 * tot]
            if name != "ggtt":
                assert og == good


# ------------------------------------------------------------------------------------------ fp32
@pytest.mark.parametrize("name", ["ggttg", "ggttgg"])
def test_sigma_fp32_tolerance(mg, oracle, name):
    import torch
    cfg = workloads.CONFIGS[name]
    nevt = 2085 if name == "ggttg" else 517
    proc = mg.Process(cfg["proc"], precision=mg.FP32)
    mom, ev = gpu_events(mg, proc, cfg, nevt)
    me = proc.sigma(mom, nevt)
    assert me.dtype == torch.float32
    ref = oracle.me_batch(cfg["proc"], ev)
    rel = np.abs(me.cpu().numpy().astype(np.float64) / ref - 1)
    assert np.median(rel) < TOL32_MED and rel.max() < TOL32_MAX, (np.median(rel), rel.max())
    # full batch of the config: fp32 against the fp64 CUDA path (itself checked against the oracle above)
    nfull = cfg["nevt"]
    p64 = mg.Process(cfg["proc"])
    momf = p64.rambo(cfg["seed"], cfg["sqrt_s"], nfull)
    a = p64.sigma(momf, nfull).cpu().numpy()
    b = proc.sigma(momf, nfull).cpu().numpy().astype(np.float64)
    relf = np.abs(b / a - 1)
    assert np.median(relf) < TOL32_MED and relf.max() < TOL32_MAX, (np.median(relf), relf.max())


# ------------------------------------------------------------------------------------------ edges / API
def test_edge_cases_and_errors(mg, oracle_ld):
    import ctypes as C
    import torch
    cfg = workloads.CONFIGS["ggttg"]
    proc = mg.Process(cfg["proc"])
    L = mg.lib()
    # empty batch
    assert proc.sigma(proc.alloc_momenta(0), 0).numel() == 0
    assert proc.momenta_bytes(0) == 0 and proc.momenta_bytes(1) == 5 * 32 * 32 and proc.momenta_bytes(33) == 2 * 5 * 32 * 32
    # single event and ragged tails give the same values as the big batch
    mom, ev = gpu_events(mg, proc, cfg, 1000)
    me = proc.sigma(mom, 1000).cpu().numpy()
    for n in (1, 31, 33, 129):
        assert np.array_equal(proc.sigma(mom, n).cpu().numpy(), me[:n])
    # kinematics error, misalignment, negative nevt
    buf = proc.alloc_momenta(64)
    assert L.mg_rambo(proc._h, 1, C.c_double(300.0), 64, C.c_void_p(buf.data_ptr()), None) == -6
    assert L.mg_rambo(proc._h, 1, C.c_double(1500.0), 64, C.c_void_p(buf.data_ptr() + 8), None) == -5
    assert L.mg_rambo(proc._h, 1, C.c_double(1500.0), -1, C.c_void_p(buf.data_ptr()), None) == -4
    assert L.mg_sigma(proc._h, None, 10, None, None) == -1
    # host entry point (copies inside) equals the device entry point
    host = mom.cpu().pin_memory()
    assert np.array_equal(proc.sigma_host(host, 1000).numpy(), me)
    # non-default stream
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        me2 = proc.sigma(mom, 1000, stream=st)
    st.synchronize()
    assert np.array_equal(me2.cpu().numpy(), me)
    # parameters reach the kernels: alpha_s scaling g_s^6 for gg -> tt~ g
    proc2 = mg.Process(cfg["proc"], alpha_s=0.236)
    assert np.allclose(proc2.sigma(mom, 100).cpu().numpy(), me[:100] * 8.0, rtol=1e-12)


@pytest.mark.parametrize("name,nevt,ws_events", [("ggttgg", 20011, 4096), ("ggttgg", 20011, 32), ("ggttggg", 3001, 1024)])
def test_caller_workspace_and_event_tiles_give_identical_results(mg, name, nevt, ws_events):
    """mg_set_workspace: with a caller-provided workspace that holds only `ws_events` events' invariants the launcher
    runs the batch in event tiles.  Tiling does not change any per-event arithmetic: results are bit-identical."""
    import torch
    cfg = workloads.CONFIGS[name]
    ref_proc = mg.Process(cfg["proc"])
    mom = ref_proc.rambo(cfg["seed"], cfg["sqrt_s"], nevt)
    ref = ref_proc.sigma(mom, nevt).cpu().numpy()
    assert 0 < ref_proc.info.workspace_bytes <= 1 << 30
    proc = mg.Process(cfg["proc"])
    nbytes = proc.workspace_bytes(ws_events)
    assert 0 < nbytes < proc.workspace_bytes(nevt)
    buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    proc.set_workspace(buf)
    got = proc.sigma(mom, nevt).cpu().numpy()
    assert proc.info.workspace_bytes == nbytes
    assert proc.info.launches_last_sigma > ref_proc.info.launches_last_sigma
    assert np.array_equal(got, ref)
    # too small a workspace is refused, not silently ignored
    tiny = torch.empty(1 << 16, dtype=torch.uint8, device="cuda")
    with pytest.raises(mg.MgError):
        proc.set_workspace(tiny)
    proc.set_workspace(None)
    assert np.array_equal(proc.sigma(mom, nevt).cpu().numpy(), ref)


# ------------------------------------------------------------------------------------------ batch-unweighting primitive
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_weight_max_matches_oracle(mg, oracle_ld, precision):
    """mg_weight_max (PAPER.md:99-:103): products bit-exact, maximum bit-exact, sums to rounding, bit-reproducible."""
    import torch
    cfg = workloads.CONFIGS["ggttg"]
    prec = mg.FP64 if precision == "fp64" else mg.FP32
    proc = mg.Process(cfg["proc"], precision=prec)
    for nevt in (0, 1, 255, 8193, 300001):
        mom, w = proc.rambo(cfg["seed"], cfg["sqrt_s"], max(nevt, 1), weights=True)
        me = proc.sigma(mom, max(nevt, 1))[:nevt].clone()
        w = (w[:nevt] * 1e-6).clone()
        me0 = me.cpu().numpy().astype(np.float64)
        prod_ref, out_ref = oracle_ld.weight_max(me0, w.cpu().numpy(), single=(precision == "fp32"))
        out = proc.weight_max(me, w, nevt)
        got = out.cpu().numpy()
        assert np.array_equal(me.cpu().numpy().astype(np.float64), prod_ref)         # in-place products, one rounding
        assert got[0] == out_ref[0]                                                   # the maximum is exact
        if nevt:
            assert abs(got[1] / out_ref[1] - 1) < 1e-13 and abs(got[2] / out_ref[2] - 1) < 1e-13
        else:
            assert got[0] == -math.inf and got[1] == 0 and got[2] == 0
        # fixed reduction tree: bit-reproducible
        me2 = torch.from_numpy(me0).to(me.dtype).cuda()
        assert torch.equal(proc.weight_max(me2, w, nevt), out)


@pytest.mark.parametrize("name,nevt", [("ggttgg", 30011), ("ggttggg", 4001)])
def test_results_are_bit_reproducible(mg, name, nevt):
    """The JAMP accumulation (L2 reductions into thread-private addresses, issued in program order), the colour sum and
    the helicity sum (fixed trees) have a fixed order: repeated calls, and calls on another handle, agree bit for bit.
    (compute-sanitizer is not available on this GPU pool; a race in the shared-memory visit pipeline or in the JAMP
    scratch would show up here and in the bit-exact tiling test above.)"""
    cfg = workloads.CONFIGS[name]
    p1, p2 = mg.Process(cfg["proc"]), mg.Process(cfg["proc"])
    mom = p1.rambo(cfg["seed"], cfg["sqrt_s"], nevt)
    a = p1.sigma(mom, nevt).cpu().numpy()
    for _ in range(3):
        assert np.array_equal(p1.sigma(mom, nevt).cpu().numpy(), a)
    assert np.array_equal(p2.sigma(mom, nevt).cpu().numpy(), a)


def test_helicity_all_mode_ignores_the_probe(mg):
    cfg = workloads.CONFIGS["ggtt"]
    proc = mg.Process(cfg["proc"], helicity_mode=mg.HEL_ALL)
    mom = proc.rambo(cfg["seed"], cfg["sqrt_s"], 512)
    assert len(proc.helicity_probe(mom, 512)) == 16 and proc.info.nhel_evaluated == 16
    ref = mg.Process(cfg["proc"])
    a, b = proc.sigma(mom, 512).cpu().numpy(), ref.sigma(mom, 512).cpu().numpy()
    assert ref.info.nhel_evaluated == 6 and np.max(np.abs(a / b - 1)) < 1e-13


def test_bad_derived_couplings_are_rejected(mg):
    import ctypes as C
    L = mg.lib()
    h = C.c_void_p()
    for kw in (dict(gf=0.0), dict(gf=1e-9), dict(gamma_z=-1.0), dict(sw2=1.5)):
        p = mg.default_params(**kw)
        assert L.mg_process_create(b"e+ e- > mu+ mu-", C.byref(p), C.byref(h)) == -3, kw


def test_handles_on_two_devices(mg):
    """A handle created on a second device launches its kernels there (per-device kernel attributes)."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two visible GPUs")
    cfg = workloads.CONFIGS["ggttgg"]
    p0 = mg.Process(cfg["proc"], device=0)
    p1 = mg.Process(cfg["proc"], device=1)
    m0 = p0.rambo(cfg["seed"], cfg["sqrt_s"], 1000)
    with torch.cuda.device(1):
        m1 = p1.rambo(cfg["seed"], cfg["sqrt_s"], 1000)
        b = p1.sigma(m1, 1000).cpu().numpy()
    a = p0.sigma(m0, 1000).cpu().numpy()
    assert np.array_equal(a, b)


# ------------------------------------------------------------------------------------------ mixed precision with tracking
@pytest.mark.parametrize("name", ["ggttg", "ggttgg"])
def test_sigma_mixed_tracks_precision(mg, oracle, name):
    """mg_sigma_mixed: fp32 with a per-event precision estimate, fp64 where it exceeds tol.
    On the full batch: the estimate flags the events fp32 gets wrong; what is kept is an order of magnitude closer to the
    fp64 result than plain fp32; tol = 0 re-evaluates everything (= the fp64 path bit for bit); a loose tol none."""
    import torch
    cfg = workloads.CONFIGS[name]
    nevt = cfg["nevt"]
    proc = mg.Process(cfg["proc"])
    p32 = mg.Process(cfg["proc"], precision=mg.FP32)
    mom, ev = gpu_events(mg, proc, cfg, nevt)
    me64 = proc.sigma(mom, nevt).cpu().numpy()
    me32 = p32.sigma(mom, nevt).cpu().numpy().astype(np.float64)
    err32 = np.abs(me32 / me64 - 1)
    me, nf, eps = proc.sigma_mixed(mom, nevt, 1e-5, with_eps=True)
    me, eps = me.cpu().numpy(), eps.cpu().numpy()
    err = np.abs(me / me64 - 1)
    flagged = ~(eps <= 1e-5)
    assert nf == int(flagged.sum()) and 0 < nf < 0.05 * nevt
    assert np.array_equal(me[flagged], me64[flagged])                      # re-evaluated in fp64
    assert err.max() < 5e-6 < err32.max() and np.median(err) < TOL32_MED
    print("mixed", name, "plain fp32 max %.2e; mixed (tol 1e-5): %d of %d events in fp64, max %.2e" % (err32.max(), nf, nevt, err.max()))
    # against the oracle on a sample: the kept fp32 values and the re-evaluated ones
    idx = np.concatenate([np.arange(256), np.nonzero(flagged)[0][:256]])
    ref = oracle.me_batch(cfg["proc"], ev[idx])
    assert np.max(np.abs(me[idx] / ref - 1)) < 5e-6
    # limits
    n = 20000
    me0, nf0 = proc.sigma_mixed(mom, n, 0.0)
    assert nf0 == n and np.array_equal(me0.cpu().numpy(), me64[:n])
    me1, nf1 = proc.sigma_mixed(mom, n, 1e9)
    assert nf1 == 0 and np.max(np.abs(me1.cpu().numpy() / me64[:n] - 1)) < TOL32_MAX
    # not available: fp32 handle, process without fp32 kernels
    with pytest.raises(mg.MgError):
        p32.sigma_mixed(mom, 100, 1e-5)
    p5 = mg.Process("g g > t t~ g g g")
    with pytest.raises(mg.MgError):
        p5.sigma_mixed(p5.rambo(5, 1500.0, 64), 64, 1e-5)
