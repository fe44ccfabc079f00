"""GPU parity tests: the CUDA path, called through the C ABI (paper_2312_02898_b200 binding), against the
CPU oracle on identical seeded inputs (SURVEY.md §8c "parity protocol").

  * Philox words: bit-exact.   * RAMBO momenta: <= 1e-12 sqrt(s) per component (libm differs).
  * |M|^2 fp64: relative 1e-10 per event vs the long-double oracle on the GPU-generated momenta.
  * |M|^2 fp32: median 1e-5, max 1e-3 (north_star).
All tests need a CUDA device (-m gpu).
"""
import math

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

TOL64 = 1e-10           # north_star
TOL32_MED, TOL32_MAX = 1e-5, 1e-3


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
def test_rambo_matches_oracle_and_invariants(mg, oracle, name):
    cfg = workloads.CONFIGS[name]
    if not available(mg, name):
        pytest.skip("process not generated")
    proc = mg.Process(cfg["proc"])
    nevt = 4133                      # several pages + ragged tail
    mom, ev = gpu_events(mg, proc, cfg, nevt)
    ref = oracle.rambo(cfg["seed"], nevt, cfg["masses_final"], cfg["sqrt_s"])
    # libm log/sincos differ by an ulp between glibc and CUDA; RAMBO's conformal boost amplifies that by
    # (Q0/M)^2 for nearly collinear massless q's, so the bound is on quantiles, with a loose cap
    dev = np.abs(ev - ref).reshape(nevt, -1).max(axis=1) / cfg["sqrt_s"]
    assert np.median(dev) <= 1e-14 and np.quantile(dev, 0.99) <= 1e-12 and dev.max() <= 1e-9, (np.median(dev), dev.max())
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


@pytest.mark.parametrize("name", ["eemumu", "ggtt", "ggttg", "ggttgg", "ggttggg"])
def test_sigma_fp64_full_size_sampled(mg, oracle, oracle_ld, name):
    """BASELINE.json's full sizes, in the launch configuration bench.py times: sampled events are
    checked one by one against the oracle (plus the numerically hardest ones: smallest min s_ij)."""
    cfg = workloads.CONFIGS[name]
    if not available(mg, name):
        pytest.skip("process not generated")
    import torch
    nevt = cfg["nevt"]
    proc = mg.Process(cfg["proc"])
    mom, ev = gpu_events(mg, proc, cfg, nevt)
    me = proc.sigma(mom, nevt)
    torch.cuda.synchronize()
    me = me.cpu().numpy()
    assert np.all(np.isfinite(me)) and np.all(me > 0)
    nsamp = {"eemumu": 2048, "ggtt": 2048, "ggttg": 1024, "ggttgg": 256, "ggttggg": 12}[name]
    rng = np.random.default_rng(12345)
    idx = rng.choice(nevt, size=nsamp, replace=False)
    idx[:3] = [0, nevt - 1, nevt // 2]
    orc = oracle_ld
    ref = orc.me_batch(cfg["proc"], ev[idx])
    rel = np.abs(me[idx] / ref - 1)
    assert np.median(rel) < 1e-12 and rel.max() < TOL64, (rel.max(), np.median(rel))
    if name.startswith("ggttg"):
        # the numerically hardest events of the batch (smallest invariants: soft / collinear gluons).  Both sides
        # are given the same doubles, but near a soft or collinear pole |M|^2 is ill-conditioned in them: the fp64
        # result carries rounding amplified by ~ s / min s_ij (reading A12), so the bound is a
        # conditioning cap: median 1e-9, max 1e-8 over the hardest events of the batch.
        npar = ev.shape[1]
        smin = np.full(nevt, np.inf)
        for a in range(npar):
            for b in range(a + 1, npar):
                if a in (2, 3) and b in (2, 3):
                    continue
                d = ev[:, a, 0] * ev[:, b, 0] - (ev[:, a, 1:] * ev[:, b, 1:]).sum(-1)
                smin = np.minimum(smin, np.abs(d))
        hard = np.argsort(smin)[: max(4, nsamp // 8)]
        refh = orc.me_batch(cfg["proc"], ev[hard])
        relh = np.abs(me[hard] / refh - 1)
        assert relh.max() < 1e-8 and np.median(relh) < 1e-9, (relh.max(), np.median(relh))


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
    want = {"eemumu": (4, 4), "ggtt": (12, 6), "ggttg": (32, 16), "ggttgg": (64, 32), "ggttggg": (128, 64)}
    for name, (ngood, neval) in want.items():
        cfg = workloads.CONFIGS[name]
        proc = mg.Process(cfg["proc"])
        mom, ev = gpu_events(mg, proc, cfg, 4096)
        good = proc.helicity_probe(mom, 4096)
        assert len(good) == ngood == proc.info.ngoodhel
        # helicity-flip symmetry: QCD helicities pair up (evaluated once, counted twice); e+e- (Z exchange) does not
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
