"""GPU parity of the quark channels of p p -> t t~ + 0..2 jets: the generated fused
kernels (gen/quark.py), called through the C ABI, against the colour-dressed oracle (oracle/me_qchannel.c) on the
momenta the CUDA RAMBO generated.  Same bound as the gluon channels (tests/test_gpu_parity.py, reading A12).
"""
import numpy as np
import pytest

import workloads
from test_gpu_parity import TOL32_MAX, TOL32_MED, gpu_events, parity_bound, report

pytestmark = pytest.mark.gpu

# events per subprocess: the oracle costs ~2 ms (0 jets), 0.1 s (1 jet), 5 s (2 jets) per event and core
NEVT = {4: 4133, 5: 1029, 6: 37}
NEVT2 = 261                      # two light lines, no gluon: 0.25 - 0.5 s per event


@pytest.fixture(scope="module")
def mg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2312_02898_b200 as m
    m.lib()
    return m


@pytest.mark.parametrize("spec", workloads.QUARK_SPECS + workloads.QUARK2_SPECS)
def test_quark_channel_fp64_parity(mg, oracle, oracle_ld, spec):
    import torch
    cfg = workloads.QUARK_CHANNELS[spec]
    nevt = NEVT2 if spec in workloads.QUARK2_SPECS else NEVT[len(spec)]
    ref = None
    for mode in (mg.HEL_ALL, mg.HEL_FILTER):
        proc = mg.Process(cfg["proc"], helicity_mode=mode)
        assert proc.info.npar == len(spec)
        mom, ev = gpu_events(mg, proc, cfg, nevt)
        me = proc.sigma(mom, nevt)
        torch.cuda.synchronize()
        me = me.cpu().numpy()
        if ref is None:
            orc = oracle_ld if len(spec) < 6 else oracle          # the long-double build is 4x slower: 2-jet events use double
            ref = orc.me_qchannel_batch(spec, ev)
        rel = np.abs(me / ref - 1)
        bound = parity_bound(ev, cfg["sqrt_s"])
        rec = report("quark %s mode %d" % (spec, mode), rel, bound)
        assert np.all(np.isfinite(me)) and np.all(me > 0)
        assert rec["above_bound"] == 0, (spec, mode, rel.max(), int(rel.argmax()))
        assert rec["median"] < 1e-12
        proc.close()


@pytest.mark.parametrize("spec", ["qQtTg", "gQtTQ", "qgtTqg", "qrtTqr", "qQtTqQ"])
def test_quark_channel_per_helicity_and_filter(mg, oracle, spec):
    """Per-helicity |M_h|^2 against the oracle's, and the helicity bookkeeping: chirality conservation along the massless
    line halves the good helicities, the helicity-flip symmetry halves the evaluated ones again."""
    import torch
    cfg = workloads.QUARK_CHANNELS[spec]
    nevt = 8 if len(spec) == 6 else 64
    proc = mg.Process(cfg["proc"])
    mom, ev = gpu_events(mg, proc, cfg, nevt)
    proc.helicity_probe(mom, nevt)
    info = proc.info
    assert info.nhel == 1 << len(spec)
    # chirality along every massless line: each line halves the non-vanishing helicities (same flavour twice: either
    # pairing may conserve it, 6 of the 16 light-quark helicity combinations survive)
    nlines = sum(c in "qQrR" for c in spec) // 2
    frac = {1: 2, 2: 4}[nlines] if set(spec) & set("rR") or nlines == 1 else None
    if frac:
        assert info.ngoodhel == info.nhel // frac and info.nhel_evaluated == info.nhel // (2 * frac)
    else:
        assert info.ngoodhel == info.nhel * 6 // 16 and info.nhel_evaluated == info.ngoodhel // 2
    ph = proc.sigma_per_helicity(mom, nevt)
    torch.cuda.synchronize()
    ph = ph.cpu().numpy()
    for e in range(min(nevt, 4)):
        tot, hel = oracle.me_qchannel(spec, ev[e], per_helicity=True)
        scale = hel.max()
        assert np.abs(ph[:, e] - hel).max() < 1e-9 * scale
    proc.close()


@pytest.mark.parametrize("spec", ["qQtTg", "qgtTqg"])
def test_quark_channel_fp32(mg, oracle, spec):
    import torch
    cfg = workloads.QUARK_CHANNELS[spec]
    nevt = 4133
    p64 = mg.Process(cfg["proc"])
    p32 = mg.Process(cfg["proc"], precision=mg.FP32)
    mom, ev = gpu_events(mg, p64, cfg, nevt)
    a = p64.sigma(mom, nevt).cpu().numpy()
    b = p32.sigma(mom, nevt).cpu().numpy().astype(np.float64)
    torch.cuda.synchronize()
    rel = np.abs(b / a - 1)
    assert np.median(rel) < TOL32_MED and rel.max() < TOL32_MAX, (np.median(rel), rel.max())
    p64.close()
    p32.close()


@pytest.mark.parametrize("proc,nsub,nevt", [("p p > t t~", 3, 512), ("p p > t t~ j", 7, 256), ("p p > t t~ j j", 18, 16)])
def test_multi_subprocess_handle(mg, oracle, proc, nsub, nevt):
    """Several subprocesses behind one handle, evaluated on the SAME momenta (what a p p -> t t~ + jets event needs before
    the PDFs weight them): every row against the oracle of its subprocess."""
    import torch
    m = mg.MultiProcess(proc)
    assert len(m.names) == nsub == len(set(m.names))
    spec_of = {v["proc"]: k for k, v in workloads.QUARK_CHANNELS.items()}
    cfg = dict(sqrt_s=1500.0, seed=77)
    mom, ev = gpu_events(mg, m.sub[0], cfg, nevt)
    me = m.sigma(mom, nevt)
    torch.cuda.synchronize()
    me = me.cpu().numpy()
    assert me.shape == (nsub, nevt)
    for i, name in enumerate(m.names):
        ref = oracle.me_qchannel_batch(spec_of[name], ev) if name in spec_of else oracle.me_batch(name, ev)
        assert np.abs(me[i] / ref - 1).max() < 1e-9, name
        assert m.sub[i].info.npar == ev.shape[1]
    m.close()
    with pytest.raises(mg.MgError) as err:
        mg.MultiProcess("p p > b b~ j")
    assert err.value.status == -2
