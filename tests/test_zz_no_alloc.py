"""mg_weight_max_noalloc (csrc/mg_noalloc.cu): the batch-unweighting primitive for callers that cannot allocate device
memory — its scratch is a fixed __device__ array inside the library.  Checked against the existing path (mg_weight_max,
whose scratch comes from cudaMalloc at handle creation) on two calls in a row: same products, same (max, sum, sum of
squares) — the tolerances of test_weight_max_matches_oracle (products and maximum exact, sums to 1e-13), and in fact
bit-identical since both use the same reduction tree.  Collected last on purpose (file name): the suite runs with
pytest -x.  Runs alone in a fresh process or after the other tests.
"""
import ctypes as C
import math

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2312_02898_b200 as m
    m.lib()
    return m


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_no_alloc_entry_point_matches_the_existing_path_twice(mg, precision):
    import torch
    cfg = workloads.CONFIGS["ggttg"]
    prec = mg.FP64 if precision == "fp64" else mg.FP32
    proc = mg.Process(cfg["proc"], precision=prec)
    out = torch.empty(3, dtype=torch.float64, device="cuda")            # caller-provided: nothing allocated by the call
    # second call smaller than the first: the shared scratch still holds the first call's partials beyond its own
    for call, nevt in enumerate((300001, 8193, 1, 0)):
        mom, w = proc.rambo(cfg["seed"] + call, cfg["sqrt_s"], max(nevt, 1), weights=True)
        me = proc.sigma(mom, max(nevt, 1))[:nevt].clone()
        w = (w[:nevt] * 1e-6).clone()
        me_ref = me.clone()
        ref = proc.weight_max(me_ref, w, nevt)                          # existing path
        got = mg.weight_max_noalloc(me, w, nevt, out=out)               # new entry point, same inputs
        torch.cuda.synchronize()
        assert torch.equal(me, me_ref)                                  # in-place products
        g, r = got.cpu().numpy(), ref.cpu().numpy()
        assert g[0] == r[0]                                             # the maximum is exact
        if nevt:
            assert abs(g[1] / r[1] - 1) < 1e-13 and abs(g[2] / r[2] - 1) < 1e-13
            assert np.array_equal(g, r)                                 # same tree: bit-identical
        else:
            assert g[0] == -math.inf and g[1] == 0 and g[2] == 0
    proc.close()


def test_no_alloc_entry_point_needs_no_handle_and_rejects_oversize(mg):
    """Works without any mg_process_create in the process (run alone, this is the library's first CUDA work); sizes
    beyond the fixed scratch are refused before anything is launched."""
    import torch
    n = 20000
    rng = np.random.default_rng(5)
    me0, w0 = rng.uniform(0.1, 2.0, n), rng.uniform(0.5, 1.5, n)
    me = torch.from_numpy(me0).cuda()
    w = torch.from_numpy(w0).cuda()
    for _ in range(2):                                                  # two calls in a row on fresh copies
        m = me.clone()
        out = mg.weight_max_noalloc(m, w)
        torch.cuda.synchronize()
        prod = w0 * me0
        assert np.array_equal(m.cpu().numpy(), prod)
        o = out.cpu().numpy()
        assert o[0] == prod.max() and abs(o[1] / prod.sum() - 1) < 1e-13 and abs(o[2] / (prod * prod).sum() - 1) < 1e-13
    before = me.clone()
    with pytest.raises(mg.MgError) as err:
        mg.weight_max_noalloc(me, w, nevt=mg.NOALLOC_MAX_EVENTS + 1)
    assert err.value.status == -9 and "MG_NOALLOC_MAX_EVENTS" in str(err.value)
    torch.cuda.synchronize()
    assert torch.equal(me, before)                                      # nothing ran
    L = mg.lib()
    assert L.mg_weight_max_noalloc(7, C.c_void_p(me.data_ptr()), C.c_void_p(w.data_ptr()), 10, C.c_void_p(out.data_ptr()), None) == -3
    assert L.mg_weight_max_noalloc(0, C.c_void_p(me.data_ptr()), C.c_void_p(w.data_ptr()), 10, None, None) == -1
    assert mg.status_string(-9).startswith("size beyond")
