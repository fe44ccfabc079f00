"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/mg5b200.h declares, struct layouts of the Python binding match the header, and the layout
helpers round-trip.  No compute call is made (there is no GPU here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mg5b200.h")


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mg_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_four_named_calls():
    syms = declared_symbols()
    for s in ("mg_process_create", "mg_rambo", "mg_sigma", "mg_process_destroy"):
        assert s in syms


def test_library_exports_every_declared_symbol():
    import paper_2312_02898_b200 as mg
    if not os.path.exists(mg.LIB_PATH):
        from paper_2312_02898_b200 import build
        build.build(log=False)
    L = C.CDLL(mg.LIB_PATH)
    for s in declared_symbols():
        assert hasattr(L, s), "libmg5b200.so does not export %s" % s
    assert sorted(mg.SYMBOLS) == declared_symbols()


def test_param_struct_matches_header_and_defaults():
    import paper_2312_02898_b200 as mg
    p = mg.default_params()
    assert p.struct_size == C.sizeof(mg.MgParams) == 80
    assert (p.alpha_s, p.alpha_ew_inv, p.mz, p.gamma_z, p.mt, p.gamma_t) == (0.118, 132.507, 91.188, 2.4414, 173.0, 0.0)
    assert C.sizeof(mg.MgInfo) == 8 * 4 + 2 * 8 + 8 * 8 + 2 * 4 + 8 + 8 + 2 * 4


def test_status_strings_and_argument_errors_without_gpu():
    import paper_2312_02898_b200 as mg
    L = mg.lib()
    assert mg.status_string(0) == "ok"
    assert L.mg_process_create(None, None, None) == -1           # MG_ERR_NULL
    h = C.c_void_p()
    p = mg.default_params()
    assert L.mg_process_create(b"u u~ > d d~", C.byref(p), C.byref(h)) == -2      # MG_ERR_BAD_PROC
    assert L.mg_multi_create(b"p p > b b~ j", C.byref(p), C.byref(h)) == -2        # nothing generated matches
    assert L.mg_multi_create(b"p p > t t~ > j", C.byref(p), C.byref(h)) == -2
    assert L.mg_multi_count(None) == 0 and L.mg_multi_sigma(None, None, 0, None, None) == -1
    # no-allocation entry point: size beyond its fixed scratch is refused before any CUDA call
    buf = (C.c_double * 4)()
    assert L.mg_weight_max_noalloc(0, buf, buf, 8388608 + 1, buf, None) == -9 and b"MG_NOALLOC_MAX_EVENTS" in L.mg_last_error()
    assert L.mg_weight_max_noalloc(0, buf, buf, -1, buf, None) == -4
    p.struct_size = 12
    assert L.mg_process_create(b"g g > t t~", C.byref(p), C.byref(h)) == -3       # MG_ERR_BAD_PARAM
    p = mg.default_params(gamma_t=1.5)
    assert L.mg_process_create(b"g g > t t~", C.byref(p), C.byref(h)) == -3       # reading A2: Gamma_t = 0
    import torch
    if not torch.cuda.is_available():
        p = mg.default_params()
        assert L.mg_process_create(b"g g > t t~", C.byref(p), C.byref(h)) == -8   # MG_ERR_NO_DEVICE: no CPU fallback
        with pytest.raises(mg.MgError):
            mg.Process("g g > t t~")


def test_page_layout_roundtrip():
    import paper_2312_02898_b200 as mg
    rng = np.random.default_rng(0)
    for nevt in (1, 31, 32, 33, 100):
        ev = rng.normal(size=(nevt, 5, 4))
        pages = mg.events_to_pages(ev)
        assert pages.size == ((nevt + 31) // 32) * 5 * 32 * 4
        back = mg.pages_to_events(pages, nevt, 5)
        assert np.array_equal(back, ev)
        # element (ievt, ipar, mu) sits at ((page*npar + ipar)*32 + lane)*4 + mu
        i = nevt - 1
        assert pages[((i // 32 * 5 + 3) * 32 + i % 32) * 4 + 2] == ev[i, 3, 2]
