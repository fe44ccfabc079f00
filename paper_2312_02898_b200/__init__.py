"""Thin Python binding of libmg5b200.so (include/mg5b200.h) — argument marshalling only.

Every step of the path (Philox, RAMBO, wavefunctions, currents, amplitudes, colour sum, helicity sum) runs
in the CUDA kernels behind the C ABI; PyTorch is used here only to own device buffers and streams.  There is
no CPU fallback: importing works without a GPU (so the symbol table can be checked), but creating a process
without a CUDA device raises.

    proc = Process("g g > t t~ g g")
    mom  = proc.rambo(seed=4, sqrt_s=1500.0, nevt=524288)      # torch.float64 CUDA tensor (AoSoA pages)
    me   = proc.sigma(mom, nevt=524288)                         # torch tensor [nevt]
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmg5b200.so")
NEPP = 32
FP64, FP32 = 0, 1
HEL_FILTER, HEL_ALL = 0, 1

SYMBOLS = ["mg_params_default", "mg_process_create", "mg_process_destroy", "mg_rambo", "mg_rambo_ex", "mg_philox_raw", "mg_sigma",
           "mg_sigma_host", "mg_helicity_probe", "mg_sigma_per_helicity", "mg_good_helicities", "mg_process_info",
           "mg_momenta_bytes", "mg_set_workspace", "mg_workspace_bytes", "mg_weight_max", "mg_sigma_mixed", "mg_status_string", "mg_last_error",
           "mg_weight_max_noalloc", "mg_multi_create", "mg_multi_destroy", "mg_multi_count", "mg_multi_name", "mg_multi_process", "mg_multi_sigma"]


class MgParams(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("precision", C.c_int32), ("helicity_mode", C.c_int32),
                ("device", C.c_int32), ("alpha_s", C.c_double), ("alpha_ew_inv", C.c_double), ("gf", C.c_double),
                ("sw2", C.c_double), ("mz", C.c_double), ("gamma_z", C.c_double), ("mt", C.c_double),
                ("gamma_t", C.c_double)]


class MgInfo(C.Structure):
    _fields_ = [("npar", C.c_int32), ("nfinal", C.c_int32), ("ndiagrams", C.c_int32), ("nhel", C.c_int32),
                ("ngoodhel", C.c_int32), ("ncolor", C.c_int32), ("denominator", C.c_int32), ("nepp", C.c_int32),
                ("flops_per_event_allhel", C.c_int64), ("flops_per_event_goodhel", C.c_int64),
                ("masses", C.c_double * 8), ("nkernels_per_tile", C.c_int32), ("launches_last_sigma", C.c_int32),
                ("workspace_bytes", C.c_int64), ("flops_executed_per_event_goodhel", C.c_int64),
                ("nhel_evaluated", C.c_int32), ("reserved", C.c_int32)]


class MgError(RuntimeError):
    def __init__(self, status, detail=""):
        self.status = status
        super().__init__("mg5b200 error %d (%s) %s" % (status, status_string(status), detail))


_lib = None


def lib():
    """Loads the C-ABI library (fails loudly if it was not built: run `python -m paper_2312_02898_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libmg5b200.so not built; run `python -m paper_2312_02898_b200.build`")
        L = C.CDLL(LIB_PATH)
        vp, i64, u64 = C.c_void_p, C.c_int64, C.c_uint64
        L.mg_params_default.argtypes = [C.POINTER(MgParams)]
        L.mg_process_create.argtypes = [C.c_char_p, C.POINTER(MgParams), C.POINTER(vp)]
        L.mg_process_destroy.argtypes = [vp]
        L.mg_rambo.argtypes = [vp, u64, C.c_double, i64, vp, vp]
        L.mg_rambo_ex.argtypes = [vp, u64, C.c_double, i64, i64, vp, vp, vp]
        L.mg_philox_raw.argtypes = [vp, u64, i64, i64, vp, vp]
        L.mg_sigma.argtypes = [vp, vp, i64, vp, vp]
        L.mg_sigma_host.argtypes = [vp, vp, i64, vp, vp]
        L.mg_helicity_probe.argtypes = [vp, vp, i64, vp]
        L.mg_sigma_per_helicity.argtypes = [vp, vp, i64, vp, vp]
        L.mg_good_helicities.argtypes = [vp, C.POINTER(C.c_int32), C.c_int32, C.POINTER(C.c_int32)]
        L.mg_process_info.argtypes = [vp, C.POINTER(MgInfo)]
        L.mg_momenta_bytes.argtypes = [vp, i64]
        L.mg_momenta_bytes.restype = C.c_size_t
        L.mg_set_workspace.argtypes = [vp, vp, C.c_size_t]
        L.mg_workspace_bytes.argtypes = [vp, i64]
        L.mg_workspace_bytes.restype = C.c_size_t
        L.mg_weight_max.argtypes = [vp, vp, vp, i64, vp, vp]
        L.mg_weight_max_noalloc.argtypes = [C.c_int, vp, vp, i64, vp, vp]
        L.mg_sigma_mixed.argtypes = [vp, vp, i64, vp, C.c_double, vp, C.POINTER(i64), vp]
        L.mg_multi_create.argtypes = [C.c_char_p, C.POINTER(MgParams), C.POINTER(vp)]
        L.mg_multi_destroy.argtypes = [vp]
        L.mg_multi_count.argtypes = [vp]
        L.mg_multi_name.argtypes = [vp, C.c_int]
        L.mg_multi_name.restype = C.c_char_p
        L.mg_multi_process.argtypes = [vp, C.c_int]
        L.mg_multi_process.restype = vp
        L.mg_multi_sigma.argtypes = [vp, vp, i64, vp, vp]
        L.mg_status_string.argtypes = [C.c_int]
        L.mg_status_string.restype = C.c_char_p
        L.mg_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def status_string(status):
    return lib().mg_status_string(status).decode()


def _check(rc):
    if rc != 0:
        raise MgError(rc, lib().mg_last_error().decode() if rc in (-7, -9) else "")


def default_params(precision=FP64, helicity_mode=HEL_FILTER, device=0, **kw):
    p = MgParams()
    _check(lib().mg_params_default(C.byref(p)))
    p.precision, p.helicity_mode, p.device = precision, helicity_mode, device
    for k, v in kw.items():
        setattr(p, k, v)
    return p


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


class Process:
    """One process handle (mg_process_t)."""

    def __init__(self, proc, precision=FP64, helicity_mode=HEL_FILTER, device=0, **params):
        self._h = C.c_void_p()
        self.params = default_params(precision, helicity_mode, device, **params)
        self.proc = proc
        _check(lib().mg_process_create(proc.encode(), C.byref(self.params), C.byref(self._h)))
        self.precision = precision
        self.device = device

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().mg_process_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def info(self):
        o = MgInfo()
        _check(lib().mg_process_info(self._h, C.byref(o)))
        return o

    def momenta_bytes(self, nevt):
        return int(lib().mg_momenta_bytes(self._h, nevt))

    def alloc_momenta(self, nevt):
        import torch
        return torch.empty(self.momenta_bytes(nevt) // 8, dtype=torch.float64, device="cuda:%d" % self.device)

    def rambo(self, seed, sqrt_s, nevt, first_event=0, out=None, weights=False, stream=None):
        """mg_rambo / mg_rambo_ex -> AoSoA momenta tensor (and weights)."""
        import torch
        mom = out if out is not None else self.alloc_momenta(nevt)
        w = torch.empty(nevt, dtype=torch.float64, device=mom.device) if weights else None
        _check(lib().mg_rambo_ex(self._h, seed, float(sqrt_s), first_event, nevt, C.c_void_p(mom.data_ptr()),
                                 C.c_void_p(w.data_ptr()) if weights else None, _stream_ptr(stream)))
        return (mom, w) if weights else mom

    def philox_raw(self, seed, nevt, first_event=0, stream=None):
        """mg_philox_raw -> int32 tensor [nevt, nfinal, 4] holding the raw uint32 words."""
        import torch
        nf = self.info.nfinal
        out = torch.empty((nevt, nf, 4), dtype=torch.int32, device="cuda:%d" % self.device)
        _check(lib().mg_philox_raw(self._h, seed, first_event, nevt, C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def _out_dtype(self):
        import torch
        return torch.float64 if self.precision == FP64 else torch.float32

    def sigma(self, momenta, nevt, out=None, stream=None):
        """mg_sigma: |M|^2 per event (device tensor in, device tensor out)."""
        import torch
        assert momenta.is_cuda and momenta.dtype == torch.float64 and momenta.numel() * 8 >= self.momenta_bytes(nevt)
        me = out if out is not None else torch.empty(nevt, dtype=self._out_dtype(), device=momenta.device)
        _check(lib().mg_sigma(self._h, C.c_void_p(momenta.data_ptr()), nevt, C.c_void_p(me.data_ptr()),
                              _stream_ptr(stream)))
        return me

    def sigma_host(self, momenta_host, nevt, out_host=None, stream=None):
        """mg_sigma_host: host (ideally pinned) tensors in and out; includes H2D/D2H copies."""
        import torch
        assert not momenta_host.is_cuda and momenta_host.dtype == torch.float64
        me = out_host if out_host is not None else torch.empty(nevt, dtype=self._out_dtype()).pin_memory()
        _check(lib().mg_sigma_host(self._h, C.c_void_p(momenta_host.data_ptr()), nevt, C.c_void_p(me.data_ptr()),
                                   _stream_ptr(stream)))
        return me

    def sigma_per_helicity(self, momenta, nevt, stream=None):
        import torch
        nhel = self.info.nhel
        out = torch.empty((nhel, nevt), dtype=self._out_dtype(), device=momenta.device)
        _check(lib().mg_sigma_per_helicity(self._h, C.c_void_p(momenta.data_ptr()), nevt, C.c_void_p(out.data_ptr()),
                                           _stream_ptr(stream)))
        return out

    def helicity_probe(self, momenta, nprobe, stream=None):
        _check(lib().mg_helicity_probe(self._h, C.c_void_p(momenta.data_ptr()), nprobe, _stream_ptr(stream)))
        return self.good_helicities()

    def set_workspace(self, buf):
        """mg_set_workspace: `buf` = a CUDA tensor the caller keeps alive (None: back to the library-owned workspace)."""
        if buf is None:
            _check(lib().mg_set_workspace(self._h, None, 0))
        else:
            _check(lib().mg_set_workspace(self._h, C.c_void_p(buf.data_ptr()), buf.numel() * buf.element_size()))
        self._ws_keepalive = buf

    def workspace_bytes(self, nevt):
        return int(lib().mg_workspace_bytes(self._h, nevt))

    def weight_max(self, me, weights, nevt=None, out=None, stream=None):
        """mg_weight_max: me <- weights * me in place; returns the device tensor (max, sum, sum of squares)."""
        import torch
        nevt = me.numel() if nevt is None else nevt
        assert me.is_cuda and weights.is_cuda and weights.dtype == torch.float64 and me.dtype == self._out_dtype()
        res = out if out is not None else torch.empty(3, dtype=torch.float64, device=me.device)
        _check(lib().mg_weight_max(self._h, C.c_void_p(me.data_ptr()), C.c_void_p(weights.data_ptr()), nevt,
                                   C.c_void_p(res.data_ptr()), _stream_ptr(stream)))
        return res

    def sigma_mixed(self, momenta, nevt, tol, with_eps=False, stream=None):
        """mg_sigma_mixed: fp32 everywhere, fp64 where the measured fp32 error exceeds tol.  Returns (|M|^2 as a
        float64 device tensor, number of re-evaluated events[, eps as a float32 device tensor])."""
        import torch
        me = torch.empty(nevt, dtype=torch.float64, device=momenta.device)
        eps = torch.empty(nevt, dtype=torch.float32, device=momenta.device) if with_eps else None
        nf = C.c_int64()
        _check(lib().mg_sigma_mixed(self._h, C.c_void_p(momenta.data_ptr()), nevt, C.c_void_p(me.data_ptr()), float(tol),
                                    C.c_void_p(eps.data_ptr()) if with_eps else None, C.byref(nf), _stream_ptr(stream)))
        return (me, nf.value, eps) if with_eps else (me, nf.value)

    def good_helicities(self):
        n = C.c_int32()
        buf = (C.c_int32 * 256)()
        _check(lib().mg_good_helicities(self._h, buf, 256, C.byref(n)))
        return [int(buf[i]) for i in range(n.value)]


NOALLOC_MAX_EVENTS = 8388608


def weight_max_noalloc(me, weights, nevt=None, out=None, stream=None):
    """mg_weight_max_noalloc: me <- weights * me in place and (max, sum, sum of squares) of the products into `out`
    (3 doubles, caller-provided so that nothing is allocated here; created with torch.empty if None).  No handle, no
    device allocation inside the library; nevt <= NOALLOC_MAX_EVENTS; calls on one device must not overlap."""
    import torch
    if nevt is None:
        nevt = me.numel()
    if out is None:
        out = torch.empty(3, dtype=torch.float64, device=me.device)
    prec = FP64 if me.dtype == torch.float64 else FP32
    _check(lib().mg_weight_max_noalloc(prec, C.c_void_p(me.data_ptr()), C.c_void_p(weights.data_ptr()), nevt,
                                       C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
    return out


class MultiProcess:
    """Several subprocesses behind one handle (mg_multi_t): "p p > t t~ j" etc.; `sub[i]` are borrowed Process views."""

    def __init__(self, proc, precision=FP64, helicity_mode=HEL_FILTER, device=0, **params):
        self._m = C.c_void_p()
        self.params = default_params(precision, helicity_mode, device, **params)
        _check(lib().mg_multi_create(proc.encode(), C.byref(self.params), C.byref(self._m)))
        self.precision, self.device = precision, device
        n = lib().mg_multi_count(self._m)
        self.names = [lib().mg_multi_name(self._m, i).decode() for i in range(n)]
        self.sub = []
        for i in range(n):
            v = Process.__new__(Process)          # a view: the multi handle owns the subprocess handle
            v._h = None
            v._borrowed = C.c_void_p(lib().mg_multi_process(self._m, i))
            v.params, v.proc, v.precision, v.device = self.params, self.names[i], precision, device
            self.sub.append(v)
        for v in self.sub:
            v._h = v._borrowed
            v.close = lambda: None                # never destroyed through the view

    def sigma(self, momenta, nevt, out=None, stream=None):
        """|M|^2 of every subprocess on the same momenta: tensor [nsub][nevt]."""
        import torch
        if out is None:
            out = torch.empty((len(self.sub), nevt), dtype=torch.float64 if self.precision == FP64 else torch.float32,
                              device=momenta.device)
        _check(lib().mg_multi_sigma(self._m, C.c_void_p(momenta.data_ptr()), nevt, C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def close(self):
        if getattr(self, "_m", None) is not None and self._m.value:
            for v in self.sub:
                v._h = C.c_void_p()
            lib().mg_multi_destroy(self._m)
            self._m = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def shard(nevt_per_gpu, rank, world_size=1):
    """Weak-scaling shard of the global event stream: rank r owns the global events
    [r * nevt_per_gpu, (r + 1) * nevt_per_gpu).  Returns (first_event, nevt).  The Philox counter is the global
    event index, so the union over ranks equals one big batch; no collective is needed on the data path."""
    if not (0 <= rank < world_size) or nevt_per_gpu < 0:
        raise ValueError("bad shard")
    return rank * nevt_per_gpu, nevt_per_gpu


def allreduce_weight_stats(out3, group=None):
    """Combines the (max, sum, sum of squares) of mg_weight_max over the ranks that sharded the event stream (SURVEY.md §8e:
    the only exchange a consumer of PAPER.md:101 needs: one all-reduce of three doubles per batch; the data path itself
    has no collective).  In place on `out3` (CUDA tensor with NCCL, CPU tensor with gloo); returns it."""
    import torch.distributed as dist
    dist.all_reduce(out3[0:1], op=dist.ReduceOp.MAX, group=group)
    dist.all_reduce(out3[1:3], op=dist.ReduceOp.SUM, group=group)
    return out3


def pages_to_events(momenta, nevt, npar):
    """AoSoA pages [page][ipar][32][4] -> plain [nevt][npar][4] (layout shuffle only; torch or numpy)."""
    pages = (nevt + NEPP - 1) // NEPP
    v = momenta[: pages * npar * NEPP * 4].reshape(pages, npar, NEPP, 4)
    if hasattr(v, "permute"):
        return v.permute(0, 2, 1, 3).reshape(pages * NEPP, npar, 4)[:nevt]
    return v.transpose(0, 2, 1, 3).reshape(pages * NEPP, npar, 4)[:nevt]


def events_to_pages(events):
    """Plain [nevt][npar][4] (numpy or torch) -> AoSoA pages, zero-padded to whole pages."""
    import numpy as np
    is_torch = hasattr(events, "permute")
    ev = events.cpu().numpy() if is_torch else np.asarray(events, dtype=np.float64)
    nevt, npar, _ = ev.shape
    pages = (nevt + NEPP - 1) // NEPP
    buf = np.zeros((pages * NEPP, npar, 4))
    buf[:nevt] = ev
    if nevt < pages * NEPP:          # pad with copies of the last event so tail lanes stay finite
        buf[nevt:] = ev[-1] if nevt else 0.0
    out = np.ascontiguousarray(buf.reshape(pages, NEPP, npar, 4).transpose(0, 2, 1, 3)).reshape(-1)
    if is_torch:
        import torch
        return torch.from_numpy(out)
    return out
