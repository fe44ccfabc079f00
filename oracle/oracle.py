"""ctypes view of the CPU oracle (TEST INFRASTRUCTURE — see oracle/oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It never imports the CUDA package.  `load(long_double=True)` gives the x87 80-bit build used to
adjudicate parity; the double build is the one that is timed.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))


class Params(C.Structure):
    _fields_ = [("alpha_s", C.c_double), ("alpha_ew_inv", C.c_double), ("sw2", C.c_double),
                ("mz", C.c_double), ("gamma_z", C.c_double), ("mt", C.c_double)]


def default_sw2(alpha_ew_inv=132.507, gf=1.16639e-5, mz=91.188):
    """A1 reading: MG5 'sm' scheme, M_W from (alpha, G_F, M_Z)."""
    import math
    a = 1.0 / alpha_ew_inv
    mw2 = mz * mz / 2 + math.sqrt(mz ** 4 / 4 - math.pi * a * mz * mz / (math.sqrt(2) * gf))
    return 1.0 - mw2 / (mz * mz)


def default_params():
    return Params(0.118, 132.507, default_sw2(), 91.188, 2.4414, 173.0)


def build():
    subprocess.check_call(["sh", os.path.join(_HERE, "build.sh")])


_dp = C.POINTER(C.c_double)


def _p(a):
    return a.ctypes.data_as(_dp)


class Oracle:
    PROCS = {"e+ e- > mu+ mu-": 0, "g g > t t~": 1, "g g > t t~ g": 2, "g g > t t~ g g": 3, "g g > t t~ g g g": 4}

    def __init__(self, long_double=False):
        name = "liboracle_ld.so" if long_double else "liboracle.so"
        path = os.path.join(_HERE, name)
        if not os.path.exists(path):
            build()
        L = self.lib = C.CDLL(path)
        L.oracle_me_eemumu.restype = C.c_double
        L.oracle_me_ggttng.restype = C.c_double
        L.oracle_me_ggttng_dressed.restype = C.c_double
        L.oracle_me_ggtt_explicit.restype = C.c_double
        L.oracle_me_ggttng_ward.restype = C.c_double
        L.oracle_rambo.argtypes = [C.c_uint64, C.c_int64, C.c_int64, C.c_int, _dp, C.c_double, _dp, _dp]
        L.oracle_me_batch.argtypes = [C.c_int, _dp, C.c_int64, C.POINTER(Params), _dp, C.c_int]
        L.oracle_me_qchannel.restype = C.c_double
        L.oracle_me_qchannel.argtypes = [C.c_char_p, _dp, C.POINTER(Params), _dp, C.c_int]
        L.oracle_me_qchannel_pauli.restype = C.c_double
        L.oracle_me_qchannel_pauli.argtypes = [C.c_char_p, _dp, C.POINTER(Params)]
        L.oracle_me_qchannel_batch.argtypes = [C.c_char_p, _dp, C.c_int64, C.POINTER(Params), _dp, C.c_int]
        L.oracle_weight_max.argtypes = [_dp, _dp, C.c_int64, C.c_int, _dp, _dp]

    def philox(self, ctr, key):
        c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
        self.lib.oracle_philox4x32_10(c, k, o)
        return [int(x) for x in o]

    def rambo(self, seed, nevt, masses_final, sqrt_s, first_event=0, weights=False):
        m = np.ascontiguousarray(masses_final, dtype=np.float64)
        n = len(m)
        mom = np.zeros((nevt, n + 2, 4))
        w = np.zeros(nevt) if weights else None
        rc = self.lib.oracle_rambo(seed, first_event, nevt, n, _p(m), sqrt_s, _p(mom), _p(w) if weights else None)
        if rc != 0:
            raise ValueError("sqrt_s <= sum of masses")
        return (mom, w) if weights else mom

    def spinor(self, kind, p, m, lam):
        out = np.zeros(8); p = np.ascontiguousarray(p, dtype=np.float64)
        fn = {"u": self.lib.oracle_spinor_u, "v": self.lib.oracle_spinor_v}[kind]
        fn(_p(p), C.c_double(m), C.c_int(lam), _p(out))
        return out[0::2] + 1j * out[1::2]

    def polvec(self, k, lam):
        out = np.zeros(8); k = np.ascontiguousarray(k, dtype=np.float64)
        self.lib.oracle_polvec(_p(k), C.c_int(lam), _p(out))
        return out[0::2] + 1j * out[1::2]

    def gamma(self, mu):
        out = np.zeros(32)
        self.lib.oracle_gamma(C.c_int(mu), _p(out))
        return (out[0::2] + 1j * out[1::2]).reshape(4, 4)

    def colour_matrix(self, n, brute=False):
        import math
        npm = math.factorial(n)
        cf = np.zeros((npm, npm))
        self.lib.oracle_colour_matrix(C.c_int(n), _p(cf), C.c_int(1 if brute else 0))
        return cf

    def me(self, proc, p, par=None, per_helicity=False):
        """|M|^2 for one event; p [npar][4]."""
        par = par or default_params()
        ip = self.PROCS[proc] if isinstance(proc, str) else proc
        p = np.ascontiguousarray(p, dtype=np.float64)
        npar = 4 if ip == 0 else ip + 3
        assert p.shape == (npar, 4)
        hel = np.zeros(1 << npar) if per_helicity else None
        hp = _p(hel) if per_helicity else None
        if ip == 0:
            v = self.lib.oracle_me_eemumu(_p(p), C.byref(par), hp)
        else:
            v = self.lib.oracle_me_ggttng(C.c_int(ip - 1), _p(p), C.byref(par), hp)
        return (v, hel) if per_helicity else v

    def me_dressed(self, nfinal_gluons, p, par=None):
        par = par or default_params(); p = np.ascontiguousarray(p, dtype=np.float64)
        return self.lib.oracle_me_ggttng_dressed(C.c_int(nfinal_gluons), _p(p), C.byref(par))

    def me_ggtt_explicit(self, p, par=None):
        par = par or default_params(); p = np.ascontiguousarray(p, dtype=np.float64)
        return self.lib.oracle_me_ggtt_explicit(_p(p), C.byref(par))

    def me_ward(self, nfinal_gluons, p, which, par=None):
        par = par or default_params(); p = np.ascontiguousarray(p, dtype=np.float64)
        return self.lib.oracle_me_ggttng_ward(C.c_int(nfinal_gluons), _p(p), C.byref(par), C.c_int(which))

    def me_batch(self, proc, momenta, par=None, nthreads=0):
        par = par or default_params()
        ip = self.PROCS[proc] if isinstance(proc, str) else proc
        mom = np.ascontiguousarray(momenta, dtype=np.float64)
        out = np.zeros(mom.shape[0])
        rc = self.lib.oracle_me_batch(ip, _p(mom), mom.shape[0], C.byref(par), _p(out), nthreads)
        assert rc == 0
        return out

    def me_qchannel(self, spec, p, par=None, per_helicity=False, ward=-1):
        """Quark channels (oracle.h): spec e.g. "qQtTg"; p [npar][4]."""
        par = par or default_params(); p = np.ascontiguousarray(p, dtype=np.float64)
        assert p.shape == (len(spec), 4)
        hel = np.zeros(1 << len(spec)) if per_helicity else None
        v = self.lib.oracle_me_qchannel(spec.encode(), _p(p), C.byref(par), _p(hel) if per_helicity else None, C.c_int(ward))
        return (v, hel) if per_helicity else v

    def me_qchannel_pauli(self, spec, p, par=None):
        """Part of |M|^2 from equal helicity and colour of the two identical final quarks (oracle.h)."""
        par = par or default_params(); p = np.ascontiguousarray(p, dtype=np.float64)
        return self.lib.oracle_me_qchannel_pauli(spec.encode(), _p(p), C.byref(par))

    def me_qchannel_batch(self, spec, momenta, par=None, nthreads=0):
        par = par or default_params()
        mom = np.ascontiguousarray(momenta, dtype=np.float64)
        out = np.zeros(mom.shape[0])
        rc = self.lib.oracle_me_qchannel_batch(spec.encode(), _p(mom), mom.shape[0], C.byref(par), _p(out), nthreads)
        assert rc == 0
        return out

    def weight_max(self, me, w, single=False):
        """(products, (max, sum, sum of squares)) of w * me."""
        me = np.ascontiguousarray(me, dtype=np.float64); w = np.ascontiguousarray(w, dtype=np.float64)
        prod = np.zeros(len(me)); out = np.zeros(3)
        self.lib.oracle_weight_max(_p(me), _p(w), len(me), 1 if single else 0, _p(prod), _p(out))
        return prod, out

    def num_threads(self):
        return int(self.lib.oracle_num_threads())


_cache = {}


def load(long_double=False):
    if long_double not in _cache:
        _cache[long_double] = Oracle(long_double)
    return _cache[long_double]
