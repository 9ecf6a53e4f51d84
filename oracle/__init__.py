"""ctypes binding of the CPU oracle (oracle/oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from the product package `paper_1201_5029_b200` and shares no code with it; argument
marshalling only -- every number comes out of liboracle.so.
"""
import ctypes as C
import math

import numpy as np

from .build import build as _build

FREE, CHAOTIC, OSCILLON, QBALL = 0, 1, 2, 3
OK, EINVAL, ENOMEM, ESTATE, ENONFINITE = 0, 1, 2, 4, 5


class Params(C.Structure):
    _fields_ = [("model", C.c_int), ("p", C.c_double * 8), ("mpl", C.c_double),
                ("rho_gamma0", C.c_double), ("rho_m0", C.c_double), ("stencil", C.c_double * 4),
                ("precision", C.c_int)]


class Energy(C.Structure):
    _fields_ = [("a", C.c_double), ("p_a", C.c_double), ("eta", C.c_double), ("kin", C.c_double * 4),
                ("grad", C.c_double * 4), ("pot", C.c_double), ("rho", C.c_double),
                ("pressure", C.c_double), ("hubble", C.c_double), ("residual", C.c_double),
                ("sum_phiDphi", C.c_double * 4)]

    def asdict(self):
        d = {}
        for name, _ in self._fields_:
            v = getattr(self, name)
            d[name] = list(v) if hasattr(v, "__len__") else v
        return d


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.c_int
        L.oracle_create.argtypes = [C.POINTER(vp), ip, C.c_double, ip, C.POINTER(Params), ip, C.c_double]
        L.oracle_set_fields.argtypes = [vp, vp, vp]
        L.oracle_set_background.argtypes = [vp, C.c_double, C.c_double]
        L.oracle_set_dt.argtypes = [vp, C.c_double]
        L.oracle_set_adaptive.argtypes = [vp, C.c_int]
        L.oracle_step.argtypes = [vp, ip]
        L.oracle_read_fields.argtypes = [vp, vp, vp]
        L.oracle_energies.argtypes = [vp, C.POINTER(Energy)]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_last_error.argtypes = [vp]
        L.oracle_last_error.restype = C.c_char_p
        L.oracle_stage_weights.argtypes = [ip, dp, ip]
        L.oracle_laplacian.argtypes = [vp, ip, dp]
        L.oracle_gradient_energy.argtypes = [vp, ip, dp]
        L.oracle_potential.argtypes = [vp, dp, dp, dp]
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("oracle status %d: %s" % (code, msg))
        self.code = code


def make_params(model, p=(), mpl=1.0, rho_gamma0=0.0, rho_m0=0.0, stencil=(0, 0, 0, 0), precision=64):
    mp = Params()
    mp.model = model
    for i, v in enumerate(p):
        mp.p[i] = v
    mp.mpl = mpl
    mp.rho_gamma0 = rho_gamma0
    mp.rho_m0 = rho_m0
    for i, v in enumerate(stencil):
        mp.stencil[i] = v
    mp.precision = precision
    return mp


def stage_weights(order):
    w = (C.c_double * 16)()
    n = lib().oracle_stage_weights(order, w, 16)
    return [w[i] for i in range(n)]


class Oracle:
    """One oracle context.  Same call names as the product binding, by design of the ABI (oracle.h)."""

    def __init__(self, N, L, nfields, model, p=(), order=4, dt=0.01, **kw):
        self.N, self.L, self.nf, self.order = N, L, nfields, order
        self.precision = kw.get("precision", 64)
        self._np = np.float32 if self.precision == 32 else np.float64
        self._mp = make_params(model, p, **kw)
        self._h = C.c_void_p()
        st = lib().oracle_create(C.byref(self._h), N, L, nfields, C.byref(self._mp), order, dt)
        if st != OK:
            raise OracleError(st, "oracle_create rejected the arguments")

    def _chk(self, st):
        if st != OK:
            raise OracleError(st, lib().oracle_last_error(self._h).decode())

    def _arr(self, x):
        x = np.ascontiguousarray(x, dtype=self._np)
        assert x.size == self.nf * self.N ** 3, "field buffer has %d elements" % x.size
        return x

    def set_fields(self, phi, pi):
        phi, pi = self._arr(phi), self._arr(pi)
        self._chk(lib().oracle_set_fields(self._h, phi.ctypes.data, pi.ctypes.data))

    def set_background(self, a=1.0, p_a=math.nan):
        self._chk(lib().oracle_set_background(self._h, a, p_a))

    def set_dt(self, dt):
        self._chk(lib().oracle_set_dt(self._h, dt))

    def set_adaptive(self, on=True):
        """dt becomes a physical-time increment: step n has conformal length dt / a_n."""
        self._chk(lib().oracle_set_adaptive(self._h, 1 if on else 0))

    def step(self, n=1):
        self._chk(lib().oracle_step(self._h, n))

    def read_fields(self):
        shape = (self.nf, self.N, self.N, self.N)
        phi, pi = np.empty(shape, self._np), np.empty(shape, self._np)
        self._chk(lib().oracle_read_fields(self._h, phi.ctypes.data, pi.ctypes.data))
        return phi, pi

    def energies(self):
        e = Energy()
        self._chk(lib().oracle_energies(self._h, C.byref(e)))
        return e

    def laplacian(self, f):
        out = np.empty((self.N,) * 3, np.float64)
        self._chk(lib().oracle_laplacian(self._h, f, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def gradient_energy(self, f):
        out = np.empty((self.N,) * 3, np.float64)
        self._chk(lib().oracle_gradient_energy(self._h, f, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def potential(self, phi):
        p = (C.c_double * 4)(*list(phi) + [0.0] * (4 - len(phi)))
        dV = (C.c_double * 4)()
        V = C.c_double()
        self._chk(lib().oracle_potential(self._h, p, C.byref(V), dV))
        return V.value, [dV[i] for i in range(self.nf)]

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
