"""Thin Python binding of libpycool.so (include/pycool.h): argument marshalling only.

PyTorch supplies device memory (the state and work buffers are torch tensors handed to
`pycool_create_ext`) and the CUDA stream; every step of the path runs in the library's sm_100a kernels.
There is no fallback: if the library is missing or no CUDA device is present, calls raise.
"""
import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpycool.so")

FREE, CHAOTIC, OSCILLON, QBALL = 0, 1, 2, 3
OK, EINVAL, ENOMEM, ECUDA, ESTATE, ENONFINITE = 0, 1, 2, 3, 4, 5

# every symbol include/pycool.h declares (tests check the library exports exactly these)
SYMBOLS = ("pycool_create", "pycool_work_bytes", "pycool_create_ext", "pycool_set_fields",
           "pycool_set_fields_device", "pycool_set_background", "pycool_set_dt", "pycool_step", "pycool_sync",
           "pycool_read_fields", "pycool_read_fields_device", "pycool_device_fields", "pycool_energies", "pycool_destroy",
           "pycool_last_error", "pycool_stage_weights", "pycool_launch_counts", "pycool_set_profiling",
           "pycool_kick_time_ms", "pycool_kick_geometry", "pycool_set_zchunk", "pycool_set_tile",
           "pycool_set_fused_tail", "pycool_set_cooperative", "pycool_set_persistent", "pycool_flush", "pycool_set_adaptive", "pycool_set_energy_kernel", "pycool_set_overlap", "pycool_set_item_order", "pycool_init_fields",
           "pycool_field_spectrum", "pycool_mode_spectra", "pycool_set_energy_cadence", "pycool_read_energy_log",
           # include/pycool_linear.h
           "pycool_linear_create", "pycool_linear_num_classes", "pycool_linear_set_background",
           "pycool_linear_set_perturbations", "pycool_linear_set_modes", "pycool_linear_step", "pycool_linear_read_modes",
           "pycool_linear_read_perturbations", "pycool_linear_background_state", "pycool_linear_growth",
           "pycool_linear_time_ms", "pycool_linear_destroy", "pycool_linear_last_error", "pycool_linear_growth_static",
           "pycool_linear_static_last_error")
GROWTH, NAIVE = 0, 1


class Params(C.Structure):
    _fields_ = [("model", C.c_int), ("p", C.c_double * 8), ("mpl", C.c_double),
                ("rho_gamma0", C.c_double), ("rho_m0", C.c_double), ("stencil", C.c_double * 4),
                ("precision", C.c_int)]


class Spectrum(C.Structure):
    _fields_ = [("mean", C.c_double), ("amp", C.c_double), ("m2", C.c_double), ("q", C.c_double), ("kmax", C.c_double)]


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


class LinearBackground(C.Structure):
    _fields_ = [("a", C.c_double), ("p_a", C.c_double), ("eta", C.c_double), ("phi0", C.c_double * 4),
                ("pi0", C.c_double * 4), ("kin", C.c_double), ("pot", C.c_double), ("rho", C.c_double),
                ("hubble", C.c_double), ("residual", C.c_double)]


class PycoolError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("pycool status %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib():
    """Load libpycool.so (built in-tree by `python -m paper_1201_5029_b200.build`).  Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libpycool.so is not built: run `python -m paper_1201_5029_b200.build` "
                               "(there is no CPU or PyTorch fallback)")
        L = C.CDLL(LIB_PATH)
        vp, ip, d = C.c_void_p, C.c_int, C.c_double
        pp = C.POINTER(Params)
        L.pycool_create.argtypes = [C.POINTER(vp), ip, d, ip, pp, ip, d]
        L.pycool_work_bytes.argtypes = [ip, ip, ip]
        L.pycool_work_bytes.restype = C.c_size_t
        L.pycool_create_ext.argtypes = [C.POINTER(vp), ip, d, ip, pp, ip, d, vp, C.c_size_t, vp]
        L.pycool_set_fields.argtypes = [vp, vp, vp]
        L.pycool_set_fields_device.argtypes = [vp, vp, vp]
        L.pycool_set_background.argtypes = [vp, d, d]
        L.pycool_set_dt.argtypes = [vp, d]
        L.pycool_step.argtypes = [vp, ip]
        L.pycool_sync.argtypes = [vp]
        L.pycool_read_fields.argtypes = [vp, vp, vp]
        L.pycool_read_fields_device.argtypes = [vp, vp, vp]
        L.pycool_device_fields.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(C.c_size_t)]
        L.pycool_energies.argtypes = [vp, C.POINTER(Energy)]
        L.pycool_destroy.argtypes = [vp]
        L.pycool_last_error.argtypes = [vp]
        L.pycool_last_error.restype = C.c_char_p
        L.pycool_stage_weights.argtypes = [ip, C.POINTER(d), ip]
        L.pycool_launch_counts.argtypes = [vp, C.POINTER(C.c_ulonglong)]
        L.pycool_set_profiling.argtypes = [vp, ip]
        L.pycool_kick_time_ms.argtypes = [vp, C.POINTER(d), C.POINTER(C.c_ulonglong)]
        L.pycool_kick_geometry.argtypes = [vp, C.POINTER(ip)]
        L.pycool_set_zchunk.argtypes = [vp, ip]
        L.pycool_set_tile.argtypes = [vp, ip]
        L.pycool_set_fused_tail.argtypes = [vp, ip]
        L.pycool_set_cooperative.argtypes = [vp, ip]
        L.pycool_set_persistent.argtypes = [vp, ip]
        L.pycool_flush.argtypes = [vp]
        L.pycool_set_adaptive.argtypes = [vp, ip]
        L.pycool_set_energy_kernel.argtypes = [vp, ip]
        L.pycool_set_overlap.argtypes = [vp, ip]
        L.pycool_set_item_order.argtypes = [vp, ip]
        L.pycool_field_spectrum.argtypes = [vp, ip, ip, ip, C.POINTER(d), C.POINTER(d)]
        L.pycool_init_fields.argtypes = [vp, C.c_ulonglong, C.POINTER(Spectrum), C.POINTER(Spectrum)]
        L.pycool_mode_spectra.argtypes = [vp, ip, d, ip, C.POINTER(d), C.POINTER(d), C.POINTER(d)]
        L.pycool_set_energy_cadence.argtypes = [vp, ip, ip]
        L.pycool_read_energy_log.argtypes = [vp, C.POINTER(Energy), ip, C.POINTER(ip), C.POINTER(C.c_ulonglong)]
        dp = C.POINTER(d)
        L.pycool_linear_create.argtypes = [C.POINTER(vp), ip, d, ip, pp, ip, d]
        L.pycool_linear_num_classes.argtypes = [ip]
        L.pycool_linear_num_classes.restype = C.c_size_t
        L.pycool_linear_set_background.argtypes = [vp, d, d, dp, dp]
        L.pycool_linear_set_perturbations.argtypes = [vp, vp, vp]
        L.pycool_linear_set_modes.argtypes = [vp, vp, vp]
        L.pycool_linear_step.argtypes = [vp, ip, ip]
        L.pycool_linear_read_modes.argtypes = [vp, vp, vp]
        L.pycool_linear_read_perturbations.argtypes = [vp, vp, vp]
        L.pycool_linear_background_state.argtypes = [vp, C.POINTER(LinearBackground)]
        L.pycool_linear_growth.argtypes = [vp, vp, C.c_size_t, C.POINTER(C.c_size_t)]
        L.pycool_linear_time_ms.argtypes = [vp, dp]
        L.pycool_linear_destroy.argtypes = [vp]
        L.pycool_linear_last_error.argtypes = [vp]
        L.pycool_linear_last_error.restype = C.c_char_p
        L.pycool_linear_growth_static.argtypes = [ip, d, ip, pp, ip, d, ip, d, d, dp, dp, vp, C.c_size_t, vp]
        L.pycool_linear_static_last_error.argtypes = []
        L.pycool_linear_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


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
    n = lib().pycool_stage_weights(order, w, 16)
    return [w[i] for i in range(n)]


def work_bytes(N, nfields, precision=64):
    return lib().pycool_work_bytes(N, nfields, precision)


class Lattice:
    """One simulation context on a CUDA device.  Same call names as the C ABI.

    device: a torch device (default cuda:0).  The field and work buffers are torch tensors owned by this
    object; the library computes in them on the stream that is torch's current stream for that device when the
    Lattice is made.  The library records the device of the work buffer and runs every later call on it,
    whatever device is current in the calling thread (several Lattices on several GPUs in one process are fine).
    """

    def __init__(self, N, L, nfields, model, p=(), order=4, dt=0.01, device=None, **kw):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1201_5029_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.N, self.L, self.nf, self.order = N, L, nfields, order
        self.precision = kw.get("precision", 64)
        self._np = np.float32 if self.precision == 32 else np.float64
        self._tdtype = torch.float32 if self.precision == 32 else torch.float64
        self.device = torch.device("cuda:0" if device is None else device)
        self._mp = make_params(model, p, **kw)
        self._h = C.c_void_p()
        need = work_bytes(N, nfields, self.precision)
        if need == 0:
            raise PycoolError(EINVAL, "invalid lattice shape")
        with torch.cuda.device(self.device):
            self._work = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
            wptr = (self._work.data_ptr() + 255) // 256 * 256
            self.stream = torch.cuda.current_stream(self.device)
            st = lib().pycool_create_ext(C.byref(self._h), N, L, nfields, C.byref(self._mp), order, dt,
                                         wptr, need, self.stream.cuda_stream)
        if st != OK:
            raise PycoolError(st, lib().pycool_last_error(None).decode())

    def _chk(self, st):
        if st != OK:
            raise PycoolError(st, lib().pycool_last_error(self._h).decode())

    def _host(self, x):
        x = np.ascontiguousarray(x, dtype=self._np)
        if x.size != self.nf * self.N ** 3:
            raise PycoolError(EINVAL, "field buffer has %d elements" % x.size)
        return x

    def _check_tensor(self, t, name, want_cuda=None):
        """A torch tensor handed to the library as a raw pointer: right dtype, size, layout and device."""
        n = self.nf * self.N ** 3
        if t.dtype != self._tdtype or t.numel() != n or not t.is_contiguous():
            raise PycoolError(EINVAL, "%s must be a contiguous %s tensor of %d elements (got %s, %d, contiguous=%s)"
                              % (name, self._tdtype, n, t.dtype, t.numel(), t.is_contiguous()))
        if want_cuda is not None and t.is_cuda != want_cuda:
            raise PycoolError(EINVAL, "%s is on %s: phi and pi must both be host or both be device tensors" % (name, t.device))
        if t.is_cuda and t.device != self.device:
            raise PycoolError(EINVAL, "%s is on %s, the lattice on %s" % (name, t.device, self.device))

    def set_fields(self, phi, pi):
        """phi, pi: host arrays (numpy, or pinned torch CPU tensors) or torch tensors on the lattice's device, of
        nf*N^3 elements each."""
        torch = self._torch
        if isinstance(phi, torch.Tensor) or isinstance(pi, torch.Tensor):
            if not (isinstance(phi, torch.Tensor) and isinstance(pi, torch.Tensor)):
                raise PycoolError(EINVAL, "phi and pi must both be torch tensors or both be arrays")
            self._check_tensor(phi, "phi")
            self._check_tensor(pi, "pi", want_cuda=phi.is_cuda)
            fn = lib().pycool_set_fields_device if phi.is_cuda else lib().pycool_set_fields
            self._chk(fn(self._h, phi.data_ptr(), pi.data_ptr()))
            return
        phi, pi = self._host(phi), self._host(pi)
        self._chk(lib().pycool_set_fields(self._h, phi.ctypes.data, pi.ctypes.data))

    def init_fields(self, seed, phi_spec, pi_spec):
        """Seeded Gaussian initial conditions generated on the device.  *_spec: per field (mean, amp, m2, q, kmax),
        spectrum A(k) = amp (k^2 + m2)^q for k <= kmax (kmax <= 0: all k); see pycool_init_fields."""
        if len(phi_spec) != self.nf or len(pi_spec) != self.nf:
            raise PycoolError(EINVAL, "one spectrum per field is needed")
        a = (Spectrum * self.nf)(*[Spectrum(*map(float, t)) for t in phi_spec])
        b = (Spectrum * self.nf)(*[Spectrum(*map(float, t)) for t in pi_spec])
        self._chk(lib().pycool_init_fields(self._h, int(seed), a, b))

    def field_spectrum(self, field, which=0, nbins=None):
        """(power, count) per shell round(|n|) of phi (which = 0) or pi (1) of one field; see pycool_field_spectrum."""
        import numpy as np
        nbins = nbins or int(math.floor(math.sqrt(3.0) * self.N / 2.0 + 0.5)) + 1
        p, c = (C.c_double * nbins)(), (C.c_double * nbins)()
        self._chk(lib().pycool_field_spectrum(self._h, field, which, nbins, p, c))
        return np.array(p[:]), np.array(c[:])

    def mode_spectra(self, field, m_eff2, nbins=None):
        """(number, energy, count) per shell round(|n|) of one field; see pycool_mode_spectra (reading G24)."""
        nbins = nbins or int(math.floor(math.sqrt(3.0) * self.N / 2.0 + 0.5)) + 1
        n, e, c = (C.c_double * nbins)(), (C.c_double * nbins)(), (C.c_double * nbins)()
        self._chk(lib().pycool_mode_spectra(self._h, field, float(m_eff2), nbins, n, e, c))
        return np.array(n[:]), np.array(e[:]), np.array(c[:])

    def set_energy_cadence(self, every, capacity=1024):
        """Log the energies on the device after every `every`-th step (0: off); see pycool_set_energy_cadence."""
        self._chk(lib().pycool_set_energy_cadence(self._h, int(every), int(capacity)))

    def read_energy_log(self, max_entries=1 << 20):
        """(list of Energy, oldest first; total number logged since the cadence was set)."""
        n, total = C.c_int(), C.c_ulonglong()
        self._chk(lib().pycool_read_energy_log(self._h, None, 0, C.byref(n), C.byref(total)))
        have = min(int(total.value), max_entries)
        buf = (Energy * max(have, 1))()
        self._chk(lib().pycool_read_energy_log(self._h, buf, have, C.byref(n), C.byref(total)))
        return [buf[i] for i in range(n.value)], int(total.value)

    def set_background(self, a=1.0, p_a=math.nan):
        self._chk(lib().pycool_set_background(self._h, a, p_a))

    def set_dt(self, dt):
        self._chk(lib().pycool_set_dt(self._h, dt))

    def step(self, n=1):
        self._chk(lib().pycool_step(self._h, n))

    def sync(self):
        self._chk(lib().pycool_sync(self._h))

    def read_fields(self, out_phi=None, out_pi=None):
        """Download to new numpy arrays, or into given host buffers (numpy or pinned torch CPU tensors)."""
        shape = (self.nf, self.N, self.N, self.N)
        out = []
        for name, buf in (("out_phi", out_phi), ("out_pi", out_pi)):
            if buf is None:
                buf = np.empty(shape, self._np)
            elif isinstance(buf, self._torch.Tensor):
                self._check_tensor(buf, name, want_cuda=False)
            elif not (isinstance(buf, np.ndarray) and buf.dtype == self._np and buf.size == self.nf * self.N ** 3
                      and buf.flags["C_CONTIGUOUS"] and buf.flags["WRITEABLE"]):
                raise PycoolError(EINVAL, "%s must be a writable C-contiguous %s array of %d elements"
                                  % (name, np.dtype(self._np).name, self.nf * self.N ** 3))
            out.append(buf)
        phi, pi = out
        ptr = lambda t: t.data_ptr() if isinstance(t, self._torch.Tensor) else t.ctypes.data
        self._chk(lib().pycool_read_fields(self._h, ptr(phi), ptr(pi)))
        return phi, pi

    def read_fields_device(self):
        """(phi, pi) as new dense torch tensors [nf,N,N,N] on the device (D2D copy on the context stream)."""
        torch = self._torch
        shape = (self.nf, self.N, self.N, self.N)
        phi = torch.empty(shape, dtype=self._tdtype, device=self.device)
        pi = torch.empty(shape, dtype=self._tdtype, device=self.device)
        self._chk(lib().pycool_read_fields_device(self._h, phi.data_ptr(), pi.data_ptr()))
        return phi, pi

    def device_fields(self):
        """(phi, pi) as strided torch views [nf,N,N,N] of the CURRENT state buffers inside the work tensor (no
        copy, no sync): the library's padded layout with the ghost columns/rows sliced away."""
        a, b, lay = C.c_void_p(), C.c_void_p(), (C.c_size_t * 4)()
        self._chk(lib().pycool_device_fields(self._h, C.byref(a), C.byref(b), lay))
        pitch, rows, gx, gy = (int(v) for v in lay)
        return self._view(a.value, pitch, rows, gx, gy), self._view(b.value, pitch, rows, gx, gy)

    def _view(self, ptr, pitch, rows, gx, gy):
        n = self.nf * self.N * rows * pitch
        esize = 4 if self.precision == 32 else 8
        off = ptr - self._work.data_ptr()
        assert 0 <= off and off + n * esize <= self._work.numel()
        full = self._work[off:off + n * esize].view(self._tdtype).view(self.nf, self.N, rows, pitch)
        return full[:, :, gy:gy + self.N, gx:gx + self.N]

    def energies(self):
        e = Energy()
        self._chk(lib().pycool_energies(self._h, C.byref(e)))
        return e

    def launch_counts(self):
        c = (C.c_ulonglong * 4)()
        self._chk(lib().pycool_launch_counts(self._h, c))
        return [int(x) for x in c]

    def set_profiling(self, on=True):
        self._chk(lib().pycool_set_profiling(self._h, int(on)))

    def kick_time_ms(self):
        ms, n = C.c_double(), C.c_ulonglong()
        self._chk(lib().pycool_kick_time_ms(self._h, C.byref(ms), C.byref(n)))
        return ms.value, int(n.value)

    def kick_geometry(self):
        t = (C.c_int * 10)()
        self._chk(lib().pycool_kick_geometry(self._h, t))
        return dict(tx=t[0], ty=t[1], zchunk=t[2], threads=t[3], blocks=t[4], items=t[4], smem_bytes=t[5], variant=t[6],
                    tma_stages=t[7], region=(t[8], t[9]))

    def set_zchunk(self, planes):
        self._chk(lib().pycool_set_zchunk(self._h, planes))

    def set_adaptive(self, on=True):
        """dt becomes a physical-time increment: step n has conformal length dt / a_n."""
        self._chk(lib().pycool_set_adaptive(self._h, 1 if on else 0))

    def set_overlap(self, on=True):
        self._chk(lib().pycool_set_overlap(self._h, 1 if on else 0))

    def set_item_order(self, tiles_per_region=-1):
        """-1: automatic regions; 0: plain x-y-z order; n: regions of about n tiles (pycool_set_item_order)."""
        self._chk(lib().pycool_set_item_order(self._h, int(tiles_per_region)))

    def set_energy_kernel(self, tma=True):
        self._chk(lib().pycool_set_energy_kernel(self._h, 1 if tma else 0))

    def flush(self):
        """Apply the deferred closing half drift of the last step call now (asynchronous)."""
        self._chk(lib().pycool_flush(self._h))

    def set_persistent(self, on):
        self._chk(lib().pycool_set_persistent(self._h, 1 if on else 0))

    def set_cooperative(self, on):
        """Small lattices: several stages per cooperative launch (pycool_set_cooperative)."""
        self._chk(lib().pycool_set_cooperative(self._h, 1 if on else 0))

    def set_fused_tail(self, on):
        self._chk(lib().pycool_set_fused_tail(self._h, 1 if on else 0))

    def set_tile(self, tile):
        self._chk(lib().pycool_set_tile(self._h, tile))

    def close(self):
        if self._h:
            lib().pycool_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class LinearLattice:
    """The linearised solver (include/pycool_linear.h): homogeneous background + Fourier-space perturbations on a CUDA
    device, double precision.  Same call names as the C ABI; the library owns its device memory and stream."""

    def __init__(self, N, L, nfields, model, p=(), order=4, dt=0.01, device=None, **kw):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1201_5029_b200 needs a CUDA device (no CPU fallback)")
        self.N, self.L, self.nf, self.order = N, L, nfields, order
        self.device = torch.device("cuda:0" if device is None else device)
        self._mp = make_params(model, p, **kw)
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            st = lib().pycool_linear_create(C.byref(self._h), N, L, nfields, C.byref(self._mp), order, dt)
        if st != OK:
            raise PycoolError(st, lib().pycool_linear_last_error(None).decode())
        self.nclasses = int(lib().pycool_linear_num_classes(N))

    def _chk(self, st):
        if st != OK:
            raise PycoolError(st, lib().pycool_linear_last_error(self._h).decode())

    def _real(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        if x.size != self.nf * self.N ** 3:
            raise PycoolError(EINVAL, "real-space buffer has %d elements" % x.size)
        return x

    def _modes_shape(self):
        return (self.nf, self.N, self.N, self.N // 2 + 1)

    def set_background(self, a, p_a, phi0, pi0):
        if len(phi0) != self.nf or len(pi0) != self.nf:
            raise PycoolError(EINVAL, "phi0 / pi0 need one value per field")
        u, v = (C.c_double * self.nf)(*map(float, phi0)), (C.c_double * self.nf)(*map(float, pi0))
        self._chk(lib().pycool_linear_set_background(self._h, float(a), float(p_a), u, v))

    def set_perturbations(self, dphi, dpi):
        dphi, dpi = self._real(dphi), self._real(dpi)
        self._chk(lib().pycool_linear_set_perturbations(self._h, dphi.ctypes.data, dpi.ctypes.data))

    def set_modes(self, dPhi, dPi):
        """Half spectra [nf, N, N, N/2+1] complex (plain DFT convention, numpy.fft.rfftn layout)."""
        a = np.ascontiguousarray(dPhi, dtype=np.complex128)
        b = np.ascontiguousarray(dPi, dtype=np.complex128)
        if a.shape != self._modes_shape() or b.shape != self._modes_shape():
            raise PycoolError(EINVAL, "half spectra must have shape %s" % (self._modes_shape(),))
        self._chk(lib().pycool_linear_set_modes(self._h, a.ctypes.data, b.ctypes.data))

    def step(self, n=1, method=GROWTH):
        self._chk(lib().pycool_linear_step(self._h, int(n), int(method)))

    def read_modes(self):
        a, b = np.empty(self._modes_shape(), np.complex128), np.empty(self._modes_shape(), np.complex128)
        self._chk(lib().pycool_linear_read_modes(self._h, a.ctypes.data, b.ctypes.data))
        return a, b

    def read_perturbations(self):
        shape = (self.nf, self.N, self.N, self.N)
        a, b = np.empty(shape, np.float64), np.empty(shape, np.float64)
        self._chk(lib().pycool_linear_read_perturbations(self._h, a.ctypes.data, b.ctypes.data))
        return a, b

    def background(self):
        out = LinearBackground()
        self._chk(lib().pycool_linear_background_state(self._h, C.byref(out)))
        return out

    def growth(self):
        """Growth matrices [classes, 2 nf, 2 nf] of the latest GROWTH step call."""
        M = np.empty((self.nclasses, 2 * self.nf, 2 * self.nf), np.float64)
        n = C.c_size_t()
        self._chk(lib().pycool_linear_growth(self._h, M.ctypes.data, self.nclasses, C.byref(n)))
        return M

    def time_ms(self):
        ms = (C.c_double * 3)()
        self._chk(lib().pycool_linear_time_ms(self._h, ms))
        return dict(background=ms[0], growth=ms[1], modes=ms[2])

    def close(self):
        if self._h:
            lib().pycool_linear_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


LINEAR_STATIC_MAX_STAGES = 4096      # PYCOOL_LINEAR_STATIC_MAX_STAGES of include/pycool_linear.h


def linear_growth_static(N, L, nfields, model, p, order, dt, nsteps, a, p_a, phi0, pi0, M_device, max_classes,
                         stream=0, **kw):
    """pycool_linear_growth_static: growth matrices of (2.51) into caller-owned device memory, no allocation on the
    way (scratch in a fixed device array of the library).  M_device: device address (int) of max_classes x (2 nf)^2
    doubles on the current device; stream: a cudaStream_t handle (int), 0 = the default stream.  Asynchronous."""
    if len(phi0) != nfields or len(pi0) != nfields:
        raise PycoolError(EINVAL, "phi0 / pi0 need one value per field")
    mp = make_params(model, p, **kw)
    u, v = (C.c_double * nfields)(*map(float, phi0)), (C.c_double * nfields)(*map(float, pi0))
    st = lib().pycool_linear_growth_static(N, L, nfields, C.byref(mp), order, dt, int(nsteps), float(a), float(p_a), u, v,
                                           C.c_void_p(int(M_device)), int(max_classes), C.c_void_p(int(stream)))
    if st != OK:
        raise PycoolError(st, lib().pycool_linear_static_last_error().decode())


def from_config(cfg, device=None, **over):
    """Lattice for a config dict of `inputs.CONFIGS` (parameters only; fields are set by the caller)."""
    kw = dict(mpl=cfg["mpl"], rho_gamma0=cfg["rho_gamma0"], rho_m0=cfg["rho_m0"])
    kw.update(over)
    order = kw.pop("order", cfg["order"])
    dt = kw.pop("dt", cfg["dt"])
    return Lattice(cfg["N"], cfg["L"], cfg["nfields"], cfg["model"], cfg["p"], order=order, dt=dt,
                   device=device, **kw)
