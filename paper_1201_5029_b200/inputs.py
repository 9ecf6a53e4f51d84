"""Seeded synthetic workloads shaped like the paper's three test models (arXiv 1201.5029 §3.1-3.3).

This module serves BOTH the CUDA path and the CPU oracle (tests, bench, smoke) and therefore holds none of
the method's arithmetic: no stencil, no potential, no integrator -- only parameter tables and random
initial lattices.  It imports numpy/scipy only (neither `oracle` nor the CUDA binding).

The paper's own initial conditions come from a Defrost-style generator that it does not describe
 and its lattices are not shipped, so these inputs stand in for them: same lattice shapes,
field counts, potentials, parameter magnitudes and fluctuation amplitudes (recipe: DESIGN.md "Inputs",
SURVEY.md 8(d)).  Everything is reproducible from `seed` via numpy's PCG64.
"""
import math

import numpy as np

try:  # multi-threaded FFT when available; numpy's otherwise (same values to rounding, both seeded)
    from scipy import fft as _fft
    _FFT_KW = {"workers": -1}
except Exception:  # pragma: no cover
    from numpy import fft as _fft
    _FFT_KW = {}

# model ids of the C ABI (the CUDA library's header and the CPU checker's header each declare these values)
FREE, CHAOTIC, OSCILLON, QBALL = 0, 1, 2, 3

# Chaotic model in program units (time, length in 1/m; fields in m_pl): PAPER.md:427-432, readings G11/G12/G19
_PHI0_BASELINE = 0.193 * math.sqrt(8.0 * math.pi)   # BASELINE.json configs[0]: 0.193 M_pl (non-reduced)
_PHIDOT0 = -0.71371                                 # from PAPER.md:432 via the constraint (G11)
_MPL_QBALL = 9.47e8                                 # m_pl / Phi_0
_H0_QBALL = 0.005                                   # radiation era at t = 100/m_sigma


def _chaotic(N, order, steps, seed, dt=None):
    L = 10.0
    return dict(model=CHAOTIC, N=N, L=L, nfields=2, p=(1.0, 1.0e4), mpl=1.0, rho_gamma0=0.0, rho_m0=0.0,
                order=order, steps=steps, dt=(L / N / 20.0 if dt is None else dt), seed=seed,
                init="vacuum", phi0=(_PHI0_BASELINE, 0.0), phidot0=(_PHIDOT0, 0.0), amp=5.0e-6)


CONFIGS = {
    # BASELINE.json configs[0..4]; see DESIGN.md for what was chosen where BASELINE/paper are silent
    "cfg0_chaotic32": _chaotic(32, 4, 100, seed=1),
    "cfg0b_chaotic32_resolved": _chaotic(32, 4, 100, seed=1, dt=0.0025),
    "cfg1_chaotic128": _chaotic(128, 6, 1000, seed=2),
    "cfg2_oscillon256": dict(model=OSCILLON, N=256, L=400.0, nfields=1, p=(1.0, 1.0, 0.3), mpl=335.41,
                             rho_gamma0=0.0, rho_m0=0.0, order=4, steps=2000, dt=0.005, seed=3,
                             init="flat", phi0=(2.0,), phidot0=(0.0,), amp=1.0e-3, kmax=1.0),
    "cfg3_qball256": dict(model=QBALL, N=256, L=8.0, nfields=2, p=(1.0, -0.1, 1.0, 0.0), mpl=_MPL_QBALL,
                          rho_gamma0=3.0 * _MPL_QBALL ** 2 * _H0_QBALL ** 2 - 1.25, rho_m0=0.0,
                          order=4, steps=2000, dt=0.005, seed=4, init="white",
                          phi0=(math.sqrt(2.0), 0.0), phidot0=(0.0, 0.5 * math.sqrt(2.0)), amp=1.0e-4),
    "cfg4_chaotic512": _chaotic(512, 4, 50, seed=5),
    "cfg4_chaotic1024": _chaotic(1024, 4, 50, seed=5),
}


def config(name, **over):
    """A copy of CONFIGS[name] with overrides (N=..., order=..., steps=..., dt=...).  Overriding N for a
    chaotic config keeps dt = L/N/20 unless dt is given too."""
    c = dict(CONFIGS[name])
    if "N" in over and "dt" not in over and c["model"] == CHAOTIC and c["dt"] == c["L"] / c["N"] / 20.0:
        c["dt"] = c["L"] / over["N"] / 20.0
    c.update(over)
    return c


def _kgrid_half(N, L):
    """|k| on the rfftn half-spectrum grid, k = 2 pi n / L, n_i in (-N/2, N/2]."""
    kf = 2.0 * math.pi / L
    k1 = np.fft.fftfreq(N, d=1.0 / N) * kf
    kz = np.fft.rfftfreq(N, d=1.0 / N) * kf
    k2 = (k1 * k1)[:, None, None] + (k1 * k1)[None, :, None] + (kz * kz)[None, None, :]
    return np.sqrt(k2)


def gaussian_field(N, L, amplitude_of_k, rng):
    """Real Gaussian random field with spectrum A(k): F_k = A(k) (g1 + i g2)/sqrt 2,
    delta = irfftn(F) * sqrt 2 * N^3 / L^1.5, zero mode removed (SURVEY.md 8(d) recipe)."""
    k = _kgrid_half(N, L)
    A = amplitude_of_k(k)
    A[0, 0, 0] = 0.0
    shape = A.shape
    F = np.empty(shape, np.complex128)
    F.real = rng.standard_normal(shape)
    F.imag = rng.standard_normal(shape)
    F *= A / math.sqrt(2.0)
    out = _fft.irfftn(F, s=(N, N, N), **_FFT_KW)
    out *= math.sqrt(2.0) * N ** 3 / L ** 1.5
    return out


def _tile(small, N):
    """Periodic replication of an n^3 realisation to N^3 (throughput-only lattices, N > 256)."""
    r = N // small.shape[0]
    return np.tile(small, (r, r, r))


def make_initial(cfg, precision=64, fft_max=256):
    """(phi, pi) as [nfields, N, N, N] arrays (x fastest) for a config dict, with a = 1 so pi = phi'.

    init = "vacuum": |delta phi_k|^2 = amp^2/(2 w_k), w_k^2 = k^2 + m_eff^2 and delta pi_k = w_k-weighted
                     independent draw (BASELINE.json configs[0]); m_eff^2 = m^2 for phi, g^2 phi0^2 for chi.
           "flat":   flat spectrum for k <= kmax, normalised to rms = amp (configs[2]); pi fluctuations 0.
           "white":  white noise of rms amp on every array (configs[3]).
    Lattices larger than fft_max are built from an fft_max^3 realisation replicated periodically (the
    host FFT of 2^27..2^30 points is too slow for a bench run; throughput does not depend on the values).
    """
    N, L, nf = cfg["N"], cfg["L"], cfg["nfields"]
    rng = np.random.default_rng(cfg["seed"])
    n_gen = N if (N <= fft_max or N % fft_max) else fft_max
    L_gen = L * n_gen / N
    dtype = np.float32 if precision == 32 else np.float64
    phi = np.empty((nf, N, N, N), dtype)
    pi = np.empty((nf, N, N, N), dtype)
    for f in range(nf):
        if cfg["init"] == "vacuum":
            meff2 = cfg["p"][0] if f == 0 else cfg["p"][1] * cfg["phi0"][0] ** 2
            amp = cfg["amp"]
            dphi = gaussian_field(n_gen, L_gen, lambda k: amp / np.sqrt(2.0 * np.sqrt(k * k + meff2)), rng)
            dpi = gaussian_field(n_gen, L_gen, lambda k: amp * np.sqrt(np.sqrt(k * k + meff2) / 2.0), rng)
        elif cfg["init"] == "flat":
            kmax = cfg["kmax"]
            dphi = gaussian_field(n_gen, L_gen, lambda k: (k <= kmax).astype(np.float64), rng)
            s = dphi.std()
            dphi *= cfg["amp"] / (s if s > 0 else 1.0)
            dpi = np.zeros_like(dphi)
        elif cfg["init"] == "white":
            dphi = cfg["amp"] * rng.standard_normal((n_gen,) * 3)
            dpi = cfg["amp"] * rng.standard_normal((n_gen,) * 3)
        else:
            raise ValueError("unknown init %r" % (cfg["init"],))
        if n_gen != N:
            dphi, dpi = _tile(dphi, N), _tile(dpi, N)
        phi[f] = cfg["phi0"][f] + dphi
        pi[f] = cfg["phidot0"][f] + dpi
    return phi, pi


def spectra(cfg):
    """The same workloads as spectrum parameters for the on-device generator (pycool_init_fields) and its oracle
    (oracle/ics.py): per field (mean, amp, m2, q, kmax) with A(k) = amp (k^2 + m2)^q for 0 < k <= kmax.
      vacuum: A_phi = c/sqrt(2 w_k) = (c/sqrt 2)(k^2 + m_eff^2)^(-1/4), A_pi = (c/sqrt 2)(k^2 + m_eff^2)^(+1/4);
      flat / white: constant A, normalised so that the EXPECTED rms is cfg["amp"]: var = 2 A^2 M / L^3 with M the
      number of modes 0 < k <= kmax (white: all N^3 - 1)."""
    N, L, nf = cfg["N"], cfg["L"], cfg["nfields"]
    phi_spec, pi_spec = [], []
    for f in range(nf):
        if cfg["init"] == "vacuum":
            meff2 = cfg["p"][0] if f == 0 else cfg["p"][1] * cfg["phi0"][0] ** 2
            c = cfg["amp"] / math.sqrt(2.0)
            phi_spec.append((cfg["phi0"][f], c, meff2, -0.25, 0.0))
            pi_spec.append((cfg["phidot0"][f], c, meff2, 0.25, 0.0))
        elif cfg["init"] in ("flat", "white"):
            kmax = cfg["kmax"] if cfg["init"] == "flat" else 0.0
            n1 = np.fft.fftfreq(N, d=1.0 / N)
            n2 = (n1 * n1)[:, None, None] + (n1 * n1)[None, :, None] + (n1 * n1)[None, None, :]
            M = np.count_nonzero((n2 > 0) & ((kmax <= 0) | (2.0 * math.pi / L * np.sqrt(n2) <= kmax))) if N <= 256 else \
                (N ** 3 - 1 if kmax <= 0 else max(1, int(4.0 / 3.0 * math.pi * (kmax * L / (2.0 * math.pi)) ** 3)))
            A = cfg["amp"] * math.sqrt(L ** 3 / (2.0 * max(M, 1)))
            phi_spec.append((cfg["phi0"][f], A, 0.0, 0.0, kmax))
            pi_spec.append((cfg["phidot0"][f], A if cfg["init"] == "white" else 0.0, 0.0, 0.0, kmax))
        else:
            raise ValueError("unknown init %r" % (cfg["init"],))
    return phi_spec, pi_spec


def random_fields(N, nf, seed, mean=0.0, amp=1.0, precision=64):
    """Plain seeded N(mean, amp) lattices for unit tests of single operators."""
    rng = np.random.default_rng(seed)
    dtype = np.float32 if precision == 32 else np.float64
    phi = (mean + amp * rng.standard_normal((nf, N, N, N))).astype(dtype)
    pi = (amp * rng.standard_normal((nf, N, N, N))).astype(dtype)
    return phi, pi
