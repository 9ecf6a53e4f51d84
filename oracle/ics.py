"""Oracle for the seeded Gaussian initial conditions.  TEST INFRASTRUCTURE ONLY.

The paper takes its fluctuations from Defrost's generator without describing it (reading G14), so
the recipe is this repository's (reading G21), the one paper_1201_5029_b200/inputs.py has used on the
host all along, made reproducible on any machine by a counter-based generator:

  half-spectrum grid (iz, iy, ix), iz, iy in [0, N), ix in [0, N/2]; n = i if i <= N/2 else i - N; k = 2 pi |n| / L
  A(k) = amp (k^2 + m2)^q for 0 < k and (kmax <= 0 or k <= kmax), else 0
  (w0, w1, w2, w3) = Philox4x32-10(counter = (j_lo, j_hi, array_id, 0), key = (seed_lo, seed_hi)),
      j = (iz N + iy)(N/2 + 1) + ix
  u1 = (w0 + 1/2) 2^-32, u2 = (w1 + 1/2) 2^-32;  g1 + i g2 = sqrt(-2 ln u1) exp(2 pi i u2)      (Box-Muller)
  F_j = A(k) (g1 + i g2) / sqrt 2
  planes ix = 0 and ix = N/2 (their own mirror images under k -> -k): with the mirror (iz', iy') = (-iz, -iy) mod N,
      self-conjugate modes take F = A g1 (real); of a mirror pair the lexicographically larger (iz, iy) takes
      conj F(mirror), so the spectrum is Hermitian and the field real
  field(x) = mean + sqrt 2 / L^(3/2) sum_k F_k exp(+2 pi i n.x / N)  =  mean + irfftn(F) sqrt 2 N^3 / L^1.5

Plain numpy, fp64; the FFT is numpy's.  Shares no code with the CUDA path (which has its own Philox, Box-Muller
and fill kernel and calls cuFFT).
"""
import math

import numpy as np

_M0, _M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_W0, _W1 = np.uint32(0x9E3779B9), np.uint32(0xBB67AE85)
_MASK = np.uint64(0xFFFFFFFF)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Philox4x32 with 10 rounds (Salmon et al., SC'11).  Arrays (or scalars) of uint32 in, four uint32 arrays out."""
    c0, c1, c2, c3 = (np.asarray(v, dtype=np.uint32).copy() for v in np.broadcast_arrays(c0, c1, c2, c3))
    k0 = np.uint32(k0)
    k1 = np.uint32(k1)
    with np.errstate(over="ignore"):
        for r in range(10):
            if r > 0:
                k0 = np.uint32((int(k0) + int(_W0)) & 0xFFFFFFFF)
                k1 = np.uint32((int(k1) + int(_W1)) & 0xFFFFFFFF)
            p0 = _M0 * c0.astype(np.uint64)
            p1 = _M1 * c2.astype(np.uint64)
            hi0, lo0 = (p0 >> np.uint64(32)).astype(np.uint32), (p0 & _MASK).astype(np.uint32)
            hi1, lo1 = (p1 >> np.uint64(32)).astype(np.uint32), (p1 & _MASK).astype(np.uint32)
            c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
    return c0, c1, c2, c3


def _gaussians(j, array_id, seed):
    """(g1, g2) of mode index j (uint64 array)."""
    j = np.asarray(j, dtype=np.uint64)
    w0, w1, _, _ = philox4x32_10((j & _MASK).astype(np.uint32), (j >> np.uint64(32)).astype(np.uint32),
                                 np.uint32(array_id), np.uint32(0), seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)
    u1 = (w0.astype(np.float64) + 0.5) * 2.0 ** -32
    u2 = (w1.astype(np.float64) + 0.5) * 2.0 ** -32
    r = np.sqrt(-2.0 * np.log(u1))
    return r * np.cos(2.0 * math.pi * u2), r * np.sin(2.0 * math.pi * u2)


def amplitude(N, L, amp, m2, q, kmax):
    """A(k) on the half-spectrum grid [iz][iy][ix]."""
    n1 = np.arange(N)
    n1 = np.where(n1 <= N // 2, n1, n1 - N).astype(np.float64)
    nx = np.arange(N // 2 + 1, dtype=np.float64)
    n2 = (n1 * n1)[:, None, None] + (n1 * n1)[None, :, None] + (nx * nx)[None, None, :]
    k = (2.0 * math.pi / L) * np.sqrt(n2)
    A = amp * np.power(k * k + m2, q, where=(n2 > 0) | (m2 > 0), out=np.zeros_like(k))
    A[n2 == 0] = 0.0
    if kmax > 0:
        A[k > kmax] = 0.0
    return A


def spectrum(N, L, seed, array_id, amp, m2, q, kmax):
    """The Hermitian half-spectrum F[iz][iy][ix] (complex128)."""
    assert N % 2 == 0
    H = N // 2 + 1
    iz, iy, ix = np.meshgrid(np.arange(N, dtype=np.uint64), np.arange(N, dtype=np.uint64),
                             np.arange(H, dtype=np.uint64), indexing="ij")
    j = (iz * np.uint64(N) + iy) * np.uint64(H) + ix
    A = amplitude(N, L, amp, m2, q, kmax)
    g1, g2 = _gaussians(j, array_id, seed)
    F = A * (g1 + 1j * g2) / math.sqrt(2.0)
    # planes that are their own mirror image under k -> -k
    mz, my = (np.uint64(N) - iz) % np.uint64(N), (np.uint64(N) - iy) % np.uint64(N)
    edge = (ix == 0) | (ix == np.uint64(N // 2))
    selfc = edge & (mz == iz) & (my == iy)
    F[selfc] = (A * g1)[selfc]
    later = edge & ~selfc & ((iz * np.uint64(N) + iy) > (mz * np.uint64(N) + my))
    jm = (mz * np.uint64(N) + my) * np.uint64(H) + ix
    h1, h2 = _gaussians(jm[later], array_id, seed)
    F[later] = A[later] * (h1 - 1j * h2) / math.sqrt(2.0)
    return F


def gaussian_field(N, L, seed, array_id, mean, amp, m2, q, kmax):
    """mean + the real Gaussian random field with spectrum A(k), shape [N, N, N] (z, y, x), fp64."""
    F = spectrum(N, L, seed, array_id, amp, m2, q, kmax)
    return mean + np.fft.irfftn(F, s=(N, N, N), axes=(0, 1, 2)) * (math.sqrt(2.0) * N ** 3 / L ** 1.5)


def init_fields(N, L, nf, seed, phi_spec, pi_spec):
    """(phi, pi) as [nf, N, N, N]; *_spec: per field (mean, amp, m2, q, kmax); array_id = 2 f (phi), 2 f + 1 (pi)."""
    phi = np.stack([gaussian_field(N, L, seed, 2 * f, *phi_spec[f]) for f in range(nf)])
    pi = np.stack([gaussian_field(N, L, seed, 2 * f + 1, *pi_spec[f]) for f in range(nf)])
    return phi, pi


def shell_spectrum(field, L):
    """Shell-summed field spectrum (reading G22): with the generator's convention
    turned around, F_k = L^1.5 / (sqrt 2 N^3) sum_x field(x) exp(-2 pi i n.x / N), returns (S, C) with
    S[i] = sum of |F_k|^2 and C[i] = number of modes over the FULL spectrum with round(|n|) = i,
    i = 0 .. round(sqrt 3 N / 2).  A field made with spectrum A(k) has <S[i] / C[i]> = A(k_i)^2."""
    N = field.shape[0]
    F = np.fft.rfftn(np.asarray(field, dtype=np.float64), axes=(0, 1, 2)) * (L ** 1.5 / (math.sqrt(2.0) * N ** 3))
    n1 = np.arange(N)
    n1 = np.where(n1 <= N // 2, n1, n1 - N).astype(np.float64)
    nx = np.arange(N // 2 + 1, dtype=np.float64)
    n2 = (n1 * n1)[:, None, None] + (n1 * n1)[None, :, None] + (nx * nx)[None, None, :]
    shell = np.floor(np.sqrt(n2) + 0.5).astype(np.int64)
    w = np.full(F.shape, 2.0)
    w[:, :, 0] = 1.0
    if N % 2 == 0:
        w[:, :, N // 2] = 1.0
    nb = int(math.floor(math.sqrt(3.0) * N / 2.0 + 0.5)) + 1
    S = np.bincount(shell.ravel(), weights=(w * np.abs(F) ** 2).ravel(), minlength=nb)[:nb]
    C = np.bincount(shell.ravel(), weights=w.ravel(), minlength=nb)[:nb]
    return S, C
