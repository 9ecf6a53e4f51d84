"""Oracle for the number-density and energy-density spectra.  TEST INFRASTRUCTURE ONLY.

The paper's post-processing writes "field, number density and energy density spectra that are used in LATTICEEASY"
 and defines none of them.  Reading G24: the spectra of the DISCRETE Hamiltonian (2.20)
the step integrates, per field f, at the current scale factor a,

  F^phi_k = L^1.5 / (sqrt 2 N^3) sum_x phi(x) exp(-2 pi i n.x/N),  F^pi_k likewise        (convention of reading G22)
  u_k = a F^phi_k,  v_k = F^pi_k / a        the canonical pair (a phi, pi / a): the comoving field and its momentum
  w_k^2 = k_eff^2(n) / dx^2 + a^2 m_eff^2   -k_eff^2 = eigenvalue of the stencil D of (2.7) on the mode n
                                            (PAPER.md:267-269), m_eff^2 given by the caller (e.g. d^2V/dphi^2 of
                                            the background)
  n_k   = 1/2 (w_k |u_k|^2 + |v_k|^2 / w_k)          occupation number of the mode
  rho_k = w_k n_k = 1/2 (|v_k|^2 + w_k^2 |u_k|^2)    comoving energy of the mode

summed over the shells round(|n|) = i of the full spectrum, next to the mode counts C_i.  With these definitions
  (2 / (a^4 L^3)) sum_i rho_i = K_f + Gr_f + 1/2 m_eff^2 <phi_f^2>                          exactly (Parseval),
K_f, Gr_f the kinetic and gradient energy densities of (2.16)-(2.17) -- the pin that ties the spectra to
`energies()`; a vacuum state made by the generator of oracle/ics.py (|phi_k|^2 = 1/(2 w_k)) has <n_k> = 1/2.
Modes with w_k^2 <= 0 (the zero mode of a massless field, tachyonic modes) carry n_k = 0 and rho_k = |v_k|^2/2 +
w_k^2 |u_k|^2 / 2 (the energy is defined for any sign, the occupation number is not).

Plain numpy, fp64; every mode of the FULL spectrum is visited (fftn, no half-spectrum weights), so the code can be
checked against the definitions by eye.  Shares no code with the CUDA path.
"""
import math

import numpy as np


def k_eff2(N, stencil):
    """k_eff^2(n) >= 0 on the full [iz][iy][ix] grid: minus the eigenvalue of (2.7) on exp(2 pi i n.x/N):
    -(c0 + 2 c1 (Cx + Cy + Cz) + 4 c2 (Cx Cy + Cy Cz + Cz Cx) + 8 c3 Cx Cy Cz),  C = cos(2 pi n / N)."""
    c0, c1, c2, c3 = stencil
    C = np.cos(2.0 * math.pi * np.arange(N) / N)
    Cz, Cy, Cx = C[:, None, None], C[None, :, None], C[None, None, :]
    return -(c0 + 2.0 * c1 * (Cx + Cy + Cz) + 4.0 * c2 * (Cx * Cy + Cy * Cz + Cz * Cx) + 8.0 * c3 * Cx * Cy * Cz)


def shells(N):
    """round(|n|) on the full grid, n_i = i for i <= N/2 else i - N."""
    n1 = np.arange(N)
    n1 = np.where(n1 <= N // 2, n1, n1 - N).astype(np.float64)
    n2 = (n1 * n1)[:, None, None] + (n1 * n1)[None, :, None] + (n1 * n1)[None, None, :]
    return np.floor(np.sqrt(n2) + 0.5).astype(np.int64)


def mode_spectra(phi, pi, L, a, m_eff2, stencil):
    """(number, energy, count) per shell i = 0 .. round(sqrt 3 N/2) for one field: arrays phi, pi of shape [N, N, N]
    (z, y, x)."""
    N = phi.shape[0]
    norm = L ** 1.5 / (math.sqrt(2.0) * N ** 3)
    u = a * norm * np.fft.fftn(np.asarray(phi, dtype=np.float64))
    v = norm * np.fft.fftn(np.asarray(pi, dtype=np.float64)) / a
    dx = L / N
    w2 = k_eff2(N, stencil) / (dx * dx) + a * a * m_eff2
    u2, v2 = np.abs(u) ** 2, np.abs(v) ** 2
    rho = 0.5 * (v2 + w2 * u2)
    ok = w2 > 0.0
    w = np.sqrt(np.where(ok, w2, 1.0))
    n = np.where(ok, 0.5 * (w * u2 + v2 / w), 0.0)
    sh = shells(N).ravel()
    nb = int(math.floor(math.sqrt(3.0) * N / 2.0 + 0.5)) + 1
    number = np.bincount(sh, weights=n.ravel(), minlength=nb)[:nb]
    energy = np.bincount(sh, weights=rho.ravel(), minlength=nb)[:nb]
    count = np.bincount(sh, minlength=nb)[:nb].astype(np.float64)
    return number, energy, count
