"""Pins for oracle/spectra.py (number- and energy-density spectra, reading G24) against what the
mathematics fixes: a single mode in closed form, Parseval's sum rule against the C++ oracle's energies(), the
generator's vacuum state, and the adiabatic invariance of n_k under the oracle's own time evolution."""
import math

import numpy as np
import pytest

from oracle import FREE, Oracle, ics, spectra

from helpers import DEFAULT_STENCIL, SEVEN_POINT, stencil_eigenvalue

INF = math.inf


def grid(N):
    return np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")      # z, y, x


@pytest.mark.parametrize("stencil", [DEFAULT_STENCIL, SEVEN_POINT])
@pytest.mark.parametrize("m", [(1, 0, 0), (0, 2, 1), (3, 3, 2), (0, 0, 5)])
def test_single_mode_closed_form(stencil, m):
    """phi = A cos(k.x + d1), pi = B cos(k.x + d2): |F_{+-k}|^2 = (L^3/2)(A/2)^2 each (as in the field-spectrum pin),
    so the shell round(|m|) holds n = 2 * 1/2 (w a^2 (L^3/2)(A/2)^2 + (L^3/2)(B/2)^2 / (a^2 w)), rho = w n, with
    w^2 = k_eff^2/dx^2 + a^2 m_eff^2 and k_eff^2 from the plane-wave eigenvalue (tests/helpers.py, P3)."""
    N, L, A, B, a, m2 = 12, 3.0, 0.7, 0.4, 1.7, 2.5
    z, y, x = grid(N)
    arg = 2 * np.pi * (m[0] * x + m[1] * y + m[2] * z) / N
    phi, pi = A * np.cos(arg + 0.3), B * np.cos(arg - 1.1)
    number, energy, count = spectra.mode_spectra(phi, pi, L, a, m2, stencil)
    w = math.sqrt(-stencil_eigenvalue(stencil, m, N) / (L / N) ** 2 + a * a * m2)
    P, Q = L ** 3 / 2 * (A / 2) ** 2, L ** 3 / 2 * (B / 2) ** 2
    want = w * a * a * P + Q / (a * a * w)
    i = int(math.floor(math.sqrt(sum(v * v for v in m)) + 0.5))
    assert abs(number[i] - want) < 1e-12 * want and abs(energy[i] - w * want) < 1e-12 * w * want
    assert np.all(np.delete(number, i) < 1e-22) and np.all(np.delete(energy, i) < 1e-22)
    assert count.sum() == N ** 3 and count[0] == 1 and count[1] == 18


@pytest.mark.parametrize("N,a", [(8, 1.0), (9, 1.6), (12, 0.7)])
def test_energy_spectrum_sums_to_the_oracles_energies(N, a):
    """(2/(a^4 L^3)) sum_i rho_i = K + Gr + <V> for a free field, K, Gr (in the phi D phi form (2.17)) and <V> =
    1/2 m^2 <phi^2> taken from the C++ oracle's energies(): ties the spectra to the energy densities of (2.16)."""
    L, m2 = 5.0, 1.3
    rng = np.random.default_rng(N)
    phi = 0.4 + 0.2 * rng.standard_normal((1, N, N, N))
    pi = 0.3 * rng.standard_normal((1, N, N, N))
    o = Oracle(N, L, 1, FREE, [m2], order=2, dt=0.01, mpl=1.0)
    o.set_fields(phi, pi)
    o.set_background(a, -1.0)
    e = o.energies()
    _, energy, _ = spectra.mode_spectra(phi[0], pi[0], L, a, m2, DEFAULT_STENCIL)
    total = 2.0 / (a ** 4 * L ** 3) * energy.sum()
    assert abs(total - (e.kin[0] + e.sum_phiDphi[0] + e.pot)) < 1e-12 * total
    assert abs(e.grad[0] - e.sum_phiDphi[0]) < 1e-11 * e.grad[0]                  # (2.17), so the G form as well


def test_vacuum_state_of_the_generator_has_half_a_quantum_per_mode():
    """|phi_k|^2 = c^2/(2 w_k), |pi_k|^2 = c^2 w_k/2 (oracle/ics.py with q = -+1/4, amp = c/sqrt 2) gives <n_k> = c^2/2;
    low shells, where the lattice k_eff and the generator's continuum k agree."""
    N, L, c, m2 = 32, 20.0, 0.3, 1.5
    phi, pi = ics.init_fields(N, L, 1, 7, [(0.0, c / math.sqrt(2), m2, -0.25, 0.0)], [(0.0, c / math.sqrt(2), m2, 0.25, 0.0)])
    number, energy, count = spectra.mode_spectra(phi[0], pi[0], L, 1.0, m2, DEFAULT_STENCIL)
    for i in (2, 4, 6):
        assert abs(number[i] / count[i] / (0.5 * c * c) - 1) < 5 / math.sqrt(count[i]) + 0.02
        k = 2 * math.pi / L * i
        assert abs(energy[i] / number[i] / math.sqrt(k * k + m2) - 1) < 0.1      # rho_k = w_k n_k, w ~ sqrt(k^2 + m^2)


@pytest.mark.parametrize("a", [1.0, 1.4])
def test_occupation_number_is_conserved_by_the_free_evolution(a):
    """A single lattice mode of a free field in a static background is a harmonic oscillator of frequency w_k in
    conformal time, w_k^2 = k_eff^2/dx^2 + a^2 m^2 (pinned for the stepper by P3), and n_k = E/w is its action: constant
    along the oracle's evolution up to the integrator's O(dt^4) -- but ONLY if w_k, the powers of a and the pairing
    of phi with pi are the right ones.  The mode (3,3,2) on N = 8 is far from the continuum (k_eff^2/dx^2 is 0.61 of
    k^2), so a spectrum built on the continuum k would swing by ~20 % over the oscillation; shown alongside."""
    N, L, m2, mode = 8, 4.0, 0.8, (3, 3, 2)
    z, y, x = grid(N)
    arg = 2 * np.pi * (mode[0] * x + mode[1] * y + mode[2] * z) / N
    phi, pi = (0.5 * np.cos(arg))[None], (0.1 * np.sin(arg))[None]
    o = Oracle(N, L, 1, FREE, [m2], order=4, dt=0.002, mpl=INF)     # (w dt)^4 ~ 1e-8
    o.set_fields(phi, pi)
    o.set_background(a, 0.0)
    i = int(math.floor(math.sqrt(sum(v * v for v in mode)) + 0.5))
    ns, wrong = [], []
    kc2 = (2 * math.pi / L) ** 2 * sum(v * v for v in mode)
    for _ in range(12):
        p, q = o.read_fields()
        number, _, _ = spectra.mode_spectra(p[0], q[0], L, a, m2, DEFAULT_STENCIL)
        ns.append(number[i])
        Fp = np.sum(np.abs(np.fft.fftn(p[0])) ** 2) * a * a
        Fq = np.sum(np.abs(np.fft.fftn(q[0])) ** 2) / (a * a)
        wc = math.sqrt(kc2 + a * a * m2)
        wrong.append(0.5 * (wc * Fp + Fq / wc))
        o.step(35)
    ns, wrong = np.array(ns), np.array(wrong)
    assert np.ptp(ns) < 1e-7 * ns.mean()
    assert np.ptp(wrong) > 0.05 * wrong.mean()
