"""Pins of the initial-condition oracle (oracle/ics.py, reading G21)."""
import math
import os

import numpy as np
import pytest

from oracle import ics


def test_philox_known_answers(golden_dir):
    """The three published Philox4x32-10 vectors (tests/golden/philox4x32_10_kat.txt)."""
    n = 0
    for line in open(os.path.join(golden_dir, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        out = ics.philox4x32_10(w[0], w[1], w[2], w[3], w[4], w[5])
        assert [int(v) for v in out] == w[6:10], line
        n += 1
    assert n == 3


def test_philox_is_a_bijection_on_counters_and_vectorises():
    """Distinct counters give distinct outputs (it is a permutation for a fixed key); the array form equals the
    scalar form element by element."""
    c0 = np.arange(5000, dtype=np.uint32)
    out = ics.philox4x32_10(c0, 7, 1, 0, 123, 456)
    packed = {tuple(int(o[i]) for o in out) for i in range(c0.size)}
    assert len(packed) == c0.size
    for i in (0, 17, 4999):
        one = ics.philox4x32_10(int(c0[i]), 7, 1, 0, 123, 456)
        assert [int(v) for v in one] == [int(o[i]) for o in out]


def test_box_muller_moments():
    g1, g2 = ics._gaussians(np.arange(400000, dtype=np.uint64), 3, 99)
    g = np.concatenate([g1, g2])
    assert abs(g.mean()) < 4 / math.sqrt(g.size) and abs(g.var() - 1) < 4 * math.sqrt(2 / g.size)
    assert abs(np.mean(g ** 4) - 3) < 0.05 and abs(np.mean(g1 * g2)) < 4 / math.sqrt(g1.size)
    assert np.isfinite(g).all() and np.abs(g).max() < 6.8          # 32-bit uniforms: |g| <= sqrt(2 ln 2^33)


@pytest.mark.parametrize("N", [8, 12])
def test_spectrum_is_hermitian_and_the_field_is_what_the_definition_says(N):
    """Full-spectrum brute force: expand the half-spectrum by F(-k) = conj F(k), check that the planes ix = 0 and
    ix = N/2 are consistent with it, and evaluate sum_k F_k exp(2 pi i n.x / N) directly (dense DFT matrices)."""
    L, seed = 3.0, 2024
    F = ics.spectrum(N, L, seed, 1, 0.7, 0.5, -0.25, 0.0)
    H = N // 2 + 1
    full = np.zeros((N, N, N), complex)
    full[:, :, :H] = F
    for iz in range(N):
        for iy in range(N):
            for ix in range(H, N):
                full[iz, iy, ix] = np.conj(F[(-iz) % N, (-iy) % N, N - ix])
            for ix in (0, N // 2):
                assert abs(F[iz, iy, ix] - np.conj(F[(-iz) % N, (-iy) % N, ix])) < 1e-15
    assert F[0, 0, 0] == 0 and abs(F[N // 2, 0, N // 2].imag) == 0
    W = np.exp(2j * np.pi * np.outer(np.arange(N), np.arange(N)) / N)
    direct = np.einsum("za,yb,xc,abc->zyx", W, W, W, full)
    assert np.abs(direct.imag).max() < 1e-12 * np.abs(direct.real).max()
    field = ics.gaussian_field(N, L, seed, 1, 2.5, 0.7, 0.5, -0.25, 0.0)
    want = 2.5 + direct.real * math.sqrt(2.0) / L ** 1.5
    assert np.abs(field - want).max() < 1e-12 * np.abs(want).max()
    assert abs(field.mean() - 2.5) < 1e-13                          # zero mode removed


def test_power_per_mode_and_real_space_variance():
    """<|F_k|^2> = A(k)^2 for every kind of mode (averaged over seeds), a cut at kmax, and Parseval:
    var(field) = (2 / L^3) sum over the FULL spectrum of |F_k|^2."""
    N, L = 8, 2.0
    amp, m2, q = 0.3, 1.5, 0.25
    A = ics.amplitude(N, L, amp, m2, q, 0.0)
    acc = np.zeros_like(A)
    ns = 600
    for s in range(ns):
        acc += np.abs(ics.spectrum(N, L, 1000 + s, 0, amp, m2, q, 0.0)) ** 2
    ratio = acc[A > 0] / ns / A[A > 0] ** 2
    assert abs(ratio.mean() - 1) < 0.01 and np.abs(ratio - 1).max() < 6 * math.sqrt(2.0 / ns)
    k1 = 2 * math.pi / L
    Acut = ics.amplitude(N, L, amp, m2, q, 2.5 * k1)
    n1 = np.where(np.arange(N) <= N // 2, np.arange(N), np.arange(N) - N)
    n2 = (n1 ** 2)[:, None, None] + (n1 ** 2)[None, :, None] + (np.arange(N // 2 + 1) ** 2)[None, None, :]
    assert np.all(Acut[n2 > 6.25] == 0) and np.all(Acut[(n2 > 0) & (n2 <= 6.25)] > 0)
    assert abs(A[1, 0, 0] - amp * (k1 ** 2 + m2) ** q) < 1e-15 and abs(A[0, N - 1, 1] - amp * (2 * k1 ** 2 + m2) ** q) < 1e-15
    F = ics.spectrum(N, L, 5, 2, amp, m2, q, 0.0)
    w = np.full(F.shape, 2.0)
    w[:, :, 0] = 1.0
    w[:, :, N // 2] = 1.0
    field = ics.gaussian_field(N, L, 5, 2, 0.0, amp, m2, q, 0.0)
    assert abs(field.var() - 2.0 / L ** 3 * np.sum(w * np.abs(F) ** 2)) < 1e-12 * field.var()


def test_arrays_and_seeds_are_independent_streams():
    a = ics.gaussian_field(8, 1.0, 1, 0, 0.0, 1.0, 1.0, 0.0, 0.0)
    b = ics.gaussian_field(8, 1.0, 1, 1, 0.0, 1.0, 1.0, 0.0, 0.0)
    c = ics.gaussian_field(8, 1.0, 2, 0, 0.0, 1.0, 1.0, 0.0, 0.0)
    assert abs(np.corrcoef(a.ravel(), b.ravel())[0, 1]) < 0.2 and abs(np.corrcoef(a.ravel(), c.ravel())[0, 1]) < 0.2
    assert np.array_equal(a, ics.gaussian_field(8, 1.0, 1, 0, 0.0, 1.0, 1.0, 0.0, 0.0))


# ---------------------------------------------------------------- shell spectrum (rank 3)
def test_shell_spectrum_of_a_single_mode_and_parseval():
    """A cos(2 pi m.x / N) has |F_{+-m}|^2 = (L^3/2)(A/2)^2 each: the shell round(|m|) holds L^3 A^2 / 4 and nothing
    else; counts: 1, 18 (|n|^2 = 1 and 2), ... and N^3 in total; Parseval: sum_i S_i = L^3 / (2 N^3) sum_x field^2."""
    N, L, A = 12, 3.0, 0.7
    rng = np.random.default_rng(0)
    z, y, x = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    for m in ((1, 0, 0), (0, 2, 1), (3, 3, 2), (0, 0, 5)):
        f = A * np.cos(2 * np.pi * (m[0] * x + m[1] * y + m[2] * z) / N + 0.3)
        S, C = ics.shell_spectrum(f, L)
        i = int(math.floor(math.sqrt(sum(v * v for v in m)) + 0.5))
        assert abs(S[i] - L ** 3 * A * A / 4) < 1e-12 * S[i]
        assert np.all(np.delete(S, i) < 1e-25)
    assert C[0] == 1 and C[1] == 6 + 12 and C.sum() == N ** 3 and len(C) == int(math.sqrt(3) * N / 2 + 0.5) + 1
    # The farthest mode sits at |n| = sqrt 3 N/2 (even N), so the last shell is round(sqrt 3 N/2), not
    # floor(sqrt 3 N/2): the two differ whenever frac(sqrt 3 N/2) >= 1/2 (N = 16: 13.86 -> 14 vs 13; N = 12 cannot
    # tell them apart).  A floor() binning would drop that shell and C.sum() would fall short of N^3.  Odd N: the
    # farthest mode is at sqrt 3 (N-1)/2, every mode must still land in a bin.
    for n in (16, 10, 9, 15):
        Sn, Cn = ics.shell_spectrum(rng.standard_normal((n, n, n)), L)
        far = math.sqrt(3) * (n // 2)
        assert len(Cn) == int(math.floor(math.sqrt(3) * n / 2 + 0.5)) + 1 and Cn.sum() == n ** 3, n
        assert Cn[int(math.floor(far + 0.5))] >= 1, n                           # the corner mode's own shell exists
    assert math.floor(math.sqrt(3) * 16 / 2) + 1 == 14 and len(ics.shell_spectrum(np.ones((16,) * 3), L)[1]) == 15
    f = rng.standard_normal((N, N, N)) + 0.4
    S, _ = ics.shell_spectrum(f, L)
    assert abs(S.sum() - L ** 3 / (2 * N ** 3) * np.sum(f * f)) < 1e-12 * S.sum()
    assert abs(S[0] - L ** 3 / 2 * f.mean() ** 2) < 1e-12 * S[0]


def test_shell_spectrum_returns_the_generators_spectrum():
    N, L, amp = 32, 5.0, 0.2
    f = ics.gaussian_field(N, L, 11, 0, 0.0, amp, 2.0, -0.25, 0.0)
    S, C = ics.shell_spectrum(f, L)
    for i in (3, 8, 14):
        k = 2 * math.pi / L * i
        want = amp ** 2 * (k * k + 2.0) ** -0.5
        assert abs(S[i] / C[i] / want - 1) < 6 / math.sqrt(C[i]) + 0.05      # shell width: k varies by +-1/(2i)
