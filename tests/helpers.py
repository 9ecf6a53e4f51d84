"""Test-side mathematics that is independent of both implementations.

Nothing here is imported by the oracle or by the CUDA path.  The closed forms below are what the paper and
textbook mathematics fix; they are written with numpy long doubles / rolls, i.e.
not in the way either implementation computes.
"""
import math
import os

import numpy as np

LD = np.longdouble


def golden_weights(golden_dir, order):
    """Full symmetric stage-weight list for order 6/8 from the decimals printed in Table 1, in long double."""
    half = []
    with open(os.path.join(golden_dir, "table1_weights.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            o, s, i, v = line.split()
            if int(o) == order:
                half.append(LD(v))
    last = LD(1) - LD(2) * sum(half, LD(0))
    half = half + [last]
    return half + half[-2::-1]


def yoshida_weights():
    """Triple-jump weights with the two defining conditions solved directly: 2 z1 + z0 = 1, 2 z1^3 + z0^3 = 0
    (reading G2)."""
    c = LD(2) ** (LD(1) / LD(3))
    z1 = LD(1) / (LD(2) - c)
    z0 = LD(1) - LD(2) * z1
    return [z1, z0, z1]


def weights(golden_dir, order):
    if order == 2:
        return [LD(1)]
    if order == 4:
        return yoshida_weights()
    return golden_weights(golden_dir, order)


def oscillator_map(w2, h):
    """Exact 2x2 map of drift(h/2) kick(h) drift(h/2) for q'' = -w2 q (static background, a = 1):
    [[1 - w2 h^2/2, h (1 - w2 h^2/4)], [-w2 h, 1 - w2 h^2/2]]."""
    w2, h = LD(w2), LD(h)
    return np.array([[1 - w2 * h * h / 2, h * (1 - w2 * h * h / 4)], [-w2 * h, 1 - w2 * h * h / 2]], dtype=LD)


def composed_map(w2, dt, ws):
    M = np.eye(2, dtype=LD)
    for w in ws:                      # stages applied in order; the list is palindromic anyway
        M = oscillator_map(w2, w * LD(dt)) @ M
    return M


def evolve_oscillator(w2, dt, ws, q0, p0, n):
    M = composed_map(w2, dt, ws)
    v = np.array([LD(q0), LD(p0)], dtype=LD)
    for _ in range(n):
        v = M @ v
    return float(v[0]), float(v[1])


def stencil_eigenvalue(c, n, N):
    """-k_eff^2 of the 27-point stencil (2.7) on the plane wave with integer wave vector n (P3)."""
    C = [math.cos(2.0 * math.pi * ni / N) for ni in n]
    return (c[0] + 2 * c[1] * (C[0] + C[1] + C[2]) + 4 * c[2] * (C[0] * C[1] + C[1] * C[2] + C[2] * C[0])
            + 8 * c[3] * C[0] * C[1] * C[2])


def laplacian_rolls(phi, c):
    """D[phi] of (2.7) straight from its definition (weight form) with modular indices via np.roll.
    phi: [N,N,N] indexed [z,y,x]."""
    out = np.zeros_like(phi, dtype=np.float64)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                d = (dx != 0) + (dy != 0) + (dz != 0)
                out += c[d] * np.roll(phi, (-dz, -dy, -dx), axis=(0, 1, 2))
    return out


def laplacian_dense(N, c):
    """(2.7) as a dense N^3 x N^3 matrix with explicitly modular indices (P10), row-major [z][y][x]."""
    V = N ** 3
    A = np.zeros((V, V))
    for z in range(N):
        for y in range(N):
            for x in range(N):
                r = (z * N + y) * N + x
                for dz in (-1, 0, 1):
                    for dy in (-1, 0, 1):
                        for dx in (-1, 0, 1):
                            d = (dx != 0) + (dy != 0) + (dz != 0)
                            col = (((z + dz) % N) * N + ((y + dy) % N)) * N + ((x + dx) % N)
                            A[r, col] += c[d]
    return A


DEFAULT_STENCIL = (-128.0 / 30.0, 14.0 / 30.0, 3.0 / 30.0, 1.0 / 30.0)
SEVEN_POINT = (-6.0, 1.0, 0.0, 0.0)


def rel_err_per_site(got, want):
    """Reading G18: max_x |got - want| / max(|want_x|, rms_x(want)) for each field array [f,...]."""
    got = np.asarray(got, np.float64)
    want = np.asarray(want, np.float64)
    worst = 0.0
    for f in range(want.shape[0]):
        rms = math.sqrt(float(np.mean(want[f] ** 2)))
        den = np.maximum(np.abs(want[f]), rms if rms > 0 else 1.0)
        worst = max(worst, float(np.max(np.abs(got[f] - want[f]) / den)))
    return worst
