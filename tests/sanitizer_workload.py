"""Small cases of every kernel of libpycool.so for compute-sanitizer: not a test, a workload.

    compute-sanitizer --tool memcheck|racecheck|initcheck python tests/sanitizer_workload.py

What it runs (each a few launches, lattices small enough for the sanitizer's 10-100x slow-down): the persistent TMA
kernel with several work items per block, short z-chunks, ragged tiles and the programmatic launch overlap on, in its
variants 3 (64 x 16), 4 (32 x 16), 5 (128 x 8, fp32), 7 (2 x 1 sites, Q-ball), 9 (2 x 4 sites, one field); the
register-prefetch kernel (odd N); the fused stage tail (last-block reduction); the deferred closing drift; both energy
kernels and the energy log; seeded initial conditions and the spectra (cuFFT); the linearised solver.
Prints one line per case; exits non-zero if a call fails.
"""
import math
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from paper_1201_5029_b200 import binding as pc, build, inputs   # noqa: E402


def lattice_case(name, N, tile, zc, precision=64, order=2, steps=2):
    cfg = inputs.config(name, N=N, order=order)
    if name != "cfg0_chaotic32":
        cfg["L"] = cfg["L"] * N / inputs.config(name)["N"]
    else:
        cfg["dt"] = 0.0025
    phi, pi = inputs.make_initial(cfg, precision=precision)
    g = pc.from_config(cfg, precision=precision)
    if tile >= 0:
        g.set_tile(tile)
    if zc > 0:
        g.set_zchunk(zc)
    g.set_fields(phi, pi)
    g.set_background(1.0)
    g.set_energy_cadence(1, 4)
    g.step(steps)
    g.step(1)
    e = g.energies()
    g.set_energy_kernel(False)
    e2 = g.energies()
    log, total = g.read_energy_log()
    g.read_fields()
    geo = g.kick_geometry()
    assert math.isfinite(e.rho) and math.isfinite(e2.rho) and total == steps + 1
    print("%-18s N %3d fp%d variant %d zc %2d items %4d: a = %.9f, residual %.2e" %
          (name, N, precision, geo["variant"], geo["zchunk"], geo["items"], e.a, e.residual), flush=True)
    g.close()


def main():
    build.build()
    lattice_case("cfg0_chaotic32", 72, 3, 5)            # 64 x 16 tile, ragged in x and y, 15 chunks
    lattice_case("cfg0_chaotic32", 40, 4, 3, order=4, steps=1)
    lattice_case("cfg0_chaotic32", 72, 5, 7, precision=32)
    lattice_case("cfg3_qball256", 40, 7, 3)
    lattice_case("cfg2_oscillon256", 130, 9, 9, steps=1)
    lattice_case("cfg0_chaotic32", 21, -1, 0)           # odd N: register-prefetch kernel, plain energy kernel
    # seeded initial conditions and spectra
    cfg = inputs.config("cfg0_chaotic32", N=24, dt=0.0025)
    g = pc.from_config(cfg)
    g.init_fields(7, *inputs.spectra(cfg))
    g.set_background(1.0)
    g.step(1)
    p, c = g.field_spectrum(0, 0)
    n, e, c2 = g.mode_spectra(1, 1.0)
    assert np.all(np.isfinite(p)) and np.all(np.isfinite(n)) and c.sum() == 24 ** 3
    print("init_fields + spectra N 24: %d shells" % len(c), flush=True)
    g.close()
    # linearised solver, both methods
    for method in (pc.GROWTH, pc.NAIVE):
        lin = pc.LinearLattice(10, 4.0, 2, pc.CHAOTIC, (1.0, 1.0e4), order=4, dt=0.005)
        lin.set_background(1.0, math.nan, (0.9676, 1e-3), (-0.71, 2e-3))
        rng = np.random.default_rng(1)
        lin.set_perturbations(1e-3 * rng.standard_normal((2, 10, 10, 10)), 1e-3 * rng.standard_normal((2, 10, 10, 10)))
        lin.step(30, method)
        P, Q = lin.read_modes()
        a, b = lin.read_perturbations()
        assert np.all(np.isfinite(P)) and np.all(np.isfinite(a))
        print("linear method %d N 10: a = %.9f" % (method, lin.background().a), flush=True)
        lin.close()
    print("sanitizer workload done", flush=True)


if __name__ == "__main__":
    main()
