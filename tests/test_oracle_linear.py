"""Pins for oracle/linear.py (the linearised solver) against what the
paper and the mathematics fix, none of them the oracle's own formulas retyped:
  L1  table of distinct k_eff^2 = the plane-wave eigenvalue of (2.7) (tests/helpers.py, P3) on every mode; the
      multiplicities add up to N^3; class count (M+1)(M+2)(M+3)/6
  L2  the growth matrices are symplectic: M^T J M = J (so det M = 1) -- (2.51) is the flow of a quadratic Hamiltonian
  L3  free field, static background: each mode is the oscillator of P2/P3, closed-form 2x2 map in long double
  L4  per-mode evolution == growth-matrix evolution, to rounding
  L5  the background equals the NON-linear oracle (oracle.cpp) run on a homogeneous lattice: (2.35)-(2.36) are (2.47)
      without gradients
  L6  small-amplitude limit: the non-linear oracle started from phi_0 + eps dphi differs from the linear solution by
      O(eps^2): halving eps quarters the difference
  L7  Hessians V_ij against central differences of the C++ oracle's dV/dphi (independent implementation)
  L8  measured convergence order 2 / 4 of the perturbation evolution in an expanding background
"""
import math

import numpy as np
import pytest

from oracle import CHAOTIC, FREE, OSCILLON, QBALL, Oracle, linear

from helpers import DEFAULT_STENCIL, LD, SEVEN_POINT, composed_map, stencil_eigenvalue, weights

INF = math.inf
CH = dict(model=CHAOTIC, p=(1.0, 1.0e4))


# ---------------------------------------------------------------- L1
@pytest.mark.parametrize("N", [4, 7, 8, 12])
@pytest.mark.parametrize("stencil", [DEFAULT_STENCIL, SEVEN_POINT])
def test_l1_distinct_k_eff2_table(N, stencil):
    triples, index, mult = linear.distinct_table(N)
    M = N // 2
    assert len(triples) == (M + 1) * (M + 2) * (M + 3) // 6 and mult.sum() == N ** 3 and mult[0] == 1
    k2 = linear.k_eff2_of(triples, N, stencil)
    for iz in range(N):
        for iy in range(N):
            for ix in range(N):
                want = -stencil_eigenvalue(stencil, (ix, iy, iz), N)
                assert abs(k2[index[iz, iy, ix]] - want) < 1e-13
    assert abs(k2[0]) < 1e-15 and np.all(k2[1:] > 0)
    if N % 2 == 0 and stencil is DEFAULT_STENCIL:
        assert abs(k2.max() - 92.0 / 15.0) < 1e-13                       # (pi, pi, pi), SURVEY P3


# ---------------------------------------------------------------- L2
@pytest.mark.parametrize("order", [2, 4, 6])
def test_l2_growth_matrices_are_symplectic(order):
    o = linear.LinearOracle(6, 2.0, 2, order=order, dt=0.01, mpl=1.0, **CH)
    o.set_background(1.0, math.nan, (0.9, 0.02), (-0.7, 0.01))
    M, _ = o.growth_matrices(5)
    J = np.zeros((4, 4))
    for i in range(2):
        J[2 * i, 2 * i + 1], J[2 * i + 1, 2 * i] = 1.0, -1.0
    for m in M:
        assert np.max(np.abs(m.T @ J @ m - J)) < 1e-11
        assert abs(np.linalg.det(m) - 1.0) < 1e-11
    assert np.max(np.abs(M[:, 0, 2])) > 1e-6                               # the two fields do couple (V_phi,chi != 0)


# ---------------------------------------------------------------- L3
@pytest.mark.parametrize("order", [2, 4, 6])
def test_l3_free_field_static_background_closed_form(order, golden_dir):
    N, L, m2, dt, n = 6, 3.0, 1.3, 0.02, 7
    o = linear.LinearOracle(N, L, 1, FREE, [m2], order=order, dt=dt, mpl=INF)
    o.set_background(1.0, 0.0, (0.3,), (0.0,))
    M, index = o.growth_matrices(n)
    triples, _, _ = linear.distinct_table(N)
    ws = weights(golden_dir, order)
    for t, tr in enumerate(triples):
        w2 = -stencil_eigenvalue(DEFAULT_STENCIL, tuple(int(v) for v in tr), N) / (L / N) ** 2 + m2
        one = composed_map(w2, dt, ws)
        want = np.eye(2, dtype=LD)
        for _ in range(n):
            want = one @ want
        assert np.max(np.abs(M[t] - want.astype(np.float64))) < 1e-13


# ---------------------------------------------------------------- L4
@pytest.mark.parametrize("model,nf,p,bg", [(CHAOTIC, 2, (1.0, 1.0e4), ((0.9, 0.01), (-0.7, 0.02))),
                                           (OSCILLON, 1, (1.0, 1.0, 0.3), ((0.8,), (0.1,))),
                                           (QBALL, 2, (1.0, -0.1, 1.0, 0.0), ((1.3, 0.2), (0.0, 0.6)))])
def test_l4_direct_equals_growth_matrix_evolution(model, nf, p, bg):
    N = 6
    rng = np.random.default_rng(3)
    dphi, dpi = rng.standard_normal((nf, N, N, N)), rng.standard_normal((nf, N, N, N))
    outs = []
    for growth in (False, True):
        o = linear.LinearOracle(N, 2.0, nf, model, p, order=4, dt=0.01, mpl=2.0)
        o.set_background(1.0, math.nan, *bg)
        o.set_perturbations(dphi, dpi)
        if growth:
            o.growth_step(3); o.growth_step(2)
        else:
            o.step(5)
        outs.append(o.read_perturbations() + (o.a, o.p_a, o.phi0[0]))
    scale = np.max(np.abs(outs[0][1]))
    assert np.max(np.abs(outs[0][0] - outs[1][0])) < 1e-12 * scale and np.max(np.abs(outs[0][1] - outs[1][1])) < 1e-12 * scale
    assert outs[0][2:] == outs[1][2:]
    assert abs(outs[0][0].mean()) < 1e-15                                 # k = 0 stays out (2.22)


# ---------------------------------------------------------------- L5
@pytest.mark.parametrize("order", [2, 4, 6])
def test_l5_background_equals_the_nonlinear_oracle_on_a_homogeneous_lattice(order):
    N, L, dt, n = 3, 2.0, 0.01, 20
    phi0, pi0 = (0.9, 0.05), (-0.7, 0.3)
    lo = linear.LinearOracle(N, L, 2, order=order, dt=dt, mpl=1.5, rho_gamma0=0.2, rho_m0=0.1, **CH)
    lo.set_background(1.0, math.nan, phi0, pi0)
    no = Oracle(N, L, 2, CHAOTIC, CH["p"], order=order, dt=dt, mpl=1.5, rho_gamma0=0.2, rho_m0=0.1)
    ones = np.ones((N, N, N))
    no.set_fields(np.stack([phi0[0] * ones, phi0[1] * ones]), np.stack([pi0[0] * ones, pi0[1] * ones]))
    no.set_background(1.0)
    e0 = no.energies()
    assert abs(lo.p_a - e0.p_a) < 1e-14 * abs(e0.p_a)
    lo.step(n); no.step(n)
    e = no.energies()
    p, q = no.read_fields()
    assert abs(lo.a - e.a) < 1e-14 and abs(lo.p_a - e.p_a) < 1e-13 * abs(e.p_a)
    for f in range(2):
        assert abs(lo.phi0[f] - p[f, 0, 0, 0]) < 1e-14 and abs(lo.pi0[f] - q[f, 1, 2, 0]) < 1e-13
    be = lo.background_energy()
    assert abs(be["rho"] - e.rho) < 1e-13 * e.rho and abs(be["hubble"] - e.hubble) < 1e-13 * e.hubble
    assert abs(be["residual"] - e.residual) < 1e-11                       # (3.1): the same number, whatever its size


# ---------------------------------------------------------------- L6
def test_l6_small_amplitude_limit_of_the_nonlinear_oracle():
    N, L, dt, n = 8, 4.0, 0.002, 25
    phi0, pi0 = (0.9, 0.0), (-0.7, 0.0)
    rng = np.random.default_rng(11)
    dphi, dpi = rng.standard_normal((2, N, N, N)), rng.standard_normal((2, N, N, N))
    dphi -= dphi.mean(axis=(1, 2, 3), keepdims=True)
    dpi -= dpi.mean(axis=(1, 2, 3), keepdims=True)
    lo = linear.LinearOracle(N, L, 2, order=4, dt=dt, mpl=1.0, **CH)
    lo.set_background(1.0, math.nan, phi0, pi0)
    pa0 = float(lo.p_a)
    lo.set_perturbations(dphi, dpi)
    lo.step(n)
    lphi, lpi = lo.read_perturbations()
    errs = []
    for eps in (2e-4, 1e-4):
        no = Oracle(N, L, 2, CHAOTIC, CH["p"], order=4, dt=dt, mpl=1.0)
        b = np.array(phi0)[:, None, None, None], np.array(pi0)[:, None, None, None]
        no.set_fields(b[0] + eps * dphi, b[1] + eps * dpi)
        no.set_background(1.0, pa0)
        no.step(n)
        p, q = no.read_fields()
        dp = (p - p.mean(axis=(1, 2, 3), keepdims=True)) / eps
        dq = (q - q.mean(axis=(1, 2, 3), keepdims=True)) / eps
        errs.append(max(np.max(np.abs(dp - lphi)), np.max(np.abs(dq - lpi)) / np.max(np.abs(lpi))))
        assert errs[-1] < 100 * eps                                        # relative difference O(eps)
    assert 1.7 < errs[0] / errs[1] < 2.3                                  # ... and it halves with eps


# ---------------------------------------------------------------- L7
@pytest.mark.parametrize("model,nf,p,pt", [(FREE, 3, (0.5, 1.5, 2.5), (0.3, -0.2, 0.7)), (CHAOTIC, 2, (1.0, 1.0e4), (0.9, 0.013)),
                                           (OSCILLON, 1, (1.0, 1.0, 0.3), (1.7,)), (QBALL, 2, (1.0, -0.1, 2.0, 0.4), (1.3, -0.4))])
def test_l7_hessian_against_differences_of_the_cpp_oracles_gradient(model, nf, p, pt):
    o = Oracle(4, 1.0, nf, model, p, mpl=1.7)
    V, dV, H = linear.potential(model, p, 1.7, [np.float64(x) for x in pt])
    V0, dV0 = o.potential(pt)
    assert abs(V - V0) < 1e-14 * max(1, abs(V0)) and all(abs(a - b) < 1e-13 * max(1, abs(b)) for a, b in zip(dV, dV0))
    h = 1e-5
    for j in range(nf):
        up, dn = list(pt), list(pt)
        up[j] += h; dn[j] -= h
        gu, gd = o.potential(up)[1], o.potential(dn)[1]
        for i in range(nf):
            fd = (gu[i] - gd[i]) / (2 * h)
            assert abs(H[i][j] - fd) < 1e-6 * max(1.0, abs(fd)), (i, j)
            assert abs(H[i][j] - H[j][i]) <= 1e-15 * abs(H[i][j])


# ---------------------------------------------------------------- L8
@pytest.mark.parametrize("order", [2, 4])
def test_l8_convergence_order(order):
    N, T = 4, 0.16
    rng = np.random.default_rng(5)
    dphi, dpi = rng.standard_normal((2, N, N, N)), rng.standard_normal((2, N, N, N))

    def run(o_, dt):
        o = linear.LinearOracle(N, 2.0, 2, CHAOTIC, (1.0, 100.0), order=o_, dt=dt, mpl=1.0, precision=80)
        o.set_background(1.0, math.nan, (0.9, 0.02), (-0.7, 0.1))
        o.set_perturbations(dphi, dpi)
        o.step(int(round(T / dt)))
        return np.concatenate([o.dPhi.ravel(), o.dPi.ravel()]), o.a

    ref, a_ref = run(6, T / 256)
    errs = []
    for dt in (T / 16, T / 32, T / 64):
        v, a = run(order, dt)
        errs.append(float(np.max(np.abs(v - ref))))
    for e0, e1 in zip(errs, errs[1:]):
        assert abs(math.log2(e0 / e1) - order) < 0.35, errs
