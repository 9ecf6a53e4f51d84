"""The linearised solver on the device (include/pycool_linear.h) against oracle/linear.py, element by
element in Fourier space: background, growth matrices (2.51), modes advanced through the matrices and on their own
("naive"), transforms in and out.  `-m gpu`.  The oracle is pinned by tests/test_oracle_linear.py (L1-L8)."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import linear
from paper_1201_5029_b200 import inputs

INF = math.inf
CHAOTIC = dict(model=1, p=(1.0, 1.0e4))
MODELS = {
    "chaotic": dict(nf=2, model=1, p=(1.0, 1.0e4), mpl=1.0, phi0=(0.9676, 1e-3), pi0=(-0.71, 2e-3)),
    "free3": dict(nf=3, model=0, p=(1.0, 2.5, 0.3), mpl=2.0, phi0=(0.5, -0.2, 0.1), pi0=(0.1, 0.2, -0.3)),
    "free4_static": dict(nf=4, model=0, p=(1.0, 2.5, 0.3, 4.0), mpl=INF, phi0=(0.5, -0.2, 0.1, 0.3), pi0=(0.1, 0.2, -0.3, 0.0)),
    "oscillon": dict(nf=1, model=2, p=(1.0, 1.0, 0.3), mpl=335.41, phi0=(2.0,), pi0=(0.05,)),
    "qball": dict(nf=2, model=3, p=(1.0, -0.1, 1.0, 0.0), mpl=30.0, phi0=(1.4, 0.1), pi0=(0.0, 0.7)),
}


@pytest.fixture(scope="module")
def pc():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1201_5029_b200 import build
    build.build()
    from paper_1201_5029_b200 import binding
    binding.lib()
    return binding


def make_pair(pc, name, N, L, order, dt, stencil=(0, 0, 0, 0), rho_m0=0.0):
    m = MODELS[name]
    g = pc.LinearLattice(N, L, m["nf"], m["model"], m["p"], order=order, dt=dt, mpl=m["mpl"], stencil=stencil, rho_m0=rho_m0)
    o = linear.LinearOracle(N, L, m["nf"], m["model"], m["p"], order=order, dt=dt, mpl=m["mpl"], stencil=stencil,
                            rho_m0=rho_m0)
    p_a = 0.0 if m["mpl"] == INF else math.nan
    rng = np.random.default_rng(N * 131 + order)
    dphi = 1e-3 * rng.standard_normal((m["nf"], N, N, N))
    dpi = 1e-3 * rng.standard_normal((m["nf"], N, N, N))
    for s in (g, o):
        s.set_background(1.0, p_a, m["phi0"], m["pi0"])
        s.set_perturbations(dphi, dpi)
    return g, o, dphi, dpi


def rel_err(got, want):
    """Per-element error relative to max(|want|, rms(want)) per array (reading G18: modes cross zero)."""
    worst = 0.0
    for f in range(want.shape[0]):
        rms = math.sqrt(float(np.mean(np.abs(want[f]) ** 2)))
        worst = max(worst, float(np.max(np.abs(got[f] - want[f]) / np.maximum(np.abs(want[f]), rms))))
    return worst


def check_background(g, o, nf, tol=1e-12):
    b, e = g.background(), o.background_energy()
    for got, want in ((b.a, o.a), (b.p_a, o.p_a), (b.eta, o.eta), (b.kin, e["kin"]), (b.pot, e["pot"]), (b.rho, e["rho"]),
                      (b.hubble, e["hubble"])):
        assert abs(got - float(want)) <= tol * max(abs(float(want)), 1e-300), (got, want)
    for f in range(nf):
        assert abs(b.phi0[f] - float(o.phi0[f])) <= tol * max(abs(float(o.phi0[f])), 1e-3)
        assert abs(b.pi0[f] - float(o.pi0[f])) <= tol * max(abs(float(o.pi0[f])), 1e-3)
    assert abs(b.residual - float(e["residual"])) <= 1e-9


def half(x):
    return x[..., : x.shape[-1] // 2 + 1]


# ------------------------------------------------------------------------------------- transforms
@pytest.mark.parametrize("N", [6, 9, 16])
def test_transforms_in_and_out(pc, N):
    """set_perturbations = plain DFT of the real arrays with the k = 0 mode removed (2.22), in the half-spectrum layout;
    read_perturbations inverts it; set_modes / read_modes round-trip bit for bit."""
    g, o, dphi, dpi = make_pair(pc, "chaotic", N, 3.0, 2, 0.01)
    P, Q = g.read_modes()
    wantP, wantQ = np.fft.rfftn(dphi, axes=(1, 2, 3)), np.fft.rfftn(dpi, axes=(1, 2, 3))
    wantP[:, 0, 0, 0] = 0; wantQ[:, 0, 0, 0] = 0
    assert rel_err(P, wantP) < 1e-13 and rel_err(Q, wantQ) < 1e-13
    assert np.all(P[:, 0, 0, 0] == 0) and np.all(Q[:, 0, 0, 0] == 0)
    assert rel_err(P, half(o.dPhi)) < 1e-13                      # the oracle's full spectrum, its half
    a, b = g.read_perturbations()
    mean = lambda x: x.mean(axis=(1, 2, 3), keepdims=True)
    assert np.max(np.abs(a - (dphi - mean(dphi)))) < 1e-15 and np.max(np.abs(b - (dpi - mean(dpi)))) < 1e-15
    g.set_modes(wantP, wantQ)
    P2, Q2 = g.read_modes()
    assert np.array_equal(P2, wantP) and np.array_equal(Q2, wantQ)


# ------------------------------------------------------------------------------------- evolution
@pytest.mark.parametrize("name,N,order,steps", [("chaotic", 8, 4, 5), ("chaotic", 12, 2, 7), ("chaotic", 7, 6, 3),
                                                ("chaotic", 16, 8, 2), ("free3", 10, 4, 6), ("free4_static", 6, 4, 6),
                                                ("oscillon", 12, 4, 8), ("qball", 10, 4, 6), ("qball", 9, 6, 3)])
@pytest.mark.parametrize("method", ["growth", "naive"])
def test_modes_and_background_match_the_oracle(pc, name, N, order, steps, method):
    """n steps on the device (one growth matrix per class applied to every mode, or every mode on its own) against
    the oracle's per-mode evolution: every Fourier coefficient of every field, the background and its energies."""
    g, o, _, _ = make_pair(pc, name, N, 4.0, order, 0.01)
    nf = MODELS[name]["nf"]
    g.step(steps, pc.GROWTH if method == "growth" else pc.NAIVE)
    o.step(steps)
    P, Q = g.read_modes()
    assert rel_err(P, half(o.dPhi)) < 1e-12 and rel_err(Q, half(o.dPi)) < 1e-12
    check_background(g, o, nf)
    # a second call continues from the state of the first (background and modes both carried on)
    g.step(2, pc.GROWTH if method == "growth" else pc.NAIVE)
    o.step(2)
    P, Q = g.read_modes()
    assert rel_err(P, half(o.dPhi)) < 2e-12 and rel_err(Q, half(o.dPi)) < 2e-12
    check_background(g, o, nf)
    a, b = g.read_perturbations()
    oa, ob = o.read_perturbations()
    assert np.max(np.abs(a - oa)) < 1e-12 * np.max(np.abs(oa)) and np.max(np.abs(b - ob)) < 1e-12 * np.max(np.abs(ob))


@pytest.mark.parametrize("name,N,order,stencil", [("chaotic", 8, 4, (0, 0, 0, 0)), ("chaotic", 11, 2, (-6.0, 1.0, 0.0, 0.0)),
                                                  ("free3", 6, 6, (0, 0, 0, 0)), ("qball", 12, 4, (0, 0, 0, 0))])
def test_growth_matrices_match_the_oracle_and_are_symplectic(pc, name, N, order, stencil):
    """(2.51): the device's matrix of every distinct-k_eff^2 class against oracle.growth_matrices -- same class order
    (reading G28: sorted triples, hi slowest) -- and M^T J M = J, which no integrator of a non-Hamiltonian system has."""
    g, o, _, _ = make_pair(pc, name, N, 4.0, order, 0.005, stencil=stencil)
    nf = MODELS[name]["nf"]
    with pytest.raises(pc.PycoolError) as ei:
        g.growth()
    assert ei.value.code == pc.ESTATE
    g.step(4, pc.GROWTH)
    M = g.growth()
    want, index = o.growth_matrices(4)
    triples, index2, mult = linear.distinct_table(N)
    assert M.shape == want.shape == (g.nclasses, 2 * nf, 2 * nf) and len(triples) == g.nclasses
    assert np.max(np.abs(M - want)) < 1e-12 * np.max(np.abs(want))
    J = np.zeros((2 * nf, 2 * nf))
    for i in range(nf):
        J[2 * i, 2 * i + 1], J[2 * i + 1, 2 * i] = 1.0, -1.0
    assert np.max(np.abs(np.einsum("tji,jk,tkl->til", M, J, M) - J)) < 1e-13 * max(1.0, np.max(np.abs(M)) ** 2)


def test_growth_and_naive_agree_on_the_device(pc):
    """evolving the modes through the growth functions is the same linear map as evolving each mode."""
    g1, _, dphi, dpi = make_pair(pc, "chaotic", 24, 5.0, 4, 0.005)
    g2, _, _, _ = make_pair(pc, "chaotic", 24, 5.0, 4, 0.005)
    g1.step(30, pc.GROWTH)
    g2.step(30, pc.NAIVE)
    (P1, Q1), (P2, Q2) = g1.read_modes(), g2.read_modes()
    assert rel_err(P1, P2) < 1e-12 and rel_err(Q1, Q2) < 1e-12
    assert g1.background().a == g2.background().a and g1.background().p_a == g2.background().p_a
    t = g1.time_ms()
    assert t["background"] > 0 and t["growth"] > 0 and t["modes"] > 0 and g2.time_ms()["growth"] == 0.0


def test_many_steps_table_larger_than_one_chunk(pc):
    """200 steps of order 6 = 1400 stages: the coefficient table streams through shared memory in 22 chunks."""
    g, o, _, _ = make_pair(pc, "chaotic", 8, 4.0, 6, 0.002)
    g.step(200, pc.GROWTH)
    o.step(200)
    P, Q = g.read_modes()
    assert rel_err(P, half(o.dPhi)) < 1e-10 and rel_err(Q, half(o.dPi)) < 1e-10
    check_background(g, o, 2, tol=1e-11)


def test_matter_term_and_explicit_p_a(pc):
    """rho_m0 enters p_a' (2.20); an explicit p_a is taken as given."""
    m = MODELS["chaotic"]
    g = pc.LinearLattice(8, 4.0, 2, m["model"], m["p"], order=4, dt=0.01, mpl=1.0, rho_m0=0.7)
    o = linear.LinearOracle(8, 4.0, 2, m["model"], m["p"], order=4, dt=0.01, mpl=1.0, rho_m0=0.7)
    for s in (g, o):
        s.set_background(1.2, -3000.0, m["phi0"], m["pi0"])
    g.step(10, pc.NAIVE); o.step(10)
    check_background(g, o, 2)


@pytest.mark.parametrize("N,method", [(128, "growth"), (256, "growth"), (256, "naive")])
def test_sampled_modes_at_bench_size(pc, N, method):
    """The size and launch configuration bench.py's `linear` block times (256^3 x 2 fields, order 4, 20 steps per call;
    also 128^3): every 97th mode of the half spectrum against the oracle's per-mode evolution of exactly those modes
    (the oracle's own arrays hold full complex spectra, so it is run on the sample: a mode's evolution depends on its
    k_eff^2 and the background only)."""
    L, steps = 10.0, 20
    m = MODELS["chaotic"]
    g = pc.LinearLattice(N, L, 2, m["model"], m["p"], order=4, dt=L / N / 20.0, mpl=1.0)
    g.set_background(1.0, math.nan, m["phi0"], m["pi0"])
    rng = np.random.default_rng(5)
    shape = (2, N, N, N // 2 + 1)
    P0 = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    Q0 = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    g.set_modes(P0, Q0)
    g.step(steps, pc.GROWTH if method == "growth" else pc.NAIVE)
    P, Q = g.read_modes()
    # the oracle on the sampled modes: a tiny LinearOracle carries the background, the modes' own k_eff^2 is passed in
    o = linear.LinearOracle(4, L * 4 / N, 2, m["model"], m["p"], order=4, dt=L / N / 20.0, mpl=1.0)
    o.VL = o.T(N) ** 3                                            # the background's V_L is the big lattice's
    o.set_background(1.0, math.nan, m["phi0"], m["pi0"])
    flat = np.arange(0, N * N * (N // 2 + 1), 97)
    ix = flat % (N // 2 + 1); iy = (flat // (N // 2 + 1)) % N; iz = flat // ((N // 2 + 1) * N)
    fold = lambda i: np.where(i <= N // 2, i, i - N)
    k2 = linear.k_eff2_of(np.stack([ix, fold(iy), fold(iz)], axis=-1), N, o.stencil)
    Phi = np.stack([P0[f].reshape(-1)[flat] for f in range(2)])
    Pi = np.stack([Q0[f].reshape(-1)[flat] for f in range(2)])
    zero = flat == 0
    Phi[:, zero] = 0; Pi[:, zero] = 0
    o._advance(steps, Phi, Pi, k2)
    got_P = np.stack([P[f].reshape(-1)[flat] for f in range(2)])
    got_Q = np.stack([Q[f].reshape(-1)[flat] for f in range(2)])
    assert rel_err(got_P, Phi) < 1e-12 and rel_err(got_Q, Pi) < 1e-12
    b = g.background()
    assert abs(b.a - float(o.a)) < 1e-13 * b.a and abs(b.p_a - float(o.p_a)) < 1e-12 * abs(b.p_a)
