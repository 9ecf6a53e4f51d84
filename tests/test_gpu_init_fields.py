"""pycool_init_fields (seeded Gaussian initial conditions on the device) against oracle/ics.py."""
import math

import numpy as np
import pytest

import oracle
from oracle import ics
from paper_1201_5029_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pc():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1201_5029_b200 import build
    build.build()
    from paper_1201_5029_b200 import binding
    binding.lib()
    return binding


def _check(got, want, means, precision):
    """Element by element.  fp64: rounding of mean + delta (a few ulp of the mean) plus FFT / Box-Muller rounding
    (1e-12 of the fluctuation rms); fp32: one rounding of the fp64 value."""
    for f in range(got.shape[0]):
        d = np.abs(got[f].astype(np.float64) - want[f])
        if precision == 64:
            rms = float(np.std(want[f]))
            assert d.max() <= 4 * np.spacing(abs(means[f]) + 6 * rms) + 1e-12 * rms, (f, d.max(), rms)
        else:
            assert np.all(d <= 0.51 * np.spacing(np.abs(want[f]).astype(np.float32)).astype(np.float64) + 1e-12 * np.std(want[f]))


@pytest.mark.parametrize("name,N", [("cfg0_chaotic32", 16), ("cfg0_chaotic32", 40), ("cfg0_chaotic32", 64),
                                    ("cfg2_oscillon256", 24), ("cfg3_qball256", 36)])
@pytest.mark.parametrize("precision", [64, 32])
def test_device_initial_conditions_match_the_oracle(pc, name, N, precision):
    cfg = inputs.config(name, N=N)
    cfg["L"] = cfg["L"] * N / inputs.config(name)["N"] * (4 if name == "cfg2_oscillon256" else 1)
    phi_spec, pi_spec = inputs.spectra(cfg)
    seed = 0x1234567 + N
    g = pc.from_config(cfg, precision=precision)
    g.init_fields(seed, phi_spec, pi_spec)
    pg, qg = g.read_fields()
    po, qo = ics.init_fields(N, cfg["L"], cfg["nfields"], seed, phi_spec, pi_spec)
    assert pg.dtype == (np.float64 if precision == 64 else np.float32)
    _check(pg, po, [t[0] for t in phi_spec], precision)
    _check(qg, qo, [t[0] for t in pi_spec], precision)
    assert np.std(po[0]) > 0                                      # there are fluctuations to compare


def test_same_seed_same_lattice_and_ghost_images_carry_a_step(pc):
    """Bitwise reproducible; another seed differs; and the lattice is usable as it stands (ghost images written by
    the generator): two steps from the device-made lattice against the oracle stepper started from the oracle's."""
    cfg = inputs.config("cfg0b_chaotic32_resolved", N=40)
    phi_spec, pi_spec = inputs.spectra(cfg)
    a, b, c = pc.from_config(cfg), pc.from_config(cfg), pc.from_config(cfg)
    a.init_fields(7, phi_spec, pi_spec); b.init_fields(7, phi_spec, pi_spec); c.init_fields(8, phi_spec, pi_spec)
    pa, qa = a.read_fields(); pb, qb = b.read_fields(); pcc, _ = c.read_fields()
    assert np.array_equal(pa, pb) and np.array_equal(qa, qb) and not np.array_equal(pa, pcc)
    po, qo = ics.init_fields(40, cfg["L"], 2, 7, phi_spec, pi_spec)
    o = oracle.Oracle(40, cfg["L"], 2, oracle.CHAOTIC, cfg["p"], order=cfg["order"], dt=cfg["dt"], mpl=cfg["mpl"])
    o.set_fields(po, qo); o.set_background(1.0)
    a.set_background(1.0)
    assert abs(a.energies().rho - o.energies().rho) <= 1e-10 * o.energies().rho
    a.step(2); o.step(2)
    p2, q2 = a.read_fields(); p3, q3 = o.read_fields()
    for x, y in ((p2, p3), (q2, q3)):
        for f in range(2):
            rms = math.sqrt(float(np.mean(y[f] ** 2)))
            assert np.max(np.abs(x[f] - y[f]) / np.maximum(np.abs(y[f]), rms)) <= 1e-10


def test_power_spectrum_of_the_device_lattice(pc):
    """Independent of the oracle: shell-averaged |FFT|^2 of the device-made field follows A(k)^2 (vacuum spectrum,
    128^3: ~1e6 modes), and the real-space variance is the Parseval sum."""
    N, L, amp, m2 = 128, 10.0, 1e-3, 4.0
    g = pc.Lattice(N, L, 1, pc.FREE, [1.0], order=2, dt=0.01, mpl=1.0)
    g.init_fields(42, [(0.5, amp, m2, -0.25, 0.0)], [(0.0, amp, m2, 0.25, 0.0)])
    phi, pi = g.read_fields()
    for arr, q in ((phi[0] - 0.5, -0.25), (pi[0], 0.25)):
        F = np.fft.rfftn(arr) * (L ** 1.5 / (math.sqrt(2.0) * N ** 3))          # back to F_k
        n1 = np.fft.fftfreq(N, d=1.0 / N)
        n2 = (n1 ** 2)[:, None, None] + (n1 ** 2)[None, :, None] + (np.arange(N // 2 + 1) ** 2)[None, None, :]
        k = 2 * math.pi / L * np.sqrt(n2)
        A2 = (amp * (k * k + m2) ** q) ** 2
        sel = (n2 > 0) & (np.arange(N // 2 + 1)[None, None, :] > 0) & (np.arange(N // 2 + 1)[None, None, :] < N // 2)
        ratio = (np.abs(F) ** 2)[sel] / A2[sel]
        assert abs(ratio.mean() - 1) < 5 / math.sqrt(ratio.size)          # exponential distribution, unit mean
        shells = np.sqrt(n2[sel]).astype(int)
        for s in (3, 10, 30, 60):
            r = ratio[shells == s]
            assert abs(r.mean() - 1) < 5 / math.sqrt(r.size)
    assert abs(phi[0].mean() - 0.5) < 1e-12


def test_init_fields_argument_errors(pc):
    g = pc.Lattice(9, 1.0, 1, pc.FREE, [1.0], order=2, dt=0.01, mpl=1.0)
    with pytest.raises(pc.PycoolError) as ei:
        g.init_fields(1, [(0, 1, 1, 0, 0)], [(0, 1, 1, 0, 0)])
    assert ei.value.code == pc.EINVAL and "even N" in str(ei.value)
    h = pc.Lattice(8, 1.0, 1, pc.FREE, [1.0], order=2, dt=0.01, mpl=1.0)
    with pytest.raises(pc.PycoolError) as ei:
        h.init_fields(1, [(0, 1, -1.0, 0, 0)], [(0, 1, 1, 0, 0)])
    assert ei.value.code == pc.EINVAL
    with pytest.raises(pc.PycoolError):
        h.step(1)                                                   # still no fields
    h.init_fields(1, [(0, 1, 1, 0, 0)], [(0, 1, 1, 0, 0)])
    h.set_background(1.0, 0.0)
    h.step(1)


# ------------------------------------------------------------------------------------- shell spectrum (rank 3)
@pytest.mark.parametrize("N,precision", [(16, 64), (40, 64), (33, 64), (64, 32), (130, 64)])
def test_field_spectrum_matches_the_oracle(pc, N, precision):
    """pycool_field_spectrum (gather + cuFFT D2Z + shell sums) of phi and pi of both fields, after two steps, against
    numpy's rfftn + bincount on the lattice read back; even, odd and ragged N; mode counts exact."""
    cfg = inputs.config("cfg0b_chaotic32_resolved", N=N)
    cfg["amp"] = 1e-3
    phi, pi = inputs.make_initial(cfg, precision=precision)
    g = pc.from_config(cfg, precision=precision)
    g.set_fields(phi, pi); g.set_background(1.0)
    g.step(2)
    pg, qg = g.read_fields()
    for f in range(2):
        for which, arr in ((0, pg), (1, qg)):
            S, Cn = g.field_spectrum(f, which)
            So, Co = ics.shell_spectrum(arr[f], cfg["L"])
            assert len(S) == len(So) == int(math.sqrt(3) * N / 2 + 0.5) + 1
            assert np.array_equal(Cn, Co) and Cn.sum() == N ** 3
            nz = So > 0
            assert np.max(np.abs(S[nz] - So[nz]) / So[nz]) <= 1e-10
            assert np.all(S[~nz] == 0)
    short, _ = g.field_spectrum(0, 0, nbins=5)
    full, _ = g.field_spectrum(0, 0)
    assert np.allclose(short, full[:5], rtol=1e-12, atol=0)


def test_spectrum_of_the_generated_lattice_returns_its_amplitude(pc):
    """Round trip on the device: init_fields with A(k), field_spectrum back: power/count = A(k_shell)^2 within the
    statistical error of the shell (and the shell's width in k)."""
    N, L, amp, m2 = 128, 10.0, 1e-3, 4.0
    g = pc.Lattice(N, L, 1, pc.FREE, [1.0], order=2, dt=0.01, mpl=1.0)
    g.init_fields(5, [(0.5, amp, m2, -0.25, 0.0)], [(0.0, amp, m2, 0.25, 0.0)])
    for which, q in ((0, -0.25), (1, 0.25)):
        S, Cn = g.field_spectrum(0, which)
        for i in (4, 10, 30, 60):
            k = 2 * math.pi / L * i
            want = (amp * (k * k + m2) ** q) ** 2
            assert abs(S[i] / Cn[i] / want - 1) < 6 / math.sqrt(Cn[i]) + 0.02
    S, _ = g.field_spectrum(0, 0)
    assert abs(S[0] - L ** 3 / 2 * 0.25) < 1e-9 * S[0]                      # the mean sits in shell 0


def test_field_spectrum_argument_errors(pc):
    g = pc.Lattice(8, 1.0, 1, pc.FREE, [1.0], order=2, dt=0.01, mpl=1.0)
    with pytest.raises(pc.PycoolError) as ei:
        g.field_spectrum(0)
    assert ei.value.code == pc.ESTATE
    g.init_fields(1, [(0, 1, 1, 0, 0)], [(0, 1, 1, 0, 0)])
    for args in ((1, 0), (0, 2), (-1, 0)):
        with pytest.raises(pc.PycoolError) as ei:
            g.field_spectrum(*args)
        assert ei.value.code == pc.EINVAL
