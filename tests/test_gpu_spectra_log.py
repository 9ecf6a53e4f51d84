"""SURVEY 8(f) rank 3 on the device, against the oracles: number- and energy-density spectra (oracle/spectra.py,
reading G24) and the energy log written at a cadence without host synchronisation.  `-m gpu`."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from oracle import spectra
from paper_1201_5029_b200 import inputs
from helpers import DEFAULT_STENCIL, SEVEN_POINT

INF = math.inf


@pytest.fixture(scope="module")
def pc():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1201_5029_b200 import build
    build.build()
    from paper_1201_5029_b200 import binding
    binding.lib()
    return binding


def energy_tuple(e, nf):
    return (e.a, e.p_a, e.eta, e.pot, e.rho, e.pressure, e.hubble, e.residual) + tuple(e.kin[:nf]) + tuple(e.grad[:nf]) + \
        tuple(e.sum_phiDphi[:nf])


# ------------------------------------------------------------------------------------- spectra
@pytest.mark.parametrize("N,precision,stencil", [(24, 64, (0, 0, 0, 0)), (32, 64, SEVEN_POINT), (18, 64, (0, 0, 0, 0)),
                                                  (24, 32, (0, 0, 0, 0))])
def test_mode_spectra_match_the_oracle(pc, N, precision, stencil):
    """Both sides evolve the chaotic lattice a few steps from the same input, then form the spectra of each field
    with their own a: number, energy and counts per shell against oracle/spectra.py (which is pinned by a single
    mode, Parseval against energies(), the vacuum state and the adiabatic invariant)."""
    cfg = inputs.config("cfg0b_chaotic32_resolved", N=N)
    cfg["amp"] = 1e-3
    phi, pi = inputs.make_initial(cfg, precision=precision)
    kw = dict(mpl=cfg["mpl"], precision=precision, stencil=stencil)
    g = pc.Lattice(N, cfg["L"], 2, cfg["model"], cfg["p"], order=4, dt=cfg["dt"], **kw)
    o = oracle.Oracle(N, cfg["L"], 2, cfg["model"], cfg["p"], order=4, dt=cfg["dt"], **kw)
    for s in (g, o):
        s.set_fields(phi, pi); s.set_background(1.0); s.step(3)
    po, qo = o.read_fields()
    a = o.energies().a
    st = DEFAULT_STENCIL if stencil == (0, 0, 0, 0) else stencil
    # fp32 fields: the removed zero mode comes back at the rounding level of a float (1e-8 of the spectrum's peak)
    tol, floor = (1e-10, 1e-300) if precision == 64 else (2e-4, 1e-8)
    for f, m2 in ((0, 1.0), (1, 1.0e4 * 0.9676 ** 2)):
        want_n, want_e, want_c = spectra.mode_spectra(po[f].astype(np.float64), qo[f].astype(np.float64), cfg["L"], a, m2, st)
        got_n, got_e, got_c = g.mode_spectra(f, m2)
        assert len(got_c) == len(want_c) and np.array_equal(got_c, want_c) and got_c.sum() == N ** 3
        assert np.max(np.abs(got_n - want_n) / (np.abs(want_n) + floor * want_n.max())) < tol, f
        assert np.max(np.abs(got_e - want_e) / (np.abs(want_e) + floor * want_e.max())) < tol, f
        # a short output: the shells beyond nbins are dropped, the others unchanged
        n8, e8, c8 = g.mode_spectra(f, m2, nbins=8)
        assert np.array_equal(c8, want_c[:8]) and np.max(np.abs(n8 - want_n[:8]) / (want_n[:8] + floor * want_n.max())) < tol


def test_energy_spectrum_sums_to_the_energies_on_the_device(pc):
    """(2/(a^4 L^3)) sum_i energy_i = kin + grad + 1/2 m^2 <phi^2> (free field): the device spectrum against the
    device's own pycool_energies, after expansion has moved a away from 1."""
    N, L, m2 = 20, 5.0, 1.3
    phi, pi = inputs.random_fields(N, 1, seed=3, mean=0.4, amp=0.2)
    g = pc.Lattice(N, L, 1, pc.FREE, [m2], order=4, dt=0.01, mpl=0.5)
    g.set_fields(phi, pi); g.set_background(1.0)
    g.step(40)
    e = g.energies()
    assert e.a > 1.05
    _, energy, _ = g.mode_spectra(0, m2)
    total = 2.0 / (e.a ** 4 * L ** 3) * energy.sum()
    assert abs(total - (e.kin[0] + e.grad[0] + e.pot)) < 1e-11 * total


def test_spectrum_argument_checks(pc):
    g = pc.Lattice(8, 1.0, 1, pc.FREE, [1.0])
    with pytest.raises(pc.PycoolError) as ei:
        g.mode_spectra(0, 1.0)
    assert ei.value.code == pc.ESTATE
    z = np.zeros((1, 8, 8, 8))
    g.set_fields(z + 1.0, z)
    for bad in (dict(field=1, m_eff2=1.0), dict(field=0, m_eff2=math.nan), dict(field=0, m_eff2=1.0, nbins=4096)):
        with pytest.raises(pc.PycoolError) as ei:
            g.mode_spectra(**bad)
        assert ei.value.code == pc.EINVAL
    with pytest.raises(pc.PycoolError) as ei:
        g.field_spectrum(0, 0, nbins=4096)                   # more than 48 KB of shared-memory histogram
    assert ei.value.code == pc.EINVAL
    # massless: the zero mode has w^2 = k_eff^2(0)/dx^2 = 0 up to the rounding of c0 + 6 c1 + 12 c2 + 8 c3 (1e-16), so
    # n = 0 and rho = |v|^2/2 + w^2 |u|^2/2 = 0 to that rounding
    n, e, c = g.mode_spectra(0, 0.0)
    assert n[0] == 0.0 and abs(e[0]) < 1e-13 and c[0] == 1


# ------------------------------------------------------------------------------------- energy log
@pytest.mark.parametrize("name,N,precision,kw", [("cfg0_chaotic32", 32, 64, {}), ("cfg0_chaotic32", 21, 64, {}),
                                                 ("cfg3_qball256", 40, 64, {}), ("cfg2_oscillon256", 72, 64, {}),
                                                 ("cfg0_chaotic32", 24, 32, {}), ("cfg0_chaotic32", 24, 64, {"adaptive": True})])
def test_energy_log_entries_are_the_synchronous_read_outs(pc, name, N, precision, kw):
    """A run of 7 steps in two calls with the log at a cadence of 2: (i) its final fields and scalars are bitwise those
    of an unlogged run -- the log does not touch the step sequence; (ii) every entry is bitwise what pycool_energies
    returns for a run stopped at that step (the flushed state and the on-the-fly closing drift see the same phi);
    (iii) each entry matches the oracle at that step.  TMA kernel (even N) and plain kernel (odd N)."""
    # cfg0's literal dt = L/N/20 is stable at N = 32 only (reading G19): the other sizes take the resolved step
    cfg = inputs.config(name, N=N) if (name != "cfg0_chaotic32" or N == 32) else inputs.config(name, N=N, dt=0.0025)
    cfg["L"] = cfg["L"] * N / inputs.config(name)["N"] if name != "cfg0_chaotic32" else cfg["L"]
    nf = cfg["nfields"]
    phi, pi = inputs.make_initial(cfg, precision=precision)

    def fresh():
        g = pc.from_config(cfg, precision=precision)
        g.set_fields(phi, pi); g.set_background(1.0)
        if kw.get("adaptive"):
            g.set_adaptive(True)
        return g

    a = fresh()
    a.set_energy_cadence(2, 8)
    a.step(3); a.step(4)
    entries, total = a.read_energy_log()
    assert total == 3 and len(entries) == 3
    b = fresh()
    b.step(3); b.step(4)
    pa, qa = a.read_fields()
    pb, qb = b.read_fields()
    assert np.array_equal(pa, pb) and np.array_equal(qa, qb)
    assert energy_tuple(a.energies(), nf) == energy_tuple(b.energies(), nf)
    o = oracle.Oracle(N, cfg["L"], nf, cfg["model"], cfg["p"], order=cfg["order"], dt=cfg["dt"], mpl=cfg["mpl"],
                      rho_gamma0=cfg["rho_gamma0"], rho_m0=cfg["rho_m0"], precision=precision)
    o.set_fields(phi, pi); o.set_background(1.0)
    if kw.get("adaptive"):
        o.set_adaptive(True)
    tol = 1e-10 if precision == 64 else 1e-4
    for i, m in enumerate((2, 4, 6)):
        c = fresh()
        c.step(m)
        assert energy_tuple(entries[i], nf) == energy_tuple(c.energies(), nf), m
        o.step(2)
        eo = o.energies()
        for got, want in zip(energy_tuple(entries[i], nf)[:7], energy_tuple(eo, nf)[:7]):
            assert abs(got - want) <= tol * max(abs(want), 1e-300), (m, got, want)
    assert entries[0].eta < entries[1].eta < entries[2].eta and entries[0].a < entries[2].a


def test_energy_log_ring_and_switch_off(pc):
    cfg = inputs.config("cfg0_chaotic32", N=16, dt=0.0025)        # L/N/20 is unstable below N = 32 (reading G19)
    phi, pi = inputs.make_initial(cfg)
    g = pc.from_config(cfg)
    g.set_fields(phi, pi); g.set_background(1.0)
    g.set_energy_cadence(1, 3)
    n0 = g.launch_counts()
    g.step(5)
    assert g.launch_counts()[3] - n0[3] == 2 * 5 and g.launch_counts()[0] - n0[0] == 15    # no extra launches besides
    entries, total = g.read_energy_log()
    assert total == 5 and len(entries) == 3
    etas = [e.eta for e in entries]
    assert all(abs(x - (k + 3) * cfg["dt"]) < 1e-15 for k, x in enumerate(etas))            # steps 3, 4, 5 survive
    newest, _ = g.read_energy_log(max_entries=1)
    assert len(newest) == 1 and newest[0].eta == etas[-1]
    g.set_energy_cadence(0)
    g.step(2)
    assert g.read_energy_log() == ([], 0)
    with pytest.raises(pc.PycoolError):
        g.set_energy_cadence(2, 0)
