"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  All tests here need a B200 (`-m gpu`).

Tolerances (north_star, fp64): per-site max relative error (reading G18) <= 1e-12 after 1 step and <= 1e-9
after 100 steps on configs[0]; scale factor and energy components <= 1e-10 relative.  fp32: <= 1e-5 after one
step.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_1201_5029_b200 import inputs
from helpers import SEVEN_POINT, rel_err_per_site

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


def make_pair(pc, cfg, precision=64, **over):
    kw = dict(mpl=cfg["mpl"], rho_gamma0=cfg["rho_gamma0"], rho_m0=cfg["rho_m0"], precision=precision)
    kw.update(over)
    order, dt = kw.pop("order", cfg["order"]), kw.pop("dt", cfg["dt"])
    g = pc.Lattice(cfg["N"], cfg["L"], cfg["nfields"], cfg["model"], cfg["p"], order=order, dt=dt, **kw)
    o = oracle.Oracle(cfg["N"], cfg["L"], cfg["nfields"], cfg["model"], cfg["p"], order=order, dt=dt, **kw)
    return g, o


def start(g, o, phi, pi, a=1.0, p_a=math.nan):
    for s in (g, o):
        s.set_fields(phi, pi)
        s.set_background(a, p_a)


def rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


def check_scalars(eg, eo, nf, tol=1e-10, static=False, tol_eta=1e-14):
    assert rel(eg.a, eo.a) <= tol and rel(eg.eta, eo.eta) <= tol_eta
    if not static:
        assert rel(eg.p_a, eo.p_a) <= tol and rel(eg.hubble, eo.hubble) <= tol
    for f in range(nf):
        assert rel(eg.kin[f], eo.kin[f]) <= tol, ("kin", f, eg.kin[f], eo.kin[f])
        assert rel(eg.grad[f], eo.grad[f]) <= tol, ("grad", f, eg.grad[f], eo.grad[f])
        assert rel(eg.sum_phiDphi[f], eo.sum_phiDphi[f]) <= max(tol, 1e-9), ("phiDphi", f)
    assert rel(eg.pot, eo.pot) <= tol and rel(eg.rho, eo.rho) <= tol and rel(eg.pressure, eo.pressure) <= tol


def compare(g, o, nf, tol_site, tol_scalar=1e-10, static=False, tol_eta=1e-14):
    pg, qg = g.read_fields()
    po, qo = o.read_fields()
    e1, e2 = rel_err_per_site(pg, po), rel_err_per_site(qg, qo)
    assert e1 <= tol_site and e2 <= tol_site, (e1, e2)
    check_scalars(g.energies(), o.energies(), nf, tol_scalar, static, tol_eta)
    return max(e1, e2)


# ------------------------------------------------------------------------------------- configs[0]
def test_cfg0_one_step_and_100_steps(pc):
    cfg = inputs.config("cfg0_chaotic32")
    phi, pi = inputs.make_initial(cfg)
    g, o = make_pair(pc, cfg)
    start(g, o, phi, pi)
    check_scalars(g.energies(), o.energies(), 2)            # initial energies and the (2.18) solve
    g.step(1); o.step(1)
    compare(g, o, 2, 1e-12)
    g.step(99); o.step(99)
    compare(g, o, 2, 1e-9)
    assert g.energies().residual < 1e-6


def test_cfg0_resolved_dt(pc):
    cfg = inputs.config("cfg0b_chaotic32_resolved")
    phi, pi = inputs.make_initial(cfg)
    g, o = make_pair(pc, cfg)
    start(g, o, phi, pi)
    g.step(1); o.step(1)
    compare(g, o, 2, 1e-12)
    g.step(99); o.step(99)
    compare(g, o, 2, 1e-9)


def test_cfg0_paper_phi0_reading_g19(pc):
    """The paper's phi0 = 1.009343 with the resolved dt (G19)."""
    cfg = inputs.config("cfg0b_chaotic32_resolved", phi0=(1.009343, 0.0))
    phi, pi = inputs.make_initial(cfg)
    g, o = make_pair(pc, cfg)
    start(g, o, phi, pi)
    assert rel(g.energies().hubble, 0.50467) < 2e-5          # H printed in the paper
    g.step(20); o.step(20)
    compare(g, o, 2, 1e-10)


# ------------------------------------------------------------------------------------- reduced-size cfg1-3
# Tolerance after one step: a 1-ulp difference in phi' (merged vs separate half drifts, FMA) enters pi through
# kD D, i.e. amplified by (|c0| + sum |c_d|) a^2 h/dx^2 ~ 8.5 * 1.35 dt/dx^2 per stage.  For cfg0-cfg2 that factor
# is < 1 and 1e-12 holds.  For the Q-ball lattice dt/dx^2 = 5.1 and |pi_1| ~ 1e-3 |phi_1|: the oracle in double
# against the oracle in long double differs by 1.7e-12 after ONE step there (measured, -m "not gpu":
# tests/test_oracle_pins.py::test_fp64_rounding_floor_of_one_step), so 1e-12 is below the floor of any fp64
# evaluation order.  The GPU's measured error on it is 1.7-1.9e-12 after one step, 2.2e-12 after two (printed by
# the tests below); the tolerance is 3 x the oracle's own floor.
QBALL_TOL_1STEP = 5.2e-12


@pytest.mark.parametrize("name,N,steps,tol1", [("cfg1_chaotic128", 48, 6, 1e-12), ("cfg2_oscillon256", 40, 20, 1e-12),
                                               ("cfg3_qball256", 40, 20, QBALL_TOL_1STEP)])
def test_models_reduced_size(pc, name, N, steps, tol1):
    cfg = inputs.config(name, N=N)
    if name == "cfg2_oscillon256":
        cfg["L"] = 400.0 * N / 256                          # keep dx of the full configuration
    if name == "cfg3_qball256":
        cfg["L"] = 8.0 * N / 256
    phi, pi = inputs.make_initial(cfg)
    g, o = make_pair(pc, cfg)
    start(g, o, phi, pi)
    g.step(1); o.step(1)
    e1 = compare(g, o, cfg["nfields"], tol1)
    g.step(steps - 1); o.step(steps - 1)
    en = compare(g, o, cfg["nfields"], 100 * tol1)
    print("%s at N = %d: per-site error %.2e after 1 step, %.2e after %d" % (name, N, e1, en, steps))


# ------------------------------------------------------------------------------------- orders, tiles, chunks
@pytest.mark.parametrize("order", [2, 4, 6, 8])
def test_all_orders(pc, order):
    cfg = inputs.config("cfg0_chaotic32", N=20, dt=0.004, order=order)
    phi, pi = inputs.make_initial(cfg)
    g, o = make_pair(pc, cfg)
    start(g, o, phi, pi)
    g.step(3); o.step(3)
    compare(g, o, 2, 5e-12)
    assert g.launch_counts()[0] == 3 * {2: 1, 4: 3, 6: 7, 8: 15}[order]


def set_tile_or_skip(pc, g, tile):
    """Variants 6 and 9 (128 x 16: twice the bytes per plane) do not fit in shared memory for two fp64 fields, and
    variant 9 (2 x 4 sites per thread) is built for one-field lattices only: EINVAL, with the reason."""
    try:
        g.set_tile(tile)
    except pc.PycoolError as e:
        assert e.code == pc.EINVAL and tile in (6, 9, 11, 12) and ("shared memory" in str(e) or "not built" in str(e))
        return False
    return True


@pytest.mark.parametrize("tile", [0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10])
@pytest.mark.parametrize("N,zc", [(40, 0), (40, 7), (40, 40), (67, 16), (3, 0), (4, 1), (5, 2), (33, 32), (6, 0),
                                  (70, 9), (136, 50)])
def test_tiles_ragged_edges_and_zchunks(pc, tile, N, zc):
    """Several tiles with ragged tails in x, y and z, wrap-around at every face, for each variant of the fused
    kernel: 0-2 register prefetch (any N), 3-8 TMA ring with ghost images (even N)."""
    cfg = inputs.config("cfg0_chaotic32", N=N, dt=0.002, order=4)
    cfg["init"], cfg["amp"] = "white", 1e-3
    phi, pi = inputs.make_initial(cfg)
    g, o = make_pair(pc, cfg)
    if tile >= 3 and N % 2:
        with pytest.raises(pc.PycoolError) as ei:
            g.set_tile(tile)
        assert ei.value.code == pc.EINVAL
        return
    if not set_tile_or_skip(pc, g, tile):
        return
    g.set_zchunk(zc)
    geo = g.kick_geometry()
    assert geo["zchunk"] >= 1 and geo["blocks"] >= 1 and geo["variant"] == tile
    assert (geo["tma_stages"] > 0) == (tile >= 3)
    start(g, o, phi, pi)
    g.step(2); o.step(2)
    compare(g, o, 2, 2e-12)


@pytest.mark.parametrize("tile", [4, 7, 8, 10, 12])
@pytest.mark.parametrize("N,zc", [(70, 9), (136, 50), (40, 0)])
def test_qball_variants_ragged_edges_and_zchunks(pc, tile, N, zc):
    """The Q-ball model (own logarithm, 2 x 1 sites per thread; variant 12 -- 32 x 8 tile, four blocks per SM -- is its
    automatic choice above N = 64, variants 7 and 8 the two-blocks-per-SM forms) on ragged tiles with short and long z-chunks, against the oracle.  Tolerance:
    the fp64 rounding floor of this lattice is 1.7e-12 per step (tests/test_oracle_pins.py,
    test_fp64_rounding_floor_of_one_step); the GPU's measured error is in DESIGN.md "Tolerances"."""
    cfg = inputs.config("cfg3_qball256", N=N)
    cfg["L"] = 8.0 * N / 256
    phi, pi = inputs.make_initial(cfg)
    g, o = make_pair(pc, cfg)
    g.set_tile(tile); g.set_zchunk(zc)
    assert g.kick_geometry()["variant"] == tile
    start(g, o, phi, pi)
    g.step(1); o.step(1)
    e1 = compare(g, o, 2, QBALL_TOL_1STEP)
    g.step(1); o.step(1)
    e2 = compare(g, o, 2, 2 * QBALL_TOL_1STEP)
    print("qball tile %d N %d zc %d: per-site error %.2e after 1 step, %.2e after 2" % (tile, N, zc, e1, e2))
    if N > 64:
        assert pc.from_config(cfg).kick_geometry()["variant"] == 12


@pytest.mark.parametrize("precision", [64, 32])
def test_variants_agree_and_ghost_images_hold(pc, precision):
    """Every kernel variant from the same state: results agree to rounding, and the ghost columns / rows of the
    padded state equal their periodic sources bit for bit after stepping (what the TMA boxes rely on)."""
    import torch
    cfg = inputs.config("cfg0_chaotic32", N=36, dt=0.002, order=4)
    cfg["init"], cfg["amp"] = "white", 1e-3
    phi, pi = inputs.make_initial(cfg, precision=precision)
    outs = []
    for tile in range(13):
        g = pc.from_config(cfg, precision=precision)
        if not set_tile_or_skip(pc, g, tile):
            assert precision == 64 or tile in (9, 12)
            continue
        g.set_fields(phi, pi)
        g.set_background(1.0)
        g.step(2)
        g.sync()
        outs.append(g.read_fields())
        a, b, lay = pc.C.c_void_p(), pc.C.c_void_p(), (pc.C.c_size_t * 4)()
        assert pc.lib().pycool_device_fields(g._h, pc.C.byref(a), pc.C.byref(b), lay) == 0
        pitch, rows, gx, gy = (int(v) for v in lay)
        assert gx == (2 if precision == 64 else 4) and gy == 1 and rows == 38 and pitch >= 36 + 2 * gx
        for ptr in (a.value, b.value):
            off = ptr - g._work.data_ptr()
            full = g._work[off:off + 2 * 36 * rows * pitch * (precision // 8)].view(g._tdtype).view(2, 36, rows, pitch)
            inner = full[:, :, gy:gy + 36, gx:gx + 36]
            want = torch.cat([inner[..., -gx:], inner, inner[..., :gx]], dim=-1)
            want = torch.cat([want[:, :, -1:, :], want, want[:, :, :1, :]], dim=2)
            assert torch.equal(full[..., :36 + 2 * gx], want), tile
        pd, qd = g.read_fields_device()
        assert np.array_equal(pd.cpu().numpy(), outs[-1][0]) and np.array_equal(qd.cpu().numpy(), outs[-1][1])
        v1, v2 = g.device_fields()
        assert torch.equal(v1, pd) and torch.equal(v2, qd)
    tol = 1e-13 if precision == 64 else 2e-5
    for p, q in outs[1:]:
        assert rel_err_per_site(p, outs[0][0]) < tol and rel_err_per_site(q, outs[0][1]) < tol


@pytest.mark.parametrize("tile", [1, 3, 4])
@pytest.mark.parametrize("N", [20, 72])
def test_fused_tail_equals_separate_scalar_update(pc, tile, N):
    """The last-block-done tail (one launch per stage) against the separate reduce + scalar-update launch: same
    partial sums added in two fixed orders, so fields and scalars agree to rounding; both match the oracle; the
    ticket counter is back at zero afterwards (a second call works) and launch counts show the difference."""
    cfg = inputs.config("cfg0_chaotic32", N=N, dt=0.004, order=4)
    phi, pi = inputs.make_initial(cfg)
    outs = []
    for fused in (True, False):
        g, o = make_pair(pc, cfg)
        g.set_tile(tile)
        g.set_fused_tail(fused)
        start(g, o, phi, pi)
        g.step(2); g.step(1); o.step(3)
        compare(g, o, 2, 5e-12)
        kicks, scalars, flushes, _ = g.launch_counts()
        assert kicks == 9 and flushes == 1 and scalars == (2 if fused else 2 + 9)   # one deferred closing drift
        outs.append((g.read_fields(), g.energies()))
    (pa, qa), ea = outs[0]
    (pb, qb), eb = outs[1]
    assert rel_err_per_site(pa, pb) < 1e-13 and rel_err_per_site(qa, qb) < 1e-13
    assert rel(ea.a, eb.a) < 1e-14 and rel(ea.p_a, eb.p_a) < 1e-13


@pytest.mark.parametrize("tile,N,zc,precision", [(3, 200, 7, 64), (4, 136, 3, 64), (7, 136, 5, 64), (5, 264, 6, 32)])
def test_item_orders_agree(pc, tile, N, zc, precision):
    """pycool_set_item_order: the order in which (x-y tile, z-chunk) items are handed out -- plain x-y-z, regions of one
    tile row, ragged regions (tile rows not divisible by the region height), the automatic regions -- changes which
    block computes what and the index of every partial sum, nothing else: after one stage the fields are bitwise
    equal, after several steps every order matches the oracle."""
    cfg = inputs.config("cfg0_chaotic32", N=N, dt=0.002, order=2)
    phi, pi = inputs.make_initial(cfg, precision=precision)
    nrows = lambda g: (N + g.kick_geometry()["ty"] - 1) // g.kick_geometry()["ty"]
    outs, seen = [], set()
    for order in (0, 1, -1, 40, 100):
        g = pc.from_config(cfg, precision=precision)
        g.set_tile(tile); g.set_zchunk(zc); g.set_item_order(order)
        geo = g.kick_geometry()
        assert geo["items"] > 148 * 3 and 1 <= geo["region"][1] <= nrows(g)
        if order == 0:
            assert geo["region"][1] == nrows(g)
        seen.add(geo["region"][1])
        g.set_fields(phi, pi); g.set_background(1.0)
        g.step(1)
        outs.append(g.read_fields())
    assert len(seen) >= 3                                          # really different orders, one of them ragged
    for p_, q_ in outs[1:]:
        assert np.array_equal(p_, outs[0][0]) and np.array_equal(q_, outs[0][1])
    cfg4 = inputs.config("cfg0_chaotic32", N=N if N < 150 else 72, dt=0.002, order=4)
    phi, pi = inputs.make_initial(cfg4, precision=precision)
    for order in (1, 40):
        g, o = make_pair(pc, cfg4, precision=precision)
        g.set_tile(tile); g.set_zchunk(3); g.set_item_order(order)
        start(g, o, phi, pi)
        g.step(2); o.step(2)
        if precision == 64:
            compare(g, o, 2, 2e-12)
        else:       # fp32 fields: the gradient energy of 1e-6 fluctuations is not resolved to 1e-5; fields and a are
            (pg, qg), (po, qo) = g.read_fields(), o.read_fields()
            assert rel_err_per_site(pg, po) <= 2e-5 and rel_err_per_site(qg, qo) <= 2e-5
            assert rel(g.energies().a, o.energies().a) <= 1e-6


@pytest.mark.parametrize("tile,N,zc", [(3, 136, 5), (4, 70, 1), (5, 260, 4), (7, 136, 1), (8, 72, 1)])
def test_persistent_launch_is_bitwise_the_one_block_per_item_launch(pc, tile, N, zc):
    """More work items than resident blocks (short z-chunks): every block walks several items with its TMA ring
    running on across them (ragged tiles, lattice faces and z-wrap included).  Partial sums are indexed by work
    item, so fields AND scalars are bitwise those of the one-block-per-item launch; and both match the oracle."""
    cfg = inputs.config("cfg0_chaotic32", N=N, dt=0.002, order=4)
    cfg["init"], cfg["amp"] = "white", 1e-3
    phi, pi = inputs.make_initial(cfg)
    outs = []
    for persistent in (True, False):
        g = pc.from_config(cfg)
        g.set_tile(tile); g.set_zchunk(zc); g.set_persistent(persistent)
        g.set_fields(phi, pi); g.set_background(1.0)
        g.step(2)
        e = g.energies()
        outs.append((g.read_fields(), (e.a, e.p_a, e.pot, e.kin[0], e.grad[1])))
        if persistent:
            assert g.kick_geometry()["blocks"] > 148 * 3       # really more items than a B200 holds at once
    assert np.array_equal(outs[0][0][0], outs[1][0][0]) and np.array_equal(outs[0][0][1], outs[1][0][1])
    assert outs[0][1] == outs[1][1]
    if N <= 136:
        o = make_pair(pc, cfg)[1]
        o.set_fields(phi, pi); o.set_background(1.0); o.step(2)
        po, qo = o.read_fields()
        assert rel_err_per_site(outs[0][0][0], po) <= 2e-12 and rel_err_per_site(outs[0][0][1], qo) <= 2e-12


@pytest.mark.parametrize("precision", [64, 32])
def test_four_fields_auto_variant_fits_shared_memory(pc, precision):
    """nf = 4 at N > 64: the default 64 x 16 ring would need more than 227 KB in fp64; the automatic choice must
    fall back to a variant that fits (and still match the oracle)."""
    N, nf = 72, 4
    phi, pi = inputs.random_fields(N, nf, seed=11, mean=0.5, amp=0.1, precision=precision)
    kw = dict(order=2, dt=0.01, mpl=INF, precision=precision)
    m2 = [0.5 + f for f in range(nf)]
    g = pc.Lattice(N, 4.0, nf, pc.FREE, m2, **kw)
    o = oracle.Oracle(N, 4.0, nf, oracle.FREE, m2, **kw)
    geo = g.kick_geometry()
    assert geo["smem_bytes"] <= 227 * 1024 and geo["tma_stages"] > 0
    start(g, o, phi, pi, 1.0, 0.0)
    g.step(2); o.step(2)
    compare(g, o, nf, 5e-13 if precision == 64 else 1e-5, tol_scalar=1e-10 if precision == 64 else 1e-5, static=True)


@pytest.mark.parametrize("N,zc", [(6, 0), (40, 7), (70, 16), (136, 5), (260, 0)])
def test_one_field_variant_two_by_four_sites_per_thread(pc, N, zc):
    """Variant 9 (128 x 16 tile, 2 x 4 sites per thread: the automatic choice for one fp64 field above N = 64) on
    the oscillon model: ragged tiles in x and y, lattice faces, z-chunks, against the oracle."""
    cfg = inputs.config("cfg2_oscillon256", N=N)
    cfg["L"] = cfg["L"] * N / 256
    phi, pi = inputs.make_initial(cfg)
    g, o = make_pair(pc, cfg)
    g.set_tile(9); g.set_zchunk(zc)
    geo = g.kick_geometry()
    assert geo["variant"] == 9 and geo["threads"] == 256 and geo["tx"] == 128 and geo["ty"] == 16
    start(g, o, phi, pi)
    g.step(3); o.step(3)
    compare(g, o, 1, 5e-12)
    if N > 64:
        assert pc.from_config(cfg).kick_geometry()["variant"] == 9


# ------------------------------------------------------------------------------------- energies (row a7)
@pytest.mark.parametrize("name,N", [("cfg0_chaotic32", 32), ("cfg0_chaotic32", 70), ("cfg2_oscillon256", 136),
                                    ("cfg3_qball256", 40), ("cfg3_qball256", 6)])
@pytest.mark.parametrize("precision", [64, 32])
def test_energy_kernels_agree_with_each_other_and_the_oracle(pc, name, N, precision):
    """pycool_energies through the TMA-fed z-march (sum G = - sum psi D[psi], the paper's identity (2.17)) and through
    the plain kernel that evaluates (2.8) term by term, after a few steps, against the oracle's direct evaluation; ragged
    tiles, several z-chunks (N = 70, 136) and a lattice smaller than a tile (N = 6)."""
    cfg = inputs.config(name, N=N)
    cfg["L"] = cfg["L"] * N / inputs.config(name)["N"]
    phi, pi = inputs.make_initial(cfg, precision=precision)
    g, o = make_pair(pc, cfg, precision=precision)
    start(g, o, phi, pi)
    g.step(2); o.step(2)
    # fp32: one ulp of phi is 1e-3 of the Q-ball lattice's 1e-4 fluctuations, and G sums their squared differences
    tol = 1e-10 if precision == 64 else 1e-4
    eo = o.energies()
    es = []
    for tma in (True, False):
        g.set_energy_kernel(tma)
        n0 = g.launch_counts()[3]
        es.append(g.energies())
        assert g.launch_counts()[3] == n0 + 2
        check_scalars(es[-1], eo, cfg["nfields"], tol)
    a, b = es
    for f in range(cfg["nfields"]):
        assert rel(a.grad[f], b.grad[f]) <= (1e-12 if precision == 64 else 1e-6)
        # sum phi D[phi] = phi_0 sum D + sum dphi D with sum D = 0 up to rounding: the order of the sum shows at 1e-10
        # (condition number sum|phi D| / |sum phi D| ~ 3e5 on this lattice; fp32 fields: compared at fp32 accuracy)
        assert rel(a.kin[f], b.kin[f]) <= 1e-13
        assert rel(a.sum_phiDphi[f], b.sum_phiDphi[f]) <= (1e-9 if precision == 64 else 1e-6)
        assert rel(a.grad[f], a.sum_phiDphi[f]) <= (1e-9 if precision == 64 else 1e-4)      # (2.17)
    assert rel(a.pot, b.pot) <= 1e-13 and rel(a.rho, b.rho) <= 1e-12


# ------------------------------------------------------------------------------------- adaptive conformal step
@pytest.mark.parametrize("order,fused", [(2, True), (4, True), (4, False), (6, True)])
def test_adaptive_step_matches_oracle(pc, order, fused):
    """Constant physical-time increments: the conformal length dt / a_n of every step is formed on
    the device from the a the step starts with; fields, a, p_a and the accumulated eta against the oracle."""
    cfg = inputs.config("cfg0_chaotic32", N=20, dt=0.004, order=order)
    phi, pi = inputs.make_initial(cfg)
    g, o = make_pair(pc, cfg)
    g.set_fused_tail(fused)
    start(g, o, phi, pi)
    g.set_adaptive(True); o.set_adaptive(True)
    g.step(2); g.step(3); o.step(5)
    compare(g, o, 2, 5e-12, tol_eta=1e-13)
    eg, eo = g.energies(), o.energies()
    assert eg.a > 1.001 and 0 < eo.eta < 5 * cfg["dt"]             # expanding: the steps did shrink
    assert rel(eg.eta, eo.eta) <= 1e-13
    h = pc.from_config(cfg)                                       # one call == split calls, bitwise
    h.set_fused_tail(fused)
    h.set_fields(phi, pi); h.set_background(1.0); h.set_adaptive(True)
    h.step(5)
    assert np.array_equal(h.read_fields()[0], g.read_fields()[0]) and h.energies().eta == eg.eta


def test_adaptive_step_radiation_only_recurrence_on_gpu(pc):
    """a' is constant in a radiation-only universe, so a_{n+1} = a_n + C dt / a_n exactly (same closed form that
    pins the oracle, P14), here for the device-side scalar update."""
    N, mpl, rg, dt, n = 8, 1.5, 3.0, 0.02, 40
    g = pc.Lattice(N, 1.0, 1, pc.FREE, [0.0], order=4, dt=dt, mpl=mpl, rho_gamma0=rg)
    z = np.zeros((1, N, N, N))
    g.set_fields(z, z); g.set_background(1.0); g.set_adaptive(True)
    g.step(n)
    C = math.sqrt(rg / 3) / mpl
    a, eta = np.longdouble(1), np.longdouble(0)
    for _ in range(n):
        hh = np.longdouble(dt) / a
        a, eta = a + np.longdouble(C) * hh, eta + hh
    e = g.energies()
    assert abs(e.a - float(a)) < 1e-13 and abs(e.eta - float(eta)) < 1e-13 and e.residual < 1e-13


def test_bitwise_reproducible(pc):
    cfg = inputs.config("cfg0_chaotic32", N=48)
    phi, pi = inputs.make_initial(cfg)
    outs = []
    for _ in range(2):
        g = pc.from_config(cfg)
        g.set_fields(phi, pi)
        g.set_background(1.0)
        g.step(5)
        p, q = g.read_fields()
        e = g.energies()
        outs.append((p.copy(), q.copy(), e.a, e.p_a, e.kin[0], e.grad[1], e.pot))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    assert outs[0][2:] == outs[1][2:]


def test_step_split_equals_one_call(pc):
    """pycool_step(3) and three pycool_step(1) calls are bitwise the same: the closing half drift of a call is
    deferred and merges with the next call's opening drift like two stages of one call; pycool_flush in between
    applies it separately instead (agreement to rounding)."""
    cfg = inputs.config("cfg0_chaotic32", N=24)
    phi, pi = inputs.make_initial(cfg)
    a, b = pc.from_config(cfg), pc.from_config(cfg)
    for g in (a, b):
        g.set_fields(phi, pi)
        g.set_background(1.0)
    a.step(3)
    for _ in range(3):
        b.step(1)
    c = pc.from_config(cfg)
    c.set_fields(phi, pi)
    c.set_background(1.0)
    for _ in range(3):
        c.step(1)
        c.flush()
    assert a.launch_counts()[2] == 0 and b.launch_counts()[2] == 0 and c.launch_counts()[2] == 3
    pa, qa = a.read_fields()
    pb, qb = b.read_fields()
    pc_, qc = c.read_fields()
    assert a.launch_counts()[2] == 1 and c.launch_counts()[2] == 3
    assert np.array_equal(pa, pb) and np.array_equal(qa, qb)
    assert a.energies().a == b.energies().a and a.energies().p_a == b.energies().p_a
    assert rel_err_per_site(pa, pc_) < 1e-14 and rel_err_per_site(qa, qc) < 1e-14
    assert rel(a.energies().a, c.energies().a) < 1e-14 and abs(a.energies().eta - 3 * cfg["dt"]) < 1e-15


# ------------------------------------------------------------------------------------- free model, stencils
@pytest.mark.parametrize("nf", [1, 2, 3, 4])
@pytest.mark.parametrize("stencil", [(0, 0, 0, 0), SEVEN_POINT])
def test_free_fields_static_background(pc, nf, stencil):
    N = 18
    phi, pi = inputs.random_fields(N, nf, seed=nf, mean=0.5, amp=0.1)
    kw = dict(order=4, dt=0.01, mpl=INF, stencil=stencil)
    m2 = [0.5 + f for f in range(nf)]
    g = pc.Lattice(N, 4.0, nf, pc.FREE, m2, **kw)
    o = oracle.Oracle(N, 4.0, nf, oracle.FREE, m2, **kw)
    start(g, o, phi, pi, 1.0, 0.0)
    g.step(4); o.step(4)
    compare(g, o, nf, 5e-13, static=True)


def test_kick_alone_gives_the_laplacian(pc):
    """V = 0, static, one 2nd-order step from pi = 0: pi' = dt D[phi + dt/2 * 0]/dx^2, so the GPU stencil is
    compared with the oracle's D of (2.7) directly, site by site."""
    N, L, dt = 21, 3.0, 0.125
    phi, _ = inputs.random_fields(N, 1, seed=5, mean=1.0, amp=1e-5)
    g = pc.Lattice(N, L, 1, pc.FREE, [0.0], order=2, dt=dt, mpl=INF)
    o = oracle.Oracle(N, L, 1, oracle.FREE, [0.0], order=2, dt=dt, mpl=INF)
    zero = np.zeros_like(phi)
    start(g, o, phi, zero, 1.0, 0.0)
    D = o.laplacian(0)
    g.step(1)
    _, q = g.read_fields()
    want = dt * D / (L / N) ** 2
    # fluctuations are 1e-5 on a mean of 1: a weight-form sum would lose 5 digits here
    assert np.max(np.abs(q[0] - want)) <= 1e-13 * np.max(np.abs(want))


# ------------------------------------------------------------------------------------- invariants on the GPU
def test_time_reversal_on_gpu(pc):
    cfg = inputs.config("cfg0_chaotic32", N=24, dt=0.004)
    phi, pi = inputs.make_initial(cfg)
    g = pc.from_config(cfg)
    g.set_fields(phi, pi)
    g.set_background(1.0)
    e0 = g.energies()
    g.step(10)
    g.set_dt(-cfg["dt"])
    g.step(10)
    p, q = g.read_fields()
    assert rel_err_per_site(p, phi) < 1e-12 and rel_err_per_site(q, pi) < 1e-12
    assert rel(g.energies().a, e0.a) < 1e-13


def test_nonfinite_is_reported_and_sticky(pc):
    cfg = inputs.config("cfg0_chaotic32", N=16)
    phi, pi = inputs.make_initial(cfg)
    bad = pi.copy()
    bad[1, 3, 4, 5] = np.inf
    g = pc.from_config(cfg)
    g.set_fields(phi, bad)
    g.set_background(1.0, -1.0e5)
    g.step(1)
    with pytest.raises(pc.PycoolError) as ei:
        g.sync()
    assert ei.value.code == pc.ENONFINITE
    with pytest.raises(pc.PycoolError):
        g.step(1)
    g.set_fields(phi, pi)                                    # clears the flag
    g.set_background(1.0)
    g.step(1)
    g.sync()


def test_state_errors(pc):
    g = pc.Lattice(8, 1.0, 1, pc.FREE, [1.0])
    with pytest.raises(pc.PycoolError) as ei:
        g.step(1)
    assert ei.value.code == pc.ESTATE
    with pytest.raises(pc.PycoolError):
        g.set_background(-1.0, 0.0)


# ------------------------------------------------------------------------------------- fp32 option
@pytest.mark.parametrize("tile", [-1, 1, 3, 6])
def test_fp32_one_step(pc, tile):
    cfg = inputs.config("cfg0b_chaotic32_resolved", N=40)
    cfg["amp"] = 1e-3
    phi, pi = inputs.make_initial(cfg, precision=32)
    g, o = make_pair(pc, cfg, precision=32)
    g.set_tile(tile)
    start(g, o, phi, pi)
    g.step(1); o.step(1)
    pg, qg = g.read_fields()
    po, qo = o.read_fields()
    assert pg.dtype == np.float32
    assert rel_err_per_site(pg, po) <= 1e-5 and rel_err_per_site(qg, qo) <= 1e-5
    check_scalars(g.energies(), o.energies(), 2, tol=1e-5)


@pytest.mark.parametrize("N,zc", [(72, 5), (136, 7), (264, 0)])
def test_fp32_x_quads(pc, N, zc):
    """Variant 11 (fp32 only): 4 x 1 sites per thread, float4 accesses.  Same per-site arithmetic as the x-pair
    variants, so after one stage the fields are bitwise those of variant 5; several steps against the fp32 oracle;
    ragged tiles (N = 72: less than one tile wide; 136, 264: 128 + 8), lattice faces, z-chunks.  Needs N % 4 == 0."""
    cfg = inputs.config("cfg0_chaotic32", N=N, dt=0.002, order=2)
    phi, pi = inputs.make_initial(cfg, precision=32)
    outs = []
    for tile in (5, 11):
        g = pc.from_config(cfg, precision=32)
        g.set_tile(tile); g.set_zchunk(zc)
        assert g.kick_geometry()["variant"] == tile
        g.set_fields(phi, pi); g.set_background(1.0)
        g.step(1)
        outs.append(g.read_fields())
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    cfg4 = inputs.config("cfg0_chaotic32", N=min(N, 136), dt=0.002, order=4)
    phi, pi = inputs.make_initial(cfg4, precision=32)
    g, o = make_pair(pc, cfg4, precision=32)
    g.set_tile(11); g.set_zchunk(zc)
    start(g, o, phi, pi)
    g.step(2); o.step(2)
    (pg, qg), (po, qo) = g.read_fields(), o.read_fields()
    assert rel_err_per_site(pg, po) <= 2e-5 and rel_err_per_site(qg, qo) <= 2e-5
    assert rel(g.energies().a, o.energies().a) <= 1e-6
    with pytest.raises(pc.PycoolError) as ei:                     # N = 70: even, but not whole quads
        h = pc.from_config(inputs.config("cfg0_chaotic32", N=70, dt=0.002), precision=32)
        h.set_tile(11)
    assert ei.value.code == pc.EINVAL
    with pytest.raises(pc.PycoolError) as ei:                     # fp64: not built
        h = pc.from_config(inputs.config("cfg0_chaotic32", N=72, dt=0.002))
        h.set_tile(11)
    assert ei.value.code == pc.EINVAL


# ------------------------------------------------------------------------------------- full size, bench configs
def replicate_on_device(arr, r, dev):
    import torch
    return torch.from_numpy(arr).to(dev).repeat(1, r, r, r).contiguous()


def worst_replica_error(big, small_np, r, base, dev):
    """max over every replica and every site of |big - small| / max(|small|, rms(small)) (reading G18), on the device."""
    import torch
    worst = 0.0
    for f in range(small_np.shape[0]):
        want = torch.from_numpy(small_np[f]).to(dev)
        rms = float(want.double().pow(2).mean().sqrt())
        den = torch.clamp(want.abs(), min=rms)
        blocks = big[f].view(r, base, r, base, r, base)
        for iz in range(r):
            d = (blocks[iz] - want[:, None, :, None, :]).abs() / den[:, None, :, None, :]
            worst = max(worst, float(d.max()))
    return worst


# (workload, N, base, order, precision, per-site tolerance after `steps` steps, steps, kernel variant expected)
FULL_SIZE = [
    ("cfg4_chaotic512", 512, 32, 4, 64, 2e-12, 2, 3),       # the bench default
    ("cfg4_chaotic512", 512, 32, 6, 64, 4e-12, 1, 3),
    ("cfg4_chaotic512", 512, 32, 4, 32, 1e-5, 1, 11),       # fp32: x quads
    ("cfg1_chaotic128", 128, 32, 6, 64, 2e-12, 2, 3),       # configs[1]: order 6 at its own size
    ("cfg2_oscillon256", 256, 32, 4, 64, 2e-12, 2, 9),      # configs[2]: one field, 2 x 4 sites per thread
    ("cfg3_qball256", 256, 32, 4, 64, 2 * QBALL_TOL_1STEP, 2, 12),  # configs[3]: QBall x (2 x 1 sites, 4 blocks/SM)
    ("cfg4_chaotic1024", 1024, 32, 4, 64, 2e-12, 1, 3),     # configs[4]: 69 GB of state, byte offsets > 2^34
    ("cfg4_chaotic1024", 1024, 32, 4, 32, 1e-5, 1, 11),     # 2^31 elements per array
]


@pytest.mark.parametrize("name,N,base,order,precision,tol,steps,variant", FULL_SIZE)
def test_full_size_periodic_replication(pc, name, N, base, order, precision, tol, steps, variant):
    """Every configuration BASELINE.md's table quotes, at its full size and in the automatic launch geometry that
    bench.py times: the input is a base^3 lattice replicated periodically; the method is translation-equivariant,
    so every output site of every replica must equal the oracle's base^3 evolution of the same tile (lattice sums
    scale with the volume, a is unchanged).  Input, output and comparison stay on the device
    (set_fields_device / read_fields_device): 1024^3 x 2 fp64 is 17 GB per array."""
    import torch
    r = N // base
    full = inputs.config(name)
    small = inputs.config(name, N=base, order=order)
    small["L"] = full["L"] * base / N                        # same dx and dt as the full configuration
    small["dt"] = full["dt"]
    phi_s, pi_s = inputs.make_initial(small, precision=precision)
    big = inputs.config(name, order=order)
    g = pc.from_config(big, precision=precision)
    kw = dict(mpl=small["mpl"], rho_gamma0=small["rho_gamma0"], rho_m0=small["rho_m0"], precision=precision)
    o = oracle.Oracle(base, small["L"], small["nfields"], small["model"], small["p"], order=order, dt=small["dt"], **kw)
    dev = g.device
    tp, tq = replicate_on_device(phi_s, r, dev), replicate_on_device(pi_s, r, dev)
    g.set_fields(tp, tq)
    del tp, tq
    torch.cuda.empty_cache()
    # the radiation background of cfg3 is derived from H0, not from the lattice: set a, p_a explicitly on both
    o.set_fields(phi_s, pi_s)
    o.set_background(1.0)
    p_a_small = o.energies().p_a
    g.set_background(1.0, p_a_small * r ** 3)                # p_a is extensive: -6 V_L mpl^2 a'
    geo = g.kick_geometry()
    assert geo["variant"] == variant and geo["tma_stages"] > 0, geo
    g.step(steps); o.step(steps)
    po, qo = o.read_fields()
    eg, eo = g.energies(), o.energies()
    ts = 1e-10 if precision == 64 else 1e-4
    nf = small["nfields"]
    assert rel(eg.a, eo.a) < (1e-12 if precision == 64 else 1e-6) and rel(eg.p_a / r ** 3, eo.p_a) < ts
    assert rel(eg.kin[0], eo.kin[0]) < ts and rel(eg.grad[nf - 1], eo.grad[nf - 1]) < 10 * ts and rel(eg.pot, eo.pot) < ts
    pg, qg = g.read_fields_device()
    e_phi = worst_replica_error(pg, po, r, base, dev)
    del pg
    e_pi = worst_replica_error(qg, qo, r, base, dev)
    print("%s %d^3 order %d fp%d variant %d zc %d: per-site error phi %.2e pi %.2e after %d step(s)"
          % (name, N, order, precision, geo["variant"], geo["zchunk"], e_phi, e_pi, steps))
    assert e_phi <= tol and e_pi <= tol, (e_phi, e_pi)


def test_context_on_a_second_device(pc):
    """A Lattice made while ANOTHER device is current, and two Lattices on two GPUs driven from one thread: the
    library records the device of the work buffer and switches to it for every call (shared-memory opt-in and
    occupancy are per context, not per process).  Needs two GPUs."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    cfg = inputs.config("cfg0_chaotic32", N=72, dt=0.002)
    phi, pi = inputs.make_initial(cfg)
    torch.cuda.set_device(0)
    a = pc.from_config(cfg, device="cuda:0")
    b = pc.from_config(cfg, device="cuda:1")                 # made while cuda:0 is current
    outs = []
    for g in (a, b):
        g.set_fields(phi, pi); g.set_background(1.0)
        g.step(2)
        outs.append(g.read_fields())
    assert torch.cuda.current_device() == 0
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


# ------------------------------------------------------------------------------------- memory safety without a sanitizer
@pytest.mark.parametrize("name,N,tile,zc,precision", [("cfg0_chaotic32", 72, 3, 5, 64), ("cfg0_chaotic32", 40, 4, 3, 64),
                                                      ("cfg0_chaotic32", 72, 5, 7, 32), ("cfg3_qball256", 40, 7, 3, 64),
                                                      ("cfg2_oscillon256", 130, 9, 9, 64), ("cfg0_chaotic32", 21, -1, 0, 64)])
def test_nothing_is_written_outside_the_work_buffer_and_nothing_uninitialised_is_read(pc, name, N, tile, zc, precision):
    """compute-sanitizer is closed on this pool (profiles/r2_sanitizer.md), so the two properties it would check are
    tested directly through the C ABI with a caller-owned work buffer (pycool_create_ext): (i) guard bands of 1 MiB on
    both sides of the buffer, filled with a byte pattern, are intact after uploads, steps with the energy log, both
    energy kernels, spectra and downloads; (ii) the buffer itself starts as NaN bytes (0xFF), so any element the
    library reads without having written it first would surface as a non-finite field or sum."""
    import ctypes as C
    import torch
    cfg = inputs.config(name, N=N, order=2) if name != "cfg0_chaotic32" else inputs.config(name, N=N, order=2, dt=0.0025)
    if name != "cfg0_chaotic32":
        cfg["L"] = cfg["L"] * N / inputs.config(name)["N"]
    nf = cfg["nfields"]
    phi, pi = inputs.make_initial(cfg, precision=precision)
    need = pc.work_bytes(N, nf, precision)
    guard = 1 << 20
    buf = torch.full((need + 2 * guard + 256,), 0xFF, dtype=torch.uint8, device="cuda:0")
    base = (buf.data_ptr() + guard + 255) // 256 * 256
    off = base - buf.data_ptr()
    buf[:off] = 0xA5
    buf[off + need:] = 0xA5
    L = pc.lib()
    mp = pc.make_params(cfg["model"], cfg["p"], mpl=cfg["mpl"], rho_gamma0=cfg["rho_gamma0"], rho_m0=cfg["rho_m0"],
                        precision=precision)
    h = C.c_void_p()
    stream = torch.cuda.current_stream()
    assert L.pycool_create_ext(C.byref(h), N, cfg["L"], nf, C.byref(mp), 2, cfg["dt"], base, need, stream.cuda_stream) == 0
    try:
        if tile >= 0:
            assert L.pycool_set_tile(h, tile) == 0
        if zc > 0:
            assert L.pycool_set_zchunk(h, zc) == 0
        assert L.pycool_set_fields(h, phi.ctypes.data, pi.ctypes.data) == 0
        assert L.pycool_set_background(h, 1.0, math.nan) == 0
        assert L.pycool_set_energy_cadence(h, 1, 4) == 0
        assert L.pycool_step(h, 2) == 0 and L.pycool_step(h, 1) == 0
        e = pc.Energy()
        assert L.pycool_energies(h, C.byref(e)) == 0
        assert L.pycool_set_energy_kernel(h, 0) == 0 and L.pycool_energies(h, C.byref(e)) == 0
        if N % 2 == 0:
            nb = int(math.floor(math.sqrt(3.0) * N / 2.0 + 0.5)) + 1
            a, b, c_ = (C.c_double * nb)(), (C.c_double * nb)(), (C.c_double * nb)()
            assert L.pycool_mode_spectra(h, 0, 1.0, nb, a, b, c_) == 0
            assert all(math.isfinite(x) for x in a) and all(math.isfinite(x) for x in b)
        out_phi, out_pi = np.empty_like(phi), np.empty_like(pi)
        assert L.pycool_read_fields(h, out_phi.ctypes.data, out_pi.ctypes.data) == 0
    finally:
        L.pycool_destroy(h)
    torch.cuda.synchronize()
    assert bool((buf[:off] == 0xA5).all()) and bool((buf[off + need:] == 0xA5).all())
    assert np.all(np.isfinite(out_phi)) and np.all(np.isfinite(out_pi))
    for v in (e.a, e.p_a, e.rho, e.pressure, e.pot) + tuple(e.kin[:nf]) + tuple(e.grad[:nf]):
        assert math.isfinite(v)


# ------------------------------------------------------------------------------------- cooperative multi-stage launches
@pytest.mark.parametrize("name,N,order,precision,kw", [("cfg0_chaotic32", 32, 4, 64, {}), ("cfg1_chaotic128", 128, 6, 64, {}),
                                                       ("cfg0_chaotic32", 64, 4, 32, {}), ("cfg2_oscillon256", 48, 4, 64, {}),
                                                       ("cfg3_qball256", 40, 4, 64, {}), ("cfg0_chaotic32", 24, 8, 64, {"adaptive": True})])
def test_cooperative_launch_is_bitwise_the_launch_per_stage_path(pc, name, N, order, precision, kw):
    """Small lattices run several stages per cooperative launch with a grid barrier between stages
    (pycool_set_cooperative, default on).  Same items, same partial-sum indices, same order of every sum: fields,
    scalars, energies and the energy log are bitwise those of the launch-per-stage path, across split calls, odd and
    even stage counts per launch (buffer parity) and log points in the middle of a call; and the default path really is
    the cooperative one (checked through the oracle as well at N = 32)."""
    cfg = inputs.config(name, N=N, order=order) if name != "cfg0_chaotic32" or N == 32 else inputs.config(name, N=N, order=order, dt=0.0025)
    if name in ("cfg2_oscillon256", "cfg3_qball256"):
        cfg["L"] = cfg["L"] * N / inputs.config(name)["N"]
    nf = cfg["nfields"]
    phi, pi = inputs.make_initial(cfg, precision=precision)

    def run(coop):
        g = pc.from_config(cfg, precision=precision)
        g.set_cooperative(coop)
        g.set_fields(phi, pi); g.set_background(1.0)
        if kw.get("adaptive"):
            g.set_adaptive(True)
        g.set_energy_cadence(2, 8)
        g.step(3); g.step(1); g.step(5)
        log, total = g.read_energy_log()
        e = g.energies()
        return g.read_fields(), e, log, total, g.launch_counts()[0]

    (pa, qa), ea, la, ta, na = run(True)
    (pb, qb), eb, lb, tb, nb = run(False)
    stages = {2: 1, 4: 3, 6: 7, 8: 15}[order]
    assert na == nb == 9 * stages and ta == tb == 4
    assert np.array_equal(pa, pb) and np.array_equal(qa, qb)
    tup = lambda e: (e.a, e.p_a, e.eta, e.rho, e.pressure, e.pot, e.hubble) + tuple(e.kin[:nf]) + tuple(e.grad[:nf])
    assert tup(ea) == tup(eb)
    assert [tup(x) for x in la] == [tup(x) for x in lb]
    if N == 32:
        o = oracle.Oracle(N, cfg["L"], nf, cfg["model"], cfg["p"], order=order, dt=cfg["dt"], mpl=cfg["mpl"])
        o.set_fields(phi, pi); o.set_background(1.0)
        o.step(9)
        po, qo = o.read_fields()
        assert rel_err_per_site(pa, po) <= 1e-11 and rel_err_per_site(qa, qo) <= 1e-11
        assert rel(ea.a, o.energies().a) <= 1e-12
