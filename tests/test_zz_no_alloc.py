"""pycool_linear_growth_static (include/pycool_linear.h): the growth matrices of (2.51) computed with no allocation --
scratch in a fixed device array of the library -- against the existing path, pycool_linear_step(.., GROWTH) +
pycool_linear_growth, which runs the same kernels on cudaMalloc'ed scratch.  `-m gpu`.

Collected last on purpose (the name): the suite runs with `pytest -x`, and a failure here must not hide the others.
Runs alone in a fresh process or after the other tests: it shares nothing with them but the library."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

INF = math.inf
# (model, nf, p, mpl, phi0, pi0, N, order, nsteps): several field counts, stage counts and table lengths
CASES = {
    "chaotic": dict(nf=2, model=1, p=(1.0, 1.0e4), mpl=1.0, phi0=(0.9676, 1e-3), pi0=(-0.71, 2e-3), N=24, order=4, nsteps=30),
    "qball": dict(nf=2, model=3, p=(1.0, -0.1, 1.0, 0.0), mpl=30.0, phi0=(1.4, 0.1), pi0=(0.0, 0.7), N=9, order=6, nsteps=5),
    "free4_static": dict(nf=4, model=0, p=(1.0, 2.5, 0.3, 4.0), mpl=INF, phi0=(0.5, -0.2, 0.1, 0.3),
                         pi0=(0.1, 0.2, -0.3, 0.0), N=6, order=8, nsteps=7),
    "oscillon_full_table": dict(nf=1, model=2, p=(1.0, 1.0, 0.3), mpl=335.41, phi0=(2.0,), pi0=(0.05,), N=16, order=2,
                                nsteps=4096),          # exactly PYCOOL_LINEAR_STATIC_MAX_STAGES stages
}
L, DT = 4.0, 0.002


@pytest.fixture(scope="module")
def pc():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1201_5029_b200 import build
    build.build()
    from paper_1201_5029_b200 import binding
    binding.lib()
    return binding


def p_a_of(c):
    return 0.0 if c["mpl"] == INF else math.nan          # NaN: solve (2.18), as the tests of the existing path do


def existing_path(pc, c):
    g = pc.LinearLattice(c["N"], L, c["nf"], c["model"], c["p"], order=c["order"], dt=DT, mpl=c["mpl"])
    g.set_background(1.0, p_a_of(c), c["phi0"], c["pi0"])
    g.step(c["nsteps"], pc.GROWTH)
    M = g.growth()
    g.close()
    return M


def static_call(pc, c, out, stream=0):
    pc.linear_growth_static(c["N"], L, c["nf"], c["model"], c["p"], c["order"], DT, c["nsteps"], 1.0, p_a_of(c), c["phi0"],
                            c["pi0"], out.data_ptr(), out.numel() // (4 * c["nf"] ** 2), stream, mpl=c["mpl"])


def new_out(pc, c):
    import torch
    n = int(pc.lib().pycool_linear_num_classes(c["N"]))
    return torch.full((n, 2 * c["nf"], 2 * c["nf"]), math.nan, dtype=torch.float64, device="cuda:0")


def assert_same(got, want):
    # the tolerance of tests/test_gpu_linear.py for growth matrices; the two paths run the same kernels on the same
    # numbers, so in fact they agree bit for bit
    assert got.shape == want.shape and np.all(np.isfinite(got))
    assert np.max(np.abs(got - want)) <= 1e-12 * np.max(np.abs(want))
    assert np.array_equal(got, want)


def test_two_calls_in_a_row_match_the_existing_path(pc):
    import torch
    torch.cuda.set_device(0)
    want = {name: existing_path(pc, c) for name, c in CASES.items()}
    # call after call on one stream, no synchronisation in between: each call finds the previous call's background,
    # weights and table in the shared scratch and must not be affected by them
    order = ["chaotic", "oscillon_full_table", "chaotic", "free4_static", "qball", "chaotic"]
    outs = [new_out(pc, CASES[name]) for name in order]
    for name, out in zip(order, outs):
        static_call(pc, CASES[name], out)
    torch.cuda.synchronize()
    for name, out in zip(order, outs):
        assert_same(out.cpu().numpy(), want[name])
    # and with a synchronisation after every call, on a stream of the caller's
    s = torch.cuda.Stream()
    for name in ("qball", "qball", "free4_static"):
        out = new_out(pc, CASES[name])
        static_call(pc, CASES[name], out, s.cuda_stream)
        s.synchronize()
        assert_same(out.cpu().numpy(), want[name])


def test_a_call_allocates_nothing(pc):
    """Free device memory does not drop across calls (the first call of a process may load the kernels' module; that
    is why one call comes first)."""
    import gc
    import torch
    torch.cuda.set_device(0)
    c = CASES["chaotic"]
    out = new_out(pc, c)
    static_call(pc, c, out)
    torch.cuda.synchronize()
    gc.collect()
    free0, _ = torch.cuda.mem_get_info(0)
    for _ in range(3):
        static_call(pc, c, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info(0)
    assert free1 >= free0        # nothing taken (objects of earlier tests may be collected, and freed, at any time)


def test_limits_and_arguments(pc):
    import torch
    torch.cuda.set_device(0)
    c = dict(CASES["chaotic"])
    out = new_out(pc, c)
    assert pc.LINEAR_STATIC_MAX_STAGES == 4096
    for order, stages in ((2, 1), (4, 3), (6, 7), (8, 15)):
        too_many = pc.LINEAR_STATIC_MAX_STAGES // stages + 1
        with pytest.raises(pc.PycoolError) as ei:
            static_call(pc, dict(c, order=order, nsteps=too_many), out)
        assert ei.value.code == pc.EINVAL and "PYCOOL_LINEAR_STATIC_MAX_STAGES" in str(ei.value)
    with pytest.raises(pc.PycoolError) as ei:                    # room for fewer classes than the lattice has
        pc.linear_growth_static(c["N"], L, 2, c["model"], c["p"], 4, DT, 1, 1.0, 0.0, c["phi0"], c["pi0"], out.data_ptr(),
                                out.shape[0] - 1)
    assert ei.value.code == pc.EINVAL
    host = np.zeros(out.numel())
    with pytest.raises(pc.PycoolError) as ei:                    # host memory where device memory is wanted
        pc.linear_growth_static(c["N"], L, 2, c["model"], c["p"], 4, DT, 1, 1.0, 0.0, c["phi0"], c["pi0"], host.ctypes.data,
                                out.shape[0])
    assert ei.value.code == pc.EINVAL and "device memory" in str(ei.value)
    for bad in (dict(nsteps=0), dict(order=5), dict(N=2)):
        with pytest.raises(pc.PycoolError) as ei:
            static_call(pc, dict(c, **bad), out)
        assert ei.value.code == pc.EINVAL
    torch.cuda.synchronize()
    assert bool(torch.isnan(out).all())                          # no refused call wrote anything
    static_call(pc, c, out)                                      # and the entry point still works after refusals
    torch.cuda.synchronize()
    assert_same(out.cpu().numpy(), existing_path(pc, c))
