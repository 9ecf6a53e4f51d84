"""Host-side checks of the C-ABI library that need no GPU: it builds, loads, exports every symbol
include/pycool.h declares, validates arguments, and refuses to run without a CUDA device."""
import ctypes as C
import math
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1201_5029_b200 import build
    build.build()
    from paper_1201_5029_b200 import binding
    return binding.lib()


def _declared():
    names = set()
    for h in ("pycool.h", "pycool_linear.h"):
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(pycool_[a-z0-9_]+)\s*\(", src))
    return names


def test_header_symbols_all_exported(L):
    from paper_1201_5029_b200 import binding
    declared = _declared()
    assert declared == set(binding.SYMBOLS)
    for name in declared:
        assert getattr(L, name) is not None


def test_only_abi_symbols_are_exported(L):
    import subprocess
    from paper_1201_5029_b200 import binding
    out = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    names = {ln.split()[-1] for ln in out.splitlines() if " T " in ln}
    assert {n for n in names if n.startswith("pycool_")} == set(binding.SYMBOLS)
    assert not any("oracle" in n for n in names)


def test_struct_sizes_match_header():
    """ctypes mirrors of pycool_params / pycool_energy / pycool_linear_background against a C compiler's view of the
    headers."""
    import subprocess
    import tempfile
    from paper_1201_5029_b200 import binding
    code = ('#include <stdio.h>\n#include "pycool_linear.h"\nint main(){printf("%zu %zu %zu\\n", sizeof(pycool_params), '
            'sizeof(pycool_energy), sizeof(pycool_linear_background));return 0;}\n')
    with tempfile.TemporaryDirectory() as d:
        src, exe = os.path.join(d, "s.c"), os.path.join(d, "s")
        open(src, "w").write(code)
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), src, "-o", exe], check=True)
        a, b, c = map(int, subprocess.run([exe], capture_output=True, text=True).stdout.split())
    assert a == C.sizeof(binding.Params) and b == C.sizeof(binding.Energy) and c == C.sizeof(binding.LinearBackground)


def test_linear_create_validates_then_needs_a_gpu(L):
    """include/pycool_linear.h: argument validation on the host, class count (reading G28), no CPU path."""
    import torch
    from paper_1201_5029_b200 import binding
    h = C.c_void_p()

    def create(N=8, Lbox=1.0, nf=1, model=binding.FREE, order=4, dt=0.1, **kw):
        mp = binding.make_params(model, kw.pop("p", (1.0,)), **kw)
        return L.pycool_linear_create(C.byref(h), N, Lbox, nf, C.byref(mp), order, dt)

    for bad in (dict(N=2), dict(Lbox=-1.0), dict(nf=5), dict(order=3), dict(dt=0.0), dict(model=9),
                dict(model=binding.CHAOTIC, nf=1), dict(model=binding.OSCILLON, nf=2), dict(mpl=-1.0),
                dict(stencil=(-5.0, 1.0, 0.0, 0.0)), dict(precision=32)):
        assert create(**bad) == binding.EINVAL, bad
        assert h.value is None and len(L.pycool_linear_last_error(None)) > 0
    for N in (3, 4, 7, 8, 256, 1024):
        M = N // 2
        assert L.pycool_linear_num_classes(N) == (M + 1) * (M + 2) * (M + 3) // 6
    assert L.pycool_linear_num_classes(2) == 0
    if not torch.cuda.is_available():
        assert create() == binding.ECUDA
        with pytest.raises(RuntimeError):
            binding.LinearLattice(8, 1.0, 1, binding.FREE, (1.0,))
    assert L.pycool_linear_step(None, 1, 0) == binding.EINVAL and L.pycool_linear_destroy(None) == binding.EINVAL


def test_linear_growth_static_validates_then_needs_a_gpu(L):
    """pycool_linear_growth_static: the size limit of its fixed scratch and its arguments are checked on the host,
    before anything touches a device."""
    import torch
    from paper_1201_5029_b200 import binding
    fake = 0x1000                                                  # never dereferenced: every call below is refused

    def call(N=8, nf=2, model=binding.CHAOTIC, order=4, nsteps=10, a=1.0, p_a=0.0, M=fake, room=None, **kw):
        room = L.pycool_linear_num_classes(N) if room is None else room
        try:
            binding.linear_growth_static(N, 1.0, nf, model, kw.pop("p", (1.0, 100.0)), order, 0.01, nsteps, a, p_a,
                                         (0.1,) * nf, (0.2,) * nf, M, room, **kw)
        except binding.PycoolError as e:
            return e.code, str(e)
        return binding.OK, ""

    for bad in (dict(N=2), dict(nf=1), dict(order=3), dict(nsteps=0), dict(a=0.0), dict(p_a=math.inf), dict(M=0),
                dict(room=3), dict(mpl=math.inf, p_a=math.nan), dict(precision=32)):
        assert call(**bad)[0] == binding.EINVAL, bad
    for order, stages in ((2, 1), (4, 3), (6, 7), (8, 15)):
        code, msg = call(order=order, nsteps=binding.LINEAR_STATIC_MAX_STAGES // stages + 1)
        assert code == binding.EINVAL and "PYCOOL_LINEAR_STATIC_MAX_STAGES = 4096" in msg
    if not torch.cuda.is_available():
        assert call()[0] == binding.ECUDA                          # valid arguments, no device: no CPU path
        assert call(order=2, nsteps=binding.LINEAR_STATIC_MAX_STAGES)[0] == binding.ECUDA   # the limit itself is allowed


def test_stage_weights_host_logic(L, golden_dir):
    from paper_1201_5029_b200 import binding
    from helpers import weights
    for order, n in ((2, 1), (4, 3), (6, 7), (8, 15)):
        w = binding.stage_weights(order)
        assert len(w) == n and w == w[::-1] and abs(sum(w) - 1) < 4e-15
        want = [float(x) for x in weights(golden_dir, order)]
        assert max(abs(a - b) for a, b in zip(w, want)) < 2e-16
    assert binding.stage_weights(3) == [] and binding.stage_weights(10) == []


def test_work_bytes(L):
    from paper_1201_5029_b200 import binding
    assert binding.work_bytes(2, 1) == 0 and binding.work_bytes(32, 5) == 0 and binding.work_bytes(32, 1, 16) == 0
    b64, b32 = binding.work_bytes(64, 2, 64), binding.work_bytes(64, 2, 32)
    assert b64 >= 2 * 2 * 64 ** 3 * 8 and b32 >= 2 * 2 * 64 ** 3 * 4 and b32 < b64
    assert binding.work_bytes(1024, 2, 64) >= 2 * 2 * 1024 ** 3 * 8


def test_create_validates_then_needs_a_gpu(L):
    import torch
    from paper_1201_5029_b200 import binding
    h = C.c_void_p()

    def create(N=8, Lbox=1.0, nf=1, model=binding.FREE, order=4, dt=0.1, **kw):
        mp = binding.make_params(model, kw.pop("p", (1.0,)), **kw)
        return L.pycool_create(C.byref(h), N, Lbox, nf, C.byref(mp), order, dt)

    for bad in (dict(N=2), dict(Lbox=0.0), dict(nf=0), dict(nf=5), dict(order=5), dict(dt=0.0),
                dict(dt=math.nan), dict(model=7), dict(model=binding.CHAOTIC, nf=1),
                dict(model=binding.OSCILLON, nf=2), dict(mpl=0.0), dict(stencil=(-5.0, 1.0, 0.0, 0.0)),
                dict(precision=16), dict(model=binding.QBALL, nf=2, p=(1.0, -0.1, 0.0, 0.0))):
        assert create(**bad) == binding.EINVAL, bad
        assert h.value is None
        assert len(L.pycool_last_error(None)) > 0
    if not torch.cuda.is_available():
        assert create() == binding.ECUDA                      # no CPU path, by design
        assert b"no CPU path" in L.pycool_last_error(None)
        with pytest.raises(RuntimeError):
            binding.Lattice(8, 1.0, 1, binding.FREE, (1.0,))
    assert L.pycool_step(None, 1) == binding.EINVAL
    assert L.pycool_destroy(None) == binding.EINVAL


def test_product_does_not_touch_the_oracle():
    """Nothing under the package or include/ may import, include or link the oracle."""
    pkg = os.path.join(ROOT, "paper_1201_5029_b200")
    for base, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(base, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert not re.search(r'#\s*include\s*["<][^">]*oracle', txt) and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1201_5029_b200" not in txt and "from paper_1201_5029_b200" not in txt, f
            assert "pycool.h" not in txt or f == "oracle.h", f


def test_device_log_against_libm(tmp_path):
    """The Q-ball kick uses its own fp64 logarithm (potentials.cuh: log_pos, __host__ __device__).  The same source
    compiled for the host against logl: <= 2.5 ulp over 1e-300..1e300, around 1, at the sqrt(2) range switch,
    and for a subnormal argument."""
    import subprocess
    exe = str(tmp_path / "log_pos_check")
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc, "-O2", "-std=c++17", "-o", exe, os.path.join(ROOT, "tests", "log_pos_check.cu")], check=True,
                   capture_output=True)
    out = subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()
    assert out[0] == "worst" and float(out[1]) <= 2.5, out
    sub = out[out.index("sub") + 1:]
    assert abs(float(sub[0]) - float(sub[1])) <= 1e-13 * abs(float(sub[1]))
