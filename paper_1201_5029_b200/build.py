"""Build paper_1201_5029_b200/libpycool.so (sm_100a only) with nvcc, in-tree.

    python -m paper_1201_5029_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  `-lineinfo` keeps ncu's source page usable; `-Xptxas -v` output
(registers, spills, shared memory per kernel) is written next to the library as libpycool.ptxas.txt.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpycool.so")
SOURCES = [os.path.join(CSRC, "pycool.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "kernels.cuh"), os.path.join(CSRC, "kick_tma.cuh"), os.path.join(CSRC, "energy_tma.cuh"), os.path.join(CSRC, "init_fields.cuh"),
                  os.path.join(CSRC, "potentials.cuh"),
                  os.path.join(os.path.dirname(HERE), "include", "pycool.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-Xptxas", "-v",
         "-Xcompiler", "-fPIC,-fvisibility=hidden", "-shared", "-cudart", "static", "-ldl"]


def up_to_date():
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(d) <= t for d in DEPS)


def build(force=False, verbose=False):
    if not force and up_to_date():
        return LIB
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = [NVCC] + FLAGS + ["-o", tmp] + SOURCES
    r = subprocess.run(cmd, cwd=HERE, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    with open(os.path.join(HERE, "libpycool.ptxas.txt"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + r.stdout)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed (exit %d)" % r.returncode)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
