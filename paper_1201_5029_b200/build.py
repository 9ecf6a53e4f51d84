"""Build paper_1201_5029_b200/libpycool.so (sm_100a only) with nvcc, in-tree.

    python -m paper_1201_5029_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The kernel template instances of each model are their own translation unit
(csrc/models_*.cu), compiled in parallel, then linked with the ABI (csrc/pycool.cu).  `-lineinfo` keeps ncu's
source page usable; the `-Xptxas -v` output (registers, spills, shared memory per kernel) goes to
build/libpycool.ptxas.txt (untracked; `python -m paper_1201_5029_b200.build --regs` prints the table of it).
"""
import concurrent.futures
import glob
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libpycool.so")
PTXAS_LOG = os.path.join(OBJ, "libpycool.ptxas.txt")
SOURCES = [os.path.join(CSRC, "pycool.cu"), os.path.join(CSRC, "linear.cu")] + sorted(glob.glob(os.path.join(CSRC, "models_*.cu")))
DEPS = SOURCES + sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + sorted(glob.glob(os.path.join(CSRC, "*.h"))) + \
    sorted(glob.glob(os.path.join(os.path.dirname(HERE), "include", "*.h"))) + [os.path.abspath(__file__)]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
CFLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-Xptxas", "-v",
          "-Xfatbin", "-compress-all",      # ~190 kernel instances with line tables: 32 MB of cubin -> 10 MB
          "-Xcompiler", "-fPIC,-fvisibility=hidden"]
LFLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-ldl"]


def up_to_date():
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(d) <= t for d in DEPS)


def _compile(src):
    obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
    cmd = [NVCC] + CFLAGS + ["-c", "-o", obj, src]
    r = subprocess.run(cmd, cwd=HERE, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    return obj, " ".join(cmd) + "\n" + r.stdout, r.returncode


def build(force=False, verbose=False):
    if not force and up_to_date():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as ex:
        results = list(ex.map(_compile, SOURCES))
    log = "".join(out for _, out, _ in results)
    tmp = LIB + ".tmp%d" % os.getpid()
    rc = max(code for _, _, code in results)
    if rc == 0:
        cmd = [NVCC] + LFLAGS + ["-o", tmp] + [obj for obj, _, _ in results]
        r = subprocess.run(cmd, cwd=HERE, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        log += " ".join(cmd) + "\n" + r.stdout
        rc = r.returncode
    with open(PTXAS_LOG, "w") as fh:
        fh.write(log)
    if verbose or rc != 0:
        sys.stderr.write(log)
    if rc != 0:
        raise RuntimeError("nvcc failed (exit %d)" % rc)
    os.replace(tmp, LIB)
    return LIB


def register_table(pattern=""):
    """(kernel, registers, spill store bytes, spill load bytes) per compiled kernel, from the last build's log."""
    txt = open(PTXAS_LOG).read()
    ents = re.findall(r"Compiling entry function '(\S+)' for 'sm_100a'\nptxas info\s+: Function properties for \S+\n"
                      r"\s+(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads\n"
                      r"ptxas info\s+: Used (\d+) registers", txt)
    names = subprocess.run(["c++filt"] + [e[0] for e in ents], stdout=subprocess.PIPE, text=True).stdout.split("\n")
    rows = []
    for (_, _, ss, sl, regs), name in zip(ents, names):
        name = re.sub(r"\(.*", "", name.replace("pycool::", "").replace("void ", ""))
        if pattern in name:
            rows.append((name, int(regs), int(ss), int(sl)))
    return rows


if __name__ == "__main__":
    if "--regs" in sys.argv:
        rows = register_table(sys.argv[sys.argv.index("--regs") + 1] if len(sys.argv) > sys.argv.index("--regs") + 1 else "")
        for r in rows:
            print("%-90s %4d regs  spill %d/%d" % r)
        print("%d kernels, %d with spills" % (len(rows), sum(1 for r in rows if r[2] or r[3])))
    else:
        print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
