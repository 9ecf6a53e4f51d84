"""Build oracle/liboracle.so from oracle.cpp with plain g++ (no CUDA, no torch).

TEST INFRASTRUCTURE ONLY (see oracle.h).  `-ffp-contract=off` keeps every product and sum a separate
IEEE operation, so the oracle's arithmetic is exactly what oracle.cpp spells out.

    python -m oracle.build        # or: python oracle/build.py
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oracle.cpp")
HDR = os.path.join(HERE, "oracle.h")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile if the library is missing or older than its sources; return its path."""
    if not force and os.path.exists(LIB):
        t = os.path.getmtime(LIB)
        if t >= os.path.getmtime(SRC) and t >= os.path.getmtime(HDR):
            return LIB
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = ["g++", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c++17", "-Wall", "-o", tmp, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
