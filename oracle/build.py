"""Builds oracle/libprs_ref.so from oracle/prs_ref.cpp with g++ (no CUDA, no torch).

Flags matter for parity: ``-ffp-contract=off`` forbids FMA contraction so every operation of
prs_ref.cpp is rounded on its own, exactly as written; never ``-ffast-math``.
Run ``python -m oracle.build`` or call :func:`build`.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "prs_ref.cpp")
HDR = os.path.join(HERE, "prs_ref.h")
LIB = os.path.join(HERE, "libprs_ref.so")

FLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
         "-Wall", "-Wextra"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in (SRC, HDR, os.path.abspath(__file__)))


def build(force: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = ["g++"] + FLAGS + ["-o", tmp, SRC]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
