"""Builds paper_1710_10420_b200/libprs.so (the C-ABI library of include/prs.h) with nvcc for sm_100a.

In-tree build: the .so sits beside this file so that it travels to the GPU box with the repository
snapshot.  The translation units (objects under _build/) are compiled in parallel, one nvcc process each.  A hash of the sources is kept beside it; :func:`build` recompiles only when they changed.
"""
import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libprs.so")
STAMP = LIB + ".srchash"

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-fmad=false",                      # belt and braces: the kernels already use *_rn intrinsics only
    "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall",
    "-Xptxas", "-v",
]
OBJDIR = os.path.join(HERE, "_build")


def units():
    """(object name, source file, extra flags): prs_api.cu plus prs_instances.cu once per kernel family,
    precision and arithmetic form (csrc/prs_instances.cu says which is which)."""
    out = [("prs_api", "prs_api.cu", [])]
    for unit, family in ((3, "tbs2d"), (2, "tbs3d"), (1, "tb2")):       # longest first
        for T in ("float", "double"):
            for arith in (0, 1, 2):
                out.append(("%s_%s_%d" % (family, T, arith), "prs_instances.cu",
                            ["-DPRS_UNIT=%d" % unit, "-DPRS_T=%s" % T, "-DPRS_ARITH=%d" % arith]))
    return out


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def sources():
    files = [os.path.join(ROOT, "include", "prs.h"), os.path.abspath(__file__)]
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh", ".h")):
            files.append(os.path.join(CSRC, name))
    return files


def source_hash():
    h = hashlib.sha256()
    for path in sources():
        h.update(os.path.basename(path).encode())
        with open(path, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def is_current():
    if not (os.path.exists(LIB) and os.path.exists(STAMP)):
        return False
    with open(STAMP) as fh:
        return fh.read().strip() == source_hash()


def _compile(unit):
    name, src, flags = unit
    obj = os.path.join(OBJDIR, name + ".o")
    cmd = [_nvcc()] + NVCC_FLAGS + flags + ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, cwd=HERE, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    return name, obj, cmd, res


def build(force=False, verbose=False, jobs=None):
    """Compiles the translation units of csrc/ in parallel and links libprs.so; returns the library
    path.  Raises on compiler failure."""
    if not force and is_current():
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    jobs = jobs or int(os.environ.get("PRS_BUILD_JOBS", "0")) or min(len(units()), os.cpu_count() or 1)
    with ThreadPoolExecutor(max_workers=jobs) as pool:
        results = list(pool.map(_compile, units()))
    log = os.path.join(HERE, "build.log")
    with open(log, "w") as fh:
        for name, obj, cmd, res in results:
            fh.write("### %s\n%s\n%s\n" % (name, " ".join(cmd), res.stdout))
    if verbose:
        print(open(log).read())
    failed = [(name, res) for name, obj, cmd, res in results if res.returncode != 0]
    if failed:
        raise RuntimeError("nvcc failed on %s (see %s):\n%s" % (failed[0][0], log, failed[0][1].stdout[-4000:]))
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc(), "--shared", "-o", tmp] + [obj for name, obj, cmd, res in results]
    res = subprocess.run(cmd, cwd=HERE, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    with open(log, "a") as fh:
        fh.write("### link\n%s\n%s\n" % (" ".join(cmd), res.stdout))
    if res.returncode != 0:
        if os.path.exists(tmp):
            os.remove(tmp)
        raise RuntimeError("link failed (see %s):\n%s" % (log, res.stdout[-4000:]))
    os.replace(tmp, LIB)
    with open(STAMP, "w") as fh:
        fh.write(source_hash() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
