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
    out = [("prs_api", "prs_api.cu", []), ("prs_static", "prs_static.cu", [])]
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


# Build variants: "" = the product; "jitter" = the same sources with -DPRS_RACE_JITTER=1 (csrc/prs_arith.cuh: random
# warp-uniform delays around every barrier and publication), used by tests/sanitize_kernels.py to look for races.
VARIANTS = {"": [], "jitter": ["-DPRS_RACE_JITTER=1"]}


def lib_path(variant=""):
    return LIB if not variant else os.path.join(HERE, "libprs_%s.so" % variant)


def is_current(variant=""):
    lib, stamp = lib_path(variant), lib_path(variant) + ".srchash"
    if not (os.path.exists(lib) and os.path.exists(stamp)):
        return False
    with open(stamp) as fh:
        return fh.read().strip() == source_hash()


def _compile(job):
    (name, src, flags), objdir, extra = job
    obj = os.path.join(objdir, name + ".o")
    cmd = [_nvcc()] + NVCC_FLAGS + extra + flags + ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, cwd=HERE, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    return name, obj, cmd, res


def build(force=False, verbose=False, jobs=None, variant=""):
    """Compiles the translation units of csrc/ in parallel and links libprs.so (or libprs_<variant>.so); returns
    the library path.  Raises on compiler failure.  Safe under concurrent callers (the ranks of a torchrun job):
    the whole build runs under an exclusive lock on a file beside the library, into a per-process object
    directory, and whoever gets the lock second finds the library current."""
    import fcntl
    import shutil

    if variant not in VARIANTS:
        raise ValueError("unknown build variant %r" % variant)
    LIBV, STAMPV = lib_path(variant), lib_path(variant) + ".srchash"
    if not force and is_current(variant):
        return LIBV
    with open(LIBV + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and is_current(variant):               # another process built it while we waited
                return LIBV
            return _build_locked(verbose, jobs, variant, LIBV, STAMPV)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)


def _build_locked(verbose, jobs, variant, LIBV, STAMPV):
    import shutil

    objdir = os.path.join(OBJDIR, "%s.%d" % (variant or "product", os.getpid()))
    shutil.rmtree(objdir, ignore_errors=True)
    os.makedirs(objdir, exist_ok=True)
    jobs = jobs or int(os.environ.get("PRS_BUILD_JOBS", "0")) or min(len(units()), os.cpu_count() or 1)
    with ThreadPoolExecutor(max_workers=jobs) as pool:
        results = list(pool.map(_compile, [(u, objdir, VARIANTS[variant]) for u in units()]))
    log = os.path.join(HERE, "build%s.log" % ("_" + variant if variant else ""))
    with open(log, "w") as fh:
        for name, obj, cmd, res in results:
            fh.write("### %s\n%s\n%s\n" % (name, " ".join(cmd), res.stdout))
    if verbose:
        print(open(log).read())
    failed = [(name, res) for name, obj, cmd, res in results if res.returncode != 0]
    if failed:
        raise RuntimeError("nvcc failed on %s (see %s):\n%s" % (failed[0][0], log, failed[0][1].stdout[-4000:]))
    tmp = LIBV + ".tmp.%d" % os.getpid()
    cmd = [_nvcc(), "--shared", "-o", tmp] + [obj for name, obj, cmd, res in results]
    res = subprocess.run(cmd, cwd=HERE, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    with open(log, "a") as fh:
        fh.write("### link\n%s\n%s\n" % (" ".join(cmd), res.stdout))
    if res.returncode != 0:
        if os.path.exists(tmp):
            os.remove(tmp)
        raise RuntimeError("link failed (see %s):\n%s" % (log, res.stdout[-4000:]))
    os.replace(tmp, LIBV)
    with open(STAMPV, "w") as fh:
        fh.write(source_hash() + "\n")
    if not verbose:
        shutil.rmtree(objdir, ignore_errors=True)
    return LIBV


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv,
                variant="jitter" if "--jitter" in sys.argv else ""))
