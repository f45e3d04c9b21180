"""Host-side checks of libprs that need no GPU: the library builds, loads and exports every symbol
declared in include/prs.h; argument validation that happens before any CUDA call."""
import ctypes as C
import os
import re

import pytest

import paper_1710_10420_b200 as prs
from paper_1710_10420_b200 import prs as binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "prs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(prs_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    L = prs.lib()
    names = declared_symbols()
    assert len(names) >= 13
    for name in names:
        assert hasattr(L, name), name
    assert sorted(binding.EXPORTS) == names


def test_workspace_bytes():
    S = 1024 ** 3
    w = prs.prs_workspace_bytes(3, 1024, prs.F32)
    assert 4 * 4 * S <= w < 4 * 4 * S + (1 << 21)          # phi x2, phidot x2 + small scratch
    assert prs.prs_workspace_bytes(3, 1024, prs.F64) >= 4 * 8 * S
    assert prs.prs_workspace_bytes(2, 16384, prs.F32) >= 4 * 4 * 16384 ** 2
    for bad in [(1, 8, 0), (4, 8, 0), (2, 0, 0), (2, -3, 0), (2, 8, 2), (3, 100000, 0)]:
        assert prs.prs_workspace_bytes(*bad) == 0


def test_create_rejects_bad_arguments_before_touching_cuda():
    L = prs.lib()
    h = C.c_void_p()
    # invalid dims / N / precision / parameters -> INVALID_ARG; null or misaligned workspace -> WORKSPACE
    assert L.prs_create(C.byref(h), 5, 8, 0, 3.0, 1.0, 0.1, 10.0, 1.0, 1, None, 0, None) == 1
    assert L.prs_create(C.byref(h), 2, 8, 0, 3.0, 1.0, -0.1, 10.0, 1.0, 1, None, 0, None) == 1
    assert L.prs_create(C.byref(h), 2, 8, 0, 3.0, 1.0, 0.1, 0.0, 1.0, 1, None, 0, None) == 1
    assert L.prs_create(C.byref(h), 2, 8, 0, -1.0, 1.0, 0.1, 10.0, 1.0, 1, None, 0, None) == 1
    assert L.prs_create(C.byref(h), 2, 8, 0, 3.0, 1.0, 0.1, 10.0, float("nan"), 1, None, 0, None) == 1
    assert L.prs_create(None, 2, 8, 0, 3.0, 1.0, 0.1, 10.0, 1.0, 1, None, 0, None) == 1
    assert L.prs_create(C.byref(h), 2, 8, 0, 3.0, 1.0, 0.1, 10.0, 1.0, 1, None, 0, None) == 3
    assert L.prs_create(C.byref(h), 2, 8, 0, 3.0, 1.0, 0.1, 10.0, 1.0, 1, 256, 16, None) == 3
    assert not h.value
    # null handles
    assert L.prs_step(None, 1) == 1 and L.prs_init(None, 1.0) == 1 and L.prs_destroy(None) == 1
    assert L.prs_last_error(None) == b"null handle"


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        prs.Simulation(2, 16)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1710_10420_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "prs_ref" not in text, f
                for ln in text.splitlines():
                    if "import" in ln or "#include" in ln or "dlopen" in ln or "CDLL" in ln:
                        assert "oracle" not in ln.lower(), (f, ln)


def test_no_fused_multiply_add_in_the_step_kernels():
    """Bit-for-bit parity with the oracle rests on every multiply and add being rounded on its own.
    ptxas contracts packed mul.rn.f32x2 + add.rn.f32x2 into FFMA2 whatever --fmad says (prs_pack.cuh
    works around it), so look at the machine code: no FFMA / FFMA2 / DFMA in any step kernel of the
    default (COEF, template argument LITERAL = false) arithmetic.  The LITERAL kernels legitimately
    contain FMAs inside the correctly rounded division routine."""
    import re
    import shutil
    import subprocess

    from paper_1710_10420_b200 import build as prs_build

    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", prs_build.build()], stdout=subprocess.PIPE, text=True, check=True).stdout
    cur, seen, bad = None, set(), []
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            continue
        if cur and "step" in cur and "Lb0E" in cur:
            seen.add(cur)
            if re.search(r"\b(FFMA2?|DFMA)\b", line):
                bad.append((cur, line.strip()))
    assert len(seen) >= 12, "expected the generic, tiled and two-step kernels in the library"
    assert not bad, bad[:5]
