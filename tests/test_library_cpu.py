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
    assert 4 * 4 * S + S // 8 <= w < 4 * 4 * S + S // 8 + (1 << 21)      # phi x2, phidot x2, one sign bit per site + small scratch
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


def test_multiply_adds_are_fused_exactly_where_the_arithmetic_form_says():
    """Bit-for-bit parity with the oracle rests on the machine code doing the operations the form
    names.  ptxas contracts packed mul.rn.f32x2 + add.rn.f32x2 into FFMA2 whatever --fmad says
    (prs_pack.cuh works around it), so look at the SASS of EVERY step kernel in the library (generic,
    tiled, two-step, the multi-step tbs / tbr kernels that are the default path, cluster-resident): no
    FFMA / FFMA2 / DFMA in any step kernel of the COEF form (template argument ARITH = 1), and fused instructions present in every kernel of
    the FMA form (ARITH = 2).  LITERAL kernels legitimately contain FMAs inside the correctly rounded
    division routine."""
    import shutil
    import subprocess

    from paper_1710_10420_b200 import build as prs_build

    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    cufilt = shutil.which("cu++filt") or "/usr/local/cuda/bin/cu++filt"
    if not (os.path.exists(cuobjdump) and os.path.exists(cufilt)):
        pytest.skip("cuobjdump / cu++filt not available")
    sass = subprocess.run([cuobjdump, "-sass", prs_build.build()], stdout=subprocess.PIPE, text=True, check=True).stdout
    names = sorted(set(re.findall(r"Function : (\S+)", sass)))
    plain = subprocess.run([cufilt] + names, stdout=subprocess.PIPE, text=True, check=True).stdout.splitlines()
    arith_of, step_kernels = {}, 0
    for mangled, dem in zip(names, plain):
        if not re.search(r"prs::step\w*_kernel<", dem):
            continue
        step_kernels += 1
        # ARITH is the second template argument of every step kernel (single-step tiled, two-step tb2, multi-step
        # tbs / tbr, cluster-resident) and the third of step_generic_kernel<T, DIMS, ARITH>
        m = re.search(r"prs::step_generic_kernel<\w+, \(int\)\d+, \(int\)(\d)>", dem) or \
            re.search(r"prs::step(?:\dd_(?:tiled|tb2|tbs|tbr|cluster|band))_kernel<\w+, \(int\)(\d)[,>]", dem)
        assert m, "step kernel the test cannot classify: " + dem
        arith_of[mangled] = int(m.group(1))
    families = set(re.search(r"prs::(step\w*_kernel)<", d).group(1) for d in plain if re.search(r"prs::step\w*_kernel<", d))
    for fam in ("step_generic_kernel", "step3d_tiled_kernel", "step2d_tiled_kernel", "step3d_tb2_kernel", "step2d_tb2_kernel",
                "step3d_tbs_kernel", "step2d_tbs_kernel", "step3d_tbr_kernel", "step2d_cluster_kernel"):
        assert fam in families, fam
    assert len(arith_of) == step_kernels >= 120 and sorted(set(arith_of.values())) == [0, 1, 2]
    for a in (0, 1, 2):                                   # every family is built in every arithmetic form
        assert sum(1 for v in arith_of.values() if v == a) == step_kernels // 3
    # Fused instructions of the kernel's OWN step precision: FFMA / FFMA2 in a float kernel, DFMA in a double one.  (A
    # float kernel may hold DFMAs -- the cluster-resident kernel measures Eqs. 7-8 inside its launches, in double, and the
    # correctly rounded FP64 division expands into DFMAs -- but its step arithmetic could only ever fuse into FFMA / FFMA2,
    # which is where ptxas's packed contraction strikes.)
    is_double = {m: ("<double," in d) for m, d in zip(names, plain)}
    is_cluster = {m: ("step2d_cluster_kernel" in d) for m, d in zip(names, plain)}
    cur, fused = None, {k: 0 for k in arith_of}
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
        elif cur in fused and re.search(r"\bDFMA\b" if is_double[cur] else r"\bFFMA2?\b", line):
            # "FFMA Rd, RZ, Ra, Rb" multiplies by zero: the FP64 division's expansion uses it as an exponent-range probe on
            # the high word of its operands (it follows the division's DFMA pair); no product is fused there
            if not re.search(r"\bFFMA\s+R\d+, RZ,", line):
                fused[cur] += 1
    # COEF: nothing fused.  One exemption, stated: the DOUBLE cluster-resident kernels, whose in-launch FP64 division
    # cannot be told from step arithmetic in SASS; they are held by bit-identity with the single-step kernel and the
    # oracle in all three forms (test_cluster_resident_kernel_equals_single_steps_bitwise), and double arithmetic has no
    # packed form for ptxas to contract in the first place.
    exempt = [k for k in arith_of if is_cluster[k] and is_double[k]]
    assert len(exempt) == 15                                # 5 shapes (vectors per thread x CTAs per cluster) x 3 forms: no more
    assert [k for k, a in arith_of.items() if a == 1 and fused[k] and k not in exempt] == []
    assert [k for k, a in arith_of.items() if a == 2 and not fused[k]] == []
