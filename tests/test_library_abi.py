"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol
include/se_mobility.h declares, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os
import subprocess

import numpy as np
import pytest

import paper_1506_08481_b200 as pk
from paper_1506_08481_b200 import build as pkbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_every_declared_symbol():
    path = pkbuild.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    names = pk.declared_symbols()
    assert "se_plan_create" in names and "far_mobility_apply" in names and "se_plan_destroy" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/se_mobility.h but not exported"


def test_header_is_plain_c():
    """The boundary is a C ABI: the header must compile as C with no CUDA or torch types."""
    src = '#include "se_mobility.h"\nint main(void){ se_plan *p = 0; (void)p; return SE_NUM_STAGES == 8 ? 0 : 1; }\n'
    out = os.path.join(ROOT, "_hdr_check.o")
    try:
        subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-x", "c", "-c", "-", "-o", out],
                       input=src.encode(), check=True)
    finally:
        if os.path.exists(out):
            os.remove(out)


def test_version_and_sass_target():
    assert "sm_100a" in pk.version()
    dump = subprocess.run(["cuobjdump", "--list-elf", pkbuild.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in dump


def test_invalid_arguments_return_status_codes_without_a_gpu():
    lib = pk.load_library()
    h = ctypes.c_void_p()
    rad = np.ones(8)
    bad = [
        dict(N=0), dict(L=0.0), dict(L=-1.0), dict(xi=0.0), dict(rc=0.0), dict(rc=6.0),  # rc > L/2
        dict(M=15), dict(M=6, P=8), dict(P=1), dict(eta0=0.0),
    ]
    base = dict(N=8, L=10.0, xi=0.5, rc=3.0, M=16, P=8, eta0=1.0)
    for b in bad:
        a = dict(base, **b)
        st = lib.se_plan_create(ctypes.byref(h), a["N"], a["L"], rad.ctypes.data, a["xi"], a["rc"], a["M"], a["P"], a["eta0"])
        assert st == 1, (b, st)
        assert not h
    assert lib.se_plan_create(ctypes.byref(h), 8, 10.0, None, 0.5, 3.0, 16, 8, 1.0) == 1
    assert lib.se_plan_create(None, 8, 10.0, rad.ctypes.data, 0.5, 3.0, 16, 8, 1.0) == 1
    assert lib.se_plan_create(ctypes.byref(h), 8, 10.0, rad.ctypes.data, 0.5, 3.0, 64, 26, 1.0) == 2   # P > 24 unsupported
    rad_bad = rad.copy(); rad_bad[3] = -1.0
    assert lib.se_plan_create(ctypes.byref(h), 8, 10.0, rad_bad.ctypes.data, 0.5, 3.0, 16, 8, 1.0) == 1
    assert lib.se_plan_destroy(None) == 0
    assert lib.far_mobility_apply(None, None, None, None, None, None, None, None, None) == 1


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(pk.SeError) as ei:
        pk.SePlan(8, 10.0, np.ones(8), 0.5, 3.0, 16, 8)
    assert "SE_ERR_CUDA" in str(ei.value) or "SE_ERR_ALLOC" in str(ei.value)


def test_product_path_does_not_touch_the_oracle():
    """Neither side imports the other; only workloads/ is shared."""
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1506_08481_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "se_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1506_08481_b200" not in text and "from paper_1506_08481_b200" not in text
            assert "se_mobility.h" not in text and "csrc" not in text
