"""CPU-side checks of the boundary: libens.so builds for sm_100a, loads without a GPU and exports exactly the
symbols include/ens.h declares; the binding refuses to run without the library (no CPU fallback)."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1208_1157_b200 import build
    return build.build()


def _declared():
    text = open(os.path.join(ROOT, "include", "ens.h")).read()
    return sorted(set(re.findall(r"ENS_API\s+[\w\s\*]*?\b(ens_\w+)\s*\(", text)))


def test_header_symbols_are_exported(libpath):
    names = _declared()
    assert len(names) >= 12
    lib = ctypes.CDLL(libpath)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in ens.h but not exported"
    out = subprocess.check_output(["nm", "-D", "--defined-only", libpath], text=True)
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l and l.split()[-1].startswith("ens_"))
    assert exported == names, "exported ens_* symbols differ from include/ens.h"


def test_binding_lists_the_same_symbols(libpath):
    from paper_1208_1157_b200 import ens
    assert sorted(ens.SYMBOLS) == _declared()
    assert ens.lib() is not None


def test_strerror_and_argument_checks_need_no_gpu(libpath):
    lib = ctypes.CDLL(libpath)
    lib.ens_strerror.restype = ctypes.c_char_p
    assert lib.ens_strerror(0) == b"ok"
    assert b"invalid" in lib.ens_strerror(-1)
    assert lib.ens_destroy(None) == 0
    h = ctypes.c_void_p()
    assert lib.ens_create(ctypes.c_int64(0), 3, ctypes.byref(h)) == -1   # EINVAL before any CUDA call
    assert lib.ens_create(ctypes.c_int64(8), 99, ctypes.byref(h)) == -1


def test_static_entry_point_checks_sizes_before_any_cuda_call(libpath):
    """ens_hermite_static: argument errors and the size limit of its static scratch are decided on the host, before the
    first CUDA call (so they are testable here); the limit is ENS_STATIC_MAX_GROUPS warp-groups of 32 / L systems."""
    lib = ctypes.CDLL(libpath)
    vp, i64, ci, cd = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
    lib.ens_hermite_static.argtypes = [vp, vp, vp, vp, vp, vp, i64, i64, ci, cd, cd, i64, cd, cd, vp]
    lib.ens_strerror.restype = ctypes.c_char_p
    text = open(os.path.join(ROOT, "include", "ens.h")).read()
    max_groups = int(re.search(r"#define\s+ENS_STATIC_MAX_GROUPS\s+(\d+)", text).group(1))
    from paper_1208_1157_b200 import ens
    assert max_groups == ens.STATIC_MAX_GROUPS and ens.ETOOLARGE == -6
    buf = (ctypes.c_double * 8)()
    p = ctypes.addressof(buf)  # never dereferenced: every call below returns before touching memory

    def call(n_sys, n_pad, n_body, dt=0.01, t_end=float("inf"), steps=10, first=p):
        return lib.ens_hermite_static(first, p, p, p, p, p, n_sys, n_pad, n_body, dt, t_end, steps, 0.0, float("inf"), None)

    assert call(8, 8, 3, first=None) == -1
    assert call(0, 8, 3) == -1 and call(9, 8, 3) == -1 and call(8, 8, 1) == -1 and call(8, 8, 17) == -1
    assert call(8, 8, 3, dt=0.0) == -1 and call(8, 8, 3, dt=float("nan")) == -1 and call(8, 8, 3, t_end=float("nan")) == -1
    assert call(8, 8, 3, steps=-1) == -1
    # lanes per system: 1 up to 8 bodies, 3 for 9, 11, 12, 5 for 10 and 13..16 -> systems per warp-group 32, 10, 6
    for n_body, per_group in ((2, 32), (8, 32), (9, 10), (10, 6), (11, 10), (12, 10), (13, 6), (16, 6)):
        n = max_groups * per_group + 1
        assert call(n, n, n_body) == -6, n_body
    assert b"static scratch" in lib.ens_strerror(-6)


def test_no_cpu_fallback_without_device(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1208_1157_b200 import ens
    with pytest.raises(ens.EnsError) as ei:
        ens.Ensemble(16, 3)
    assert ei.value.code == ens.ECUDA


def test_sass_is_sm100a_fp64(libpath):
    """The hot kernel is compiled for sm_100a and its inner loop is FP64 (DFMA) with the MUFU.RSQ seed."""
    r = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True)
    if r.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in r.stdout
    sass = subprocess.check_output(["cuobjdump", "-sass", "-fun", "hermite_kernel", libpath], text=True, errors="ignore") \
        if False else subprocess.run(["cuobjdump", "-sass", libpath], capture_output=True, text=True).stdout
    assert "DFMA" in sass and "MUFU.RSQ" in sass


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1208_1157_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dp, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "ens_oracle" not in text, f
