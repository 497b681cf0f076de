"""CPU-side checks of the C-ABI boundary: the library builds, loads, and exports every symbol that
include/sim3ba.h declares; argument validation that needs no device; loud failure without a GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2605_30488_b200 import build, load_library
    build.build()
    return load_library()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "sim3ba.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sim3ba_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2605_30488_b200 import EXPORTS
    decl = declared_symbols()
    assert len(decl) >= 20
    for name in decl:
        assert hasattr(lib, name), name
    assert sorted(EXPORTS) == decl


def test_default_params_are_the_papers(lib):
    from paper_2605_30488_b200 import Params
    p = Params()
    assert lib.sim3ba_default_params(C.byref(p)) == 0
    assert abs(p.sigma_ray - 0.003) < 1e-9 and p.sigma_dist == 10.0 and abs(p.huber_k - 1.345) < 1e-6
    assert p.conf_min == 0.0 and p.lm_lambda == 0.0 and p.eps0 == 1e-6 and p.max_attempts == 6
    assert lib.sim3ba_default_params(None) == -1
    assert b"sm_100a" in lib.sim3ba_version()


def test_null_context_is_rejected(lib):
    for fn in ("sim3ba_build_system", "sim3ba_solve", "sim3ba_step", "sim3ba_retract", "sim3ba_destroy"):
        assert getattr(lib, fn)(None) == -1


def test_create_validates_before_touching_the_device(lib):
    from paper_2605_30488_b200 import make_params
    out = C.c_void_p()
    prm = make_params()
    one = C.c_void_p(16)
    fixed = (C.c_int32 * 1)(0)
    # non-positive dimensions / NULL pointers / invalid params -> INVALID_ARG (-1), no device needed
    assert lib.sim3ba_create(C.byref(out), 0, 4, 4, 1, one, one, one, one, fixed, 1, C.byref(prm), None) == -1
    assert lib.sim3ba_create(C.byref(out), 2, 4, 4, 1, None, one, one, one, fixed, 1, C.byref(prm), None) == -1
    bad = make_params(huber_k=-1.0)
    assert lib.sim3ba_create(C.byref(out), 2, 4, 4, 1, one, one, one, one, fixed, 1, C.byref(bad), None) == -1
    assert b"param" in lib.sim3ba_last_error(None)
    # maximum sizes: more than 2^28 pixels per keyframe (the per-slice index sums are 32-bit), more than 2^20 unknowns
    assert lib.sim3ba_create(C.byref(out), 2, 1 << 15, (1 << 13) + 1, 1, one, one, one, one, fixed, 1, C.byref(prm), None) == -1
    assert lib.sim3ba_create(C.byref(out), (1 << 20) // 7 + 1, 4, 4, 1, one, one, one, one, fixed, 1, C.byref(prm), None) == -1
    assert b"oversized" in lib.sim3ba_last_error(None)
    # the host jobs check their arguments the same way
    assert lib.sim3ba_optimize_host(2, 4, 4, 1, None, one, one, one, fixed, 1, C.byref(prm), one, 1, one, None, None) == -1
    assert lib.sim3ba_probe_fp64(None, None, None) == -1


def test_product_path_fails_loudly_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2605_30488_b200 import make_params
    out = C.c_void_p()
    prm = make_params()
    one = C.c_void_p(16)
    fixed = (C.c_int32 * 1)(0)
    rc = lib.sim3ba_create(C.byref(out), 2, 4, 4, 1, one, one, one, one, fixed, 1, C.byref(prm), None)
    assert rc == -2 and b"no CPU fallback" in lib.sim3ba_last_error(None)


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2605_30488_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "oracle/" not in txt.replace("oracle/:", ""), f
