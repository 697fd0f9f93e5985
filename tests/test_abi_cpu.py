"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every
symbol include/mm.h declares, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def mm():
    from paper_1406_7635_b200 import build
    build.build()
    import paper_1406_7635_b200 as mm
    return mm


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mm_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(mm):
    lib = mm.lib()
    names = _declared_symbols()
    assert "mm_create" in names and "mm_step_rk45" in names and "mm_run" in names and "mm_b_eff" in names
    for name in names:
        assert hasattr(lib, name), name
    assert set(names) == set(mm.EXPORTS)


def test_version_and_error_strings(mm):
    lib = mm.lib()
    assert b"sm_100a" in lib.mm_version()
    for code in (0, -1, -2, -3, -4, -5, -6):
        assert len(lib.mm_strerror(code)) > 0
    assert lib.mm_strerror(-3) != lib.mm_strerror(-1)


def test_params_struct_layout_matches_the_header(mm):
    # int + 5*256 doubles + 256*3 + 3*256 + 2*256*3 + 3 doubles + pointer + double, 8-byte aligned
    n = 256
    expect = 8 + 8 * (5 * n + 3 * n + 3 * n + 2 * 3 * n + 3) + 8 + 8
    assert C.sizeof(mm.mm_params) == expect
    assert C.sizeof(mm.mm_step_info) == 4 * 8 + 8 + 8


def test_invalid_arguments_are_rejected_without_a_gpu(mm):
    lib = mm.lib()
    h = C.c_void_p()
    assert lib.mm_create(C.byref(h), 0, 4, 1, 1e-9, 1e-9, 1e-9, 0, 0, 0) == mm.MM_EINVAL
    assert lib.mm_create(C.byref(h), 4, 4, 1, -1e-9, 1e-9, 1e-9, 0, 0, 0) == mm.MM_EINVAL
    assert lib.mm_create(None, 4, 4, 1, 1e-9, 1e-9, 1e-9, 0, 0, 0) == mm.MM_EINVAL
    assert lib.mm_destroy(None) == mm.MM_OK
    assert lib.mm_steps(None, 1) == mm.MM_EINVAL


def test_no_cpu_fallback(mm):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p()
    assert mm.lib().mm_create(C.byref(h), 8, 8, 1, 1e-9, 1e-9, 1e-9, 0, 0, 0) == mm.MM_ECUDA
    with pytest.raises(RuntimeError):
        mm.Sim((8, 8, 1), (1e-9, 1e-9, 1e-9))


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1406_7635_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_1406_7635_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "(`paper_1406_7635_b200/`)", ""), f
