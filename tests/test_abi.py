"""CPU-only checks of the C-ABI boundary: libmr.so builds, loads without a GPU, exports every symbol that
include/mr.h declares, validates arguments before touching CUDA and fails loudly (never falls back) without a GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def mr():
    from paper_1405_0942_b200 import build
    build.build()
    from paper_1405_0942_b200 import mr as m
    return m


def declared_functions():
    src = open(os.path.join(ROOT, "include", "mr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mr_[A-Za-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for must in ("mr_create", "mr_set_B0", "mr_step", "mr_diagnostics", "mr_get_fields", "mr_destroy", "mr_set_x",
                 "mr_workspace_bytes", "mr_last_error"):
        assert must in names


def test_library_exports_every_declared_symbol(mr):
    for name in declared_functions():
        assert hasattr(mr.lib, name), "libmr.so does not export %s" % name


def test_workspace_bytes_is_pure_host_arithmetic(mr):
    assert mr.workspace_bytes((4, 16, 16)) == 0          # below the minimum of 5
    assert mr.workspace_bytes((16, 16, 5000)) == 0       # above the maximum
    n = (256, 256, 512)
    b64, b32 = mr.workspace_bytes(n, "f64"), mr.workspace_bytes(n, "f32")
    field = 3 * 256 * 256 * 512 * 8
    assert 4 * field <= b64 < 4 * field + (1 << 20)
    assert 2 * field <= b32 < 2 * field + (1 << 20)
    # odd sizes are padded to 16-element rows
    assert mr.workspace_bytes((17, 9, 7)) >= (3 * 3 * 32 * 9 * 7 + 3 * 17 * 9 * 7) * 8
    # a periodic axis adds its ghost layers (two planes / rows, 16 bytes of columns either side) to the three padded fields
    assert mr.workspace_bytes(n, "f64", ("line_tied",) * 3) == b64 == mr.lib.mr_workspace_bytes(C.byref(mr.mr_grid(*n)), mr.MR_F64)
    bz = mr.workspace_bytes(n, "f64", ("line_tied", "line_tied", "periodic"))
    assert bz - b64 == 3 * (3 * 256 * 256 * 4 * 8)
    ball = mr.workspace_bytes(n, "f64", ("periodic",) * 3)
    assert ball - b64 == 3 * 3 * 8 * (272 * 260 * 516 - 256 * 256 * 512)
    bad = (C.c_int32 * 3)(0, 7, 0)
    assert mr.lib.mr_workspace_bytes_bc(C.byref(mr.mr_grid(*n)), mr.MR_F64, bad) == 0
    assert mr.lib.mr_adaptive_workspace_bytes_bc(C.byref(mr.mr_grid(*n)), mr.MR_F64, bad) == 0


def _create(mr, n=(16, 16, 32), lo=(-4, -4, -8), hi=(4, 4, 8), bc=(0, 0, 0), gamma=1.0, dtype=0, ws=256, ws_bytes=1 << 40):
    g = mr.mr_grid(*n)
    d = mr.mr_domain((C.c_double * 3)(*lo), (C.c_double * 3)(*hi))
    b = mr.mr_boundary((C.c_int * 3)(*bc), gamma, dtype, ws, ws_bytes, None)
    ctx = C.c_void_p()
    st = mr.lib.mr_create(C.byref(g), C.byref(d), C.byref(b), C.byref(ctx))
    return st, ctx, (mr.lib.mr_last_error(None) or b"").decode()


def test_create_validates_before_any_cuda_call(mr):
    assert _create(mr, n=(4, 16, 16))[0] == mr.MR_ERR_INVALID_ARG
    assert _create(mr, hi=(4, -4, 8))[0] == mr.MR_ERR_INVALID_ARG
    assert _create(mr, gamma=0.0)[0] == mr.MR_ERR_INVALID_ARG
    assert _create(mr, dtype=7)[0] == mr.MR_ERR_INVALID_ARG
    st, ctx, msg = _create(mr, bc=(0, 0, 2))
    assert st == mr.MR_ERR_INVALID_ARG and "boundary" in msg and not ctx.value
    assert _create(mr, ws=None)[0] == mr.MR_ERR_WORKSPACE
    assert _create(mr, ws=264)[0] == mr.MR_ERR_WORKSPACE            # misaligned
    assert _create(mr, ws_bytes=1024)[0] == mr.MR_ERR_WORKSPACE     # too small


def test_adaptive_workspace_bytes_is_pure_host_arithmetic(mr):
    g = mr.mr_grid(256, 256, 512)
    field = 3 * 256 * 256 * 512 * 8
    nb = mr.lib.mr_adaptive_workspace_bytes(C.byref(g), mr.MR_F64)
    assert 7 * field <= nb < 7 * field + (1 << 20)           # six stage velocities and the stage state
    bad = mr.mr_grid(4, 16, 16)
    assert mr.lib.mr_adaptive_workspace_bytes(C.byref(bad), mr.MR_F64) == 0


def test_binding_rejects_unknown_boundary_names(mr):
    with pytest.raises(mr.MrError):
        mr.Relaxation((16, 16, 32), (-4, -4, -8), (4, 4, 8), bc=("line_tied", "open", "line_tied"), device="cuda")


def test_null_context_calls_return_invalid_arg(mr):
    assert mr.lib.mr_step_adaptive(None, 1.0, 1e-6, None, 0, 10, None, None, 0) == mr.MR_ERR_INVALID_ARG
    assert mr.lib.mr_rhs(None, 0, None) == mr.MR_ERR_INVALID_ARG
    assert mr.lib.mr_convexity(None, None, None) == mr.MR_ERR_INVALID_ARG
    assert mr.lib.mr_step(None, 1, 0.1, 0) == mr.MR_ERR_INVALID_ARG
    assert mr.lib.mr_set_B0(None, None) == mr.MR_ERR_INVALID_ARG
    assert mr.lib.mr_diagnostics(None, 0, None) == mr.MR_ERR_INVALID_ARG
    assert mr.lib.mr_destroy(None) == mr.MR_OK


def test_no_gpu_means_a_loud_failure_not_a_fallback(mr):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    st, ctx, msg = _create(mr)     # valid arguments, fake workspace pointer: must stop at the first CUDA call
    assert st == mr.MR_ERR_CUDA and not ctx.value and msg
    with pytest.raises(Exception):
        mr.Relaxation((16, 16, 32), (-4, -4, -8), (4, 4, 8))


def test_product_path_does_not_touch_the_oracle():
    """Neither the package nor the C-ABI sources may import, load or call anything under oracle/, and the oracle
    includes nothing of the CUDA path (the two share no code)."""
    pkg = os.path.join(ROOT, "paper_1405_0942_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert "libmro" not in src and "mro_" not in src and "mro." not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "mro.c")).read()
    assert not re.search(r"#include\s+[<\"][^>\"]*(mr\.h|\.cuh)", osrc)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_1405_0942_b200" not in open(os.path.join(ROOT, "oracle", f)).read(), f
