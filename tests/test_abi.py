"""The C ABI without a GPU: libmvd.so loads, exports every symbol include/mvd.h declares, and its
host-side planner (FFT lengths, workspace sizes, argument validation) behaves as the header says.
No compute call is made here."""
import ctypes as C
import os
import re

import pytest

import paper_1308_0730_b200 as mvd
from paper_1308_0730_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    if not os.path.exists(mvd.LIB_PATH):
        from paper_1308_0730_b200 import build
        build.build(verbose=False)
    return mvd.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mvd.h")).read()
    return sorted(set(re.findall(r"MVD_API\s+[^;(]*?\b(mvd_[a-z_0-9]+)\s*\(", text)))


def test_header_and_binding_list_the_same_symbols():
    assert _declared_symbols() == sorted(mvd.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in _declared_symbols():
        assert hasattr(lib, name), name


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1308_0730_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "_work/" not in text, f


def test_options_init_defaults(lib):
    opt = B.mvd_options()
    lib.mvd_options_init(C.byref(opt))
    assert opt.struct_size == C.sizeof(B.mvd_options)
    assert opt.eps == pytest.approx(1e-6) and opt.psi_floor == pytest.approx(1e-6)
    assert opt.kernel_mode == 0 and opt.literal_product == 0 and not opt.workspace


# SURVEY 8(a) size table: N + r must fit per axis; x is carried as a half row
@pytest.mark.parametrize("dims,box", [
    ((64, 64, 64), (15, 15, 31)),
    ((128, 128, 128), (17, 17, 35)),
    ((256, 256, 128), (19, 19, 41)),
    ((512, 512, 256), (21, 21, 45)),
    ((1024, 1024, 512), (25, 25, 51)),
    ((24, 20, 18), (5, 7, 9)),
    ((33, 17, 9), (3, 5, 7)),
])
def test_plan_dims_cover_the_alias_free_sizes(lib, dims, box):
    mx, my, mz = mvd.plan_dims(dims, [box])
    hx = (dims[0] + 1) // 2
    rx, ry, rz = [(k - 1) // 2 for k in box]
    assert mx >= hx + 2 * rx and my >= dims[1] + ry and mz >= dims[2] + rz
    # 2-3-5-7-smooth, and not wasteful (next supported length is within ~12 %)
    for m, need in ((mx, hx + 2 * rx), (my, dims[1] + ry), (mz, dims[2] + rz)):
        n = m
        for p in (2, 3, 5, 7):
            while n % p == 0:
                n //= p
        assert n == 1
        assert m <= max(need * 1.15, need + 4)


def test_plan_dims_config4_are_the_documented_ones(lib):
    assert mvd.plan_dims((512, 512, 256), [(21, 21, 45)] * 7) == (280, 525, 280)


def test_forced_fft_dims(lib):
    assert mvd.plan_dims((64, 64, 64), [(15, 15, 31)], fft_dims=(48, 72, 80)) == (48, 72, 80)
    with pytest.raises(mvd.MvdError):
        mvd.plan_dims((64, 64, 64), [(15, 15, 31)], fft_dims=(40, 72, 80))   # too short: aliasing
    with pytest.raises(mvd.MvdError):
        mvd.plan_dims((64, 64, 64), [(15, 15, 31)], fft_dims=(48, 73, 80))   # not a supported length


def test_workspace_size_matches_the_layout(lib):
    dims, box, V = (64, 64, 64), (15, 15, 31), 4
    mx, my, mz = mvd.plan_dims(dims, [box] * V)
    n = mvd.workspace_size(dims, [box] * V, "osem")
    spectra = 2 * V * mx * my * mz * 8
    work = mx * my * dims[2] * 8
    assert n >= spectra + work + 2 * 4 * 64 ** 3
    assert n < 1.1 * (spectra + work) + (8 << 20)
    # combined variants carry a second work buffer (shared forward transform of psi)
    assert mvd.workspace_size(dims, [box] * V, "efficient") >= n + work


@pytest.mark.parametrize("dims,box", [
    ((64, 64, 64), (16, 15, 31)),      # even PSF size
    ((64, 64, 64), (15, 15, 8193)),    # absurd PSF size
    ((0, 64, 64), (3, 3, 3)),
])
def test_invalid_problems_are_rejected(lib, dims, box):
    assert mvd.workspace_size(dims, [box], "osem") == 0
    with pytest.raises(mvd.MvdError):
        mvd.plan_dims(dims, [box])


def test_create_rejects_bad_arguments_without_touching_the_gpu(lib):
    ctx = C.c_void_p(123)
    dims = B._Int3(8, 8, 8)
    pd = (C.c_int * 3)(3, 3, 3)
    opt = B.mvd_options()
    lib.mvd_options_init(C.byref(opt))
    one = (C.c_void_p * 1)(0)
    st = lib.mvd_create(C.byref(ctx), 1, one, dims, one, C.cast(pd, C.c_void_p), 2, C.byref(opt))
    assert st == 1 and not ctx.value                    # NULL view / PSF pointer -> INVALID_ARG
    import numpy as np
    psf = np.ones((3, 3, 3), np.float32)
    views = (C.c_void_p * 1)(4096)
    psfs = (C.c_void_p * 1)(psf.ctypes.data)
    st = lib.mvd_create(C.byref(ctx), 1, views, dims, psfs, C.cast(pd, C.c_void_p), 2, C.byref(opt))
    assert st == 3 and not ctx.value                    # no workspace -> MVD_ERR_WORKSPACE
    st = lib.mvd_create(C.byref(ctx), 1, views, dims, psfs, C.cast(pd, C.c_void_p), 7, C.byref(opt))
    assert st == 1
    assert lib.mvd_iterate(None, 1) == 1
    lib.mvd_destroy(None)
    assert lib.mvd_status_string(3).decode().startswith("workspace")
    assert lib.mvd_last_error(None) == b""


def test_blocked_workspace_size(lib):
    opt = B._make_options("auto", False, None, None, None, False)
    pd = (C.c_int * 6)(5, 5, 9, 5, 5, 9)
    n = lib.mvd_blocked_workspace_size(2, B._Int3(40, 36, 30), C.cast(pd, C.c_void_p), 2, C.byref(opt),
                                       B._Int3(20, 18, 16), None)
    whole = mvd.workspace_size((24, 22, 24), [(5, 5, 9)] * 2, "osem")
    assert n > whole > 0


def test_no_gpu_means_a_loud_failure(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import numpy as np
    with pytest.raises(mvd.MvdError):
        mvd.Deconvolver([torch.zeros(8, 8, 8)], [np.ones((3, 3, 3), np.float32)])


def test_planner_on_random_problems(lib):
    """Host planner, seeded sweep: for any volume and (odd) PSF boxes the FFT lengths are supported lengths (2-3-5-7-
    smooth, x even), alias-free (M >= N + r, x half row: M >= ceil(Nx/2) + 2 r_x, and M >= K), never wasteful beyond the
    spacing of the length table, and the workspace covers what the layout needs."""
    import numpy as np
    rng = np.random.default_rng(20130807)
    for _ in range(300):
        dims = tuple(int(rng.integers(1, 1100)) for _ in range(3))
        V = int(rng.integers(1, 5))
        boxes = [tuple(int(2 * rng.integers(0, 32) + 1) for _ in range(3)) for _ in range(V)]
        r = [max((b[a] - 1) // 2 for b in boxes) for a in range(3)]
        need = ((dims[0] + 1) // 2 + 2 * r[0], max(dims[1] + r[1], 2 * r[1] + 1), max(dims[2] + r[2], 2 * r[2] + 1))
        if max(need) > 1296:
            assert mvd.workspace_size(dims, boxes, "osem") == 0          # no length that long: refused, not mis-planned
            continue
        m = mvd.plan_dims(dims, boxes)
        assert m[0] % 2 == 0
        for a in range(3):
            assert m[a] >= need[a], (dims, boxes, m)
            n = m[a]
            for p in (2, 3, 5, 7):
                while n % p == 0:
                    n //= p
            assert n == 1
            assert m[a] <= max(need[a] * 1.16, need[a] + 8), (dims, boxes, m)
        ws = mvd.workspace_size(dims, boxes, "osem")
        nvox = dims[0] * dims[1] * dims[2]
        assert ws >= 2 * V * m[0] * m[1] * m[2] * 8 + m[0] * m[1] * dims[2] * 8 + 2 * 4 * nvox
        assert mvd.workspace_size(dims, boxes, "efficient") >= ws + m[0] * m[1] * dims[2] * 8
