"""The C-ABI library loads and exports every symbol include/wilson_cg.h declares (-m "not gpu":
no compute call is made; on a box without a GPU wd_create must fail cleanly, not crash)."""
import ctypes
import os

import pytest

from paper_2111_14958_b200 import build as wbuild
from paper_2111_14958_b200 import wilson


@pytest.fixture(scope="module")
def lib():
    wbuild.build()
    return wilson.load_library()


def test_header_declares_the_north_star_calls():
    names = wilson.declared_symbols()
    for need in ("wd_create", "wd_destroy", "wd_apply", "cg_solve", "wd_pack_gauge", "wd_pack_spinor",
                 "wd_unpack_spinor", "wd_last_error", "wd_apply_host", "cg_solve_host", "wd_norm2"):
        assert need in names


def test_library_exports_every_declared_symbol(lib):
    missing = [n for n in wilson.declared_symbols() if not hasattr(lib, n)]
    assert not missing, f"declared in include/wilson_cg.h but not exported: {missing}"


def test_no_torch_types_in_signatures():
    text = open(wilson.HEADER_PATH).read()
    assert "torch" not in text.replace("torch.Tensor.data_ptr()", "") and "at::" not in text and "#include <torch" not in text


def test_version_and_tiles(lib):
    assert b"sm_100a" in lib.wd_version()
    shapes = wilson.tile_shapes()
    assert len(shapes) == lib.wd_num_tiles() >= 4
    for s in shapes:
        n = s[0] * s[1] * s[2] * s[3]
        assert n % 32 == 0 and 64 <= n <= 1024


def test_argument_errors_without_touching_a_gpu(lib):
    ctx = ctypes.c_void_p()
    bad = (ctypes.c_int * 4)(4, 4, 2, 4)
    assert lib.wd_create(ctypes.byref(ctx), bad, 32, -1, None) == -2  # WD_ERR_DIMS
    assert b"extent" in lib.wd_last_error(None)
    # 36 V must stay below 2^31 (32-bit plane indexing): 96^2 x 64 x 96 is the largest lattice of that shape family
    # (tests/test_gpu_parity.py::test_largest_supported_volume runs it), one more z-slab of 32 is refused
    big = (ctypes.c_int * 4)(96, 96, 96, 96)
    assert lib.wd_create(ctypes.byref(ctx), big, 32, -1, None) == -2
    assert b"too large" in lib.wd_last_error(None)
    ok = (ctypes.c_int * 4)(4, 4, 4, 4)
    assert lib.wd_create(ctypes.byref(ctx), ok, 16, -1, None) == -5   # WD_ERR_PRECISION
    assert lib.wd_create(ctypes.byref(ctx), ok, 32, 0, None) == -1    # WD_ERR_ARG
    assert lib.wd_create(None, ok, 32, -1, None) == -1
    assert lib.wd_destroy(None) == 0


def test_create_fails_loudly_without_a_device(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    ctx = ctypes.c_void_p()
    ok = (ctypes.c_int * 4)(4, 4, 4, 4)
    rc = lib.wd_create(ctypes.byref(ctx), ok, 32, -1, None)
    assert rc < 0 and not ctx.value
    assert len(lib.wd_last_error(None)) > 0
    with pytest.raises(RuntimeError):
        wilson.WilsonContext((4, 4, 4, 4))


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.dirname(wilson.__file__)
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "wilson_oracle" not in text and "from oracle" not in text and "import oracle" not in text, fn


def test_fastdiv_constants_of_the_tile_decode(lib):
    """host logic: (n*M) >> (32+sh) == n // d for every divisor the tile decode can meet and every n that can occur"""
    for d in list(range(1, 200)) + [255, 256, 257, 1000, 4095, 4096, 4097, 82944, 663552, 1 << 20, (1 << 24) - 1]:
        assert lib.wd_selftest_fastdiv(d, 300000) == 0, d
    for d in (3, 7, 24, 48, 96, 576, 13824):
        assert lib.wd_selftest_fastdiv(d, 1 << 24) == 0, d
    assert lib.wd_selftest_fastdiv(0, 10) == -1
