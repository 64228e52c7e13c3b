"""The C-ABI library loads on a GPU-less box, exports every symbol include/fs.h
declares, and validates arguments before any launch (no compute calls here)."""
import ctypes

import pytest

import paper_1702_08734_b200 as fs
from paper_1702_08734_b200 import build as fs_build


@pytest.fixture(scope="module")
def L():
    fs_build.build()
    return fs.lib()


def test_exports_every_declared_symbol(L):
    names = fs.declared_symbols()
    assert len(names) >= 23 and "fs_kselect" in names and "fs_ivfpq_search" in names
    missing = [n for n in names if not hasattr(L, n)]
    assert not missing, missing


def test_version_names_the_architecture(L):
    assert b"sm_100a" in L.fs_version()


def test_argument_validation_needs_no_gpu(L):
    i64, ci, vp, sz = ctypes.c_int64, ctypes.c_int, ctypes.c_void_p, ctypes.c_size_t
    one = vp(16)  # a non-NULL pointer that is never dereferenced: validation fails first
    # k out of range / ld < n / NULL pointers
    assert L.fs_kselect(one, i64(1), i64(8), i64(8), ci(0), one, one, vp(0), sz(0), vp(0)) == 1
    assert L.fs_kselect(one, i64(1), i64(8), i64(8), ci(2000), one, one, vp(0), sz(0), vp(0)) == 2
    assert L.fs_kselect(one, i64(1), i64(8), i64(4), ci(2), one, one, vp(0), sz(0), vp(0)) == 1
    assert L.fs_kselect(vp(0), i64(1), i64(8), i64(8), ci(2), one, one, vp(0), sz(0), vp(0)) == 1
    assert b"fs_kselect" in L.fs_last_error()
    assert L.fs_flat_l2_knn(one, i64(1), one, i64(1), ci(0), ci(1), one, one, vp(0), sz(0), vp(0)) == 1
    assert L.fs_flat_l2_knn(one, i64(1), one, i64(1), ci(4), ci(5000), one, one, vp(0), sz(0), vp(0)) == 2
    assert L.fs_flat_l2_knn(one, i64(-1), one, i64(1), ci(4), ci(1), one, one, vp(0), sz(0), vp(0)) == 1
    # prepared database: NULL / misaligned / too small block, sizes
    L.fs_flat_prepare_bytes.restype = sz
    assert L.fs_flat_prepare_bytes(i64(-1), ci(4)) == 0 and L.fs_flat_prepare_bytes(i64(1000), ci(64)) >= 1000 * 4
    assert L.fs_flat_prepare(one, i64(10), ci(4), vp(0), sz(1 << 20), vp(0)) == 1
    assert L.fs_flat_prepare(one, i64(10), ci(4), vp(256 + 16), sz(1 << 20), vp(0)) == 1
    assert L.fs_flat_prepare(one, i64(10), ci(4), vp(256), sz(8), vp(0)) == 1
    assert L.fs_flat_l2_knn_prepared(one, i64(1), one, vp(0), sz(0), i64(1), ci(4), ci(1), one, one, vp(0), sz(0), vp(0)) == 1
    assert L.fs_flat_l2_knn_prepared(one, i64(1), one, vp(256), sz(8), i64(1), ci(4), ci(1), one, one, vp(0), sz(0), vp(0)) == 1
    h = vp()
    assert L.fs_ivfpq_create(ctypes.byref(h), ci(96), ci(16), ci(7)) == 1    # d % M != 0
    assert L.fs_ivfpq_create(ctypes.byref(h), ci(256), ci(16), ci(128)) == 2  # M > 64
    assert L.fs_ivfpq_create(None, ci(96), ci(16), ci(8)) == 1
    # zero-size calls return FS_OK without touching the device
    assert L.fs_kselect(vp(0), i64(0), i64(8), i64(8), ci(2), vp(0), vp(0), vp(0), sz(0), vp(0)) == 0
    assert L.fs_flat_l2_knn(vp(0), i64(0), one, i64(4), ci(4), ci(1), vp(0), vp(0), vp(0), sz(0), vp(0)) == 0


def test_workspace_sizes_are_pure_functions(L):
    assert fs.kselect_ws_bytes(10000, 16384, 32) == 256        # one pass: only the work counter
    assert fs.kselect_ws_bytes(1, 1 << 27, 1024) > 0           # split row: partial lists
    assert fs.flat_l2_knn_ws_bytes(64, 8192, 64, 10) >= (8192 + 64) * 4
