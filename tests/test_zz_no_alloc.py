"""fs_kselect_noalloc (the entry point that allocates nothing: scratch in a built-in __device__ array)
against fs_kselect, the existing path, bit for bit -- the tolerance every k-selection test uses (one
correct answer) -- on calls in a row that share the array.  Collected last on purpose
(the file name): the run uses pytest -x.
"""
import numpy as np
import pytest
import torch

import datagen

pytestmark = pytest.mark.gpu


def both(fs, rows, k):
    n_rows = rows.shape[0]
    ev, ei = fs.kselect(rows, k)
    gv = torch.full((n_rows, k), float("nan"), dtype=torch.float32, device="cuda")
    gi = torch.full((n_rows, k), -7, dtype=torch.int32, device="cuda")
    fs.kselect_noalloc(rows, k, gv, gi)
    torch.cuda.synchronize()
    assert torch.equal(gi, ei), "indices differ (n_rows=%d, k=%d)" % (n_rows, k)
    assert torch.equal(gv.view(torch.int32), ev.view(torch.int32)), "value bits differ (n_rows=%d, k=%d)" % (n_rows, k)


def test_noalloc_matches_kselect_on_calls_in_a_row():
    import paper_1702_08734_b200 as fs
    assert fs.kselect_noalloc_max_scratch() == 4 << 20
    batch = torch.from_numpy(datagen.kselect_rows(0, 300, 16384)).cuda()       # CTA-per-row path: row counter
    ragged = torch.from_numpy(datagen.kselect_rows(7, 37, 2003, duplicates=False)).cuda()
    long_rows = torch.from_numpy(datagen.kselect_rows(11, 2, (1 << 20) + 5, duplicates=False)).cuda()  # A4: lists
    # twice over, so that every call also runs on what the other shapes left in the array
    for _ in range(2):
        for rows, ks in ((batch, (1, 32, 1024)), (long_rows, (1, 100, 1024)), (ragged, (2, 128)), (batch, (128,))):
            for k in ks:
                assert fs.kselect_ws_bytes(rows.shape[0], rows.shape[1], k) <= fs.kselect_noalloc_max_scratch()
                both(fs, rows, k)


def test_noalloc_same_call_twice_same_output():
    import paper_1702_08734_b200 as fs
    rows = torch.from_numpy(datagen.kselect_rows(3, 1, (1 << 21) + 3, duplicates=False)).cuda()
    out = []
    for _ in range(2):
        v = torch.empty((1, 1024), dtype=torch.float32, device="cuda")
        i = torch.empty((1, 1024), dtype=torch.int32, device="cuda")
        fs.kselect_noalloc(rows, 1024, v, i)
        out.append((v, i))
    torch.cuda.synchronize()
    assert torch.equal(out[0][1], out[1][1]) and torch.equal(out[0][0].view(torch.int32), out[1][0].view(torch.int32))
    ev, ei = fs.kselect(rows, 1024)
    assert torch.equal(out[1][1], ei) and torch.equal(out[1][0].view(torch.int32), ev.view(torch.int32))


def test_noalloc_allocates_nothing():
    import paper_1702_08734_b200 as fs
    rows = torch.from_numpy(datagen.kselect_rows(5, 2, 1 << 20, duplicates=False)).cuda()
    v = torch.empty((2, 64), dtype=torch.float32, device="cuda")
    i = torch.empty((2, 64), dtype=torch.int32, device="cuda")
    fs.kselect_noalloc(rows, 64, v, i)  # first use on this device: symbol address looked up
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        fs.kselect_noalloc(rows, 64, v, i)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "device memory in use changed across fs_kselect_noalloc calls"


def test_noalloc_rejects_calls_beyond_the_array():
    import paper_1702_08734_b200 as fs
    n_rows, n, k = 64, 1 << 22, 1024  # 64 long rows: survivor lists far beyond 4 MiB
    assert fs.kselect_ws_bytes(n_rows, n, k) > fs.kselect_noalloc_max_scratch()
    rows = torch.empty((n_rows, n), dtype=torch.float32, device="cuda")
    v = torch.empty((n_rows, k), dtype=torch.float32, device="cuda")
    i = torch.empty((n_rows, k), dtype=torch.int32, device="cuda")
    with pytest.raises(fs.FsError) as e:
        fs.kselect_noalloc(rows, k, v, i)
    assert "FS_NOALLOC_SCRATCH_BYTES" in str(e.value)
    # the array is still usable afterwards
    small = torch.from_numpy(datagen.kselect_rows(9, 80, 4099, duplicates=False)).cuda()
    both(fs, small, 32)
