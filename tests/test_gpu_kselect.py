"""GPU parity: fs_kselect (through the C ABI) vs the oracle, bit-exact in values
and indices (BASELINE.json: "ties broken by lower index")."""
import numpy as np
import pytest
import torch

import datagen
import oracle

pytestmark = pytest.mark.gpu

K_ALL = [1, 2, 31, 32, 33, 64, 100, 128, 200, 256, 500, 512, 1000, 1024]


def run(rows_np, k, n=None):
    import paper_1702_08734_b200 as fs
    rows = torch.from_numpy(rows_np).cuda()
    val, idx = fs.kselect(rows, k, n=n)
    torch.cuda.synchronize()
    return val.cpu().numpy(), idx.cpu().numpy()


def assert_exact(rows_np, k, n=None):
    ev, ei = oracle.kselect(rows_np, k, n=n)
    gv, gi = run(rows_np, k, n=n)
    bad = np.nonzero((gi != ei).any(1) | (gv.view(np.uint32) != ev.view(np.uint32)).any(1))[0]
    assert bad.size == 0, "rows %s differ (k=%d); first: got %s want %s" % (
        bad[:5], k, gi[bad[0]][:8], ei[bad[0]][:8])


@pytest.mark.parametrize("k", K_ALL)
def test_random_rows_ragged(k):
    # several 128-element groups, the 4x unrolled body, a vector tail and a scalar tail
    rows = datagen.kselect_rows(0, 37, 2000 + 3, duplicates=False)
    assert_exact(rows, k)


@pytest.mark.parametrize("k", [1, 32, 128, 1024])
def test_cfg2_shaped_rows_with_duplicates(k):
    """cfg2 shape (rows of 16 384) on the rows that carry duplicated runs plus plain ones."""
    dup, _ = datagen.kselect_dup_rows(0, 10000)
    sel = list(np.nonzero(dup)[0][:6]) + [0, 1, 2]
    rows = np.concatenate([datagen.kselect_rows(int(r), 1, 16384) for r in sel])
    assert_exact(rows, k)


@pytest.mark.parametrize("n", [0, 1, 3, 4, 5, 31, 32, 33, 127, 128, 129, 511, 513])
def test_small_n_and_padding(n):
    rng = np.random.default_rng(n)
    rows = rng.integers(0, 5, size=(9, max(n, 1))).astype(np.float32)[:, :max(n, 1)]
    for k in (1, 4, 32, 40, 300):
        assert_exact(rows, k, n=n)


def test_structured_rows():
    n = 5000
    asc = np.arange(n, dtype=np.float32)
    rows = np.stack([asc, asc[::-1].copy(), np.full(n, 2.5, np.float32),
                     (np.arange(n) % 7).astype(np.float32), -asc])
    for k in (1, 10, 128, 1024):
        assert_exact(rows, k)


def test_special_values():
    rng = np.random.default_rng(0)
    rows = rng.standard_normal((6, 700)).astype(np.float32)
    rows[0, ::3] = 0.0
    rows[0, 1::3] = -0.0
    rows[1, ::5] = np.inf
    rows[2, ::4] = -np.inf
    rows[3, :] = np.inf
    rows[4, 10:20] = np.nan
    rows[5, :] = np.nan
    for k in (1, 5, 64, 700, 1024):
        assert_exact(rows, k)


def test_row_stride_and_misaligned_base():
    """ld > n and rows that do not start on a 16-byte boundary."""
    import paper_1702_08734_b200 as fs
    rng = np.random.default_rng(1)
    big = rng.random((11, 1003), dtype=np.float32)
    t = torch.from_numpy(big).cuda()
    for off, n in [(1, 1000), (2, 997), (3, 900)]:
        view = t[:, off:off + n]
        for k in (1, 50, 600):
            gv, gi = fs.kselect(view, k)
            ev, ei = oracle.kselect(np.ascontiguousarray(big[:, off:off + n]), k)
            assert np.array_equal(gi.cpu().numpy(), ei)
            assert np.array_equal(gv.cpu().numpy().view(np.uint32), ev.view(np.uint32))


@pytest.mark.parametrize("k", [1, 100, 1024])
def test_long_row_is_split(k):
    """A4: a few long rows go through the chunked passes (P > 1)."""
    rows = datagen.kselect_rows(50000, 3, 300_001, duplicates=False)
    rows[1, ::2] = np.floor(rows[1, ::2] * 16) / 16  # ties across chunks
    assert_exact(rows, k)


@pytest.mark.parametrize("k", [2, 100, 1024])
def test_long_rows_monotone_constant_and_ties(k):
    """A4 on rows a first-elements sample would misjudge: ascending, descending, constant, few distinct
    values.  The long-row bound comes from a strided sample; results stay bit-exact either way."""
    n = 1 << 20
    asc = np.arange(n, dtype=np.float32)
    rows = np.stack([asc, asc[::-1].copy(), np.full(n, 1.5, np.float32), (np.arange(n) % 5).astype(np.float32)])
    assert_exact(rows, k)


@pytest.mark.parametrize("k", [2, 32, 300, 1024])
def test_batch_rows_that_mislead_the_sample(k):
    """Rows of cfg2's length whose first 2 048 elements do not represent them (sorted both ways, runs,
    a few distinct values, a block of small values at the end): the sampled bound lets too few or too
    many through and the kernel must take its second filter pass or the exact slow path."""
    n = 16384
    rng = np.random.default_rng(k)
    asc = np.sort(rng.random(n, dtype=np.float32))
    late = rng.random(n, dtype=np.float32) + 1.0
    late[-3000:] -= 1.0
    runs = np.repeat(rng.random(n // 64, dtype=np.float32), 64)
    few = rng.integers(0, 3, n).astype(np.float32)
    rows = np.stack([asc, asc[::-1].copy(), late, late[::-1].copy(), runs, few, np.zeros(n, np.float32)])
    rows = np.concatenate([rows, datagen.kselect_rows(0, 500, n, duplicates=False)[:, :n]])  # enough rows to fill the GPU
    assert_exact(rows, k)


@pytest.mark.parametrize("n", [8191, 8192, 8193, 8199, 12288 + 5, 16384 + 1, 20000])
def test_stage_boundaries_of_the_k1024_class(n):
    """k > 256: rows of >= 8 192 elements keep the counting arrays in the row's last two ring stages (16 KB
    each), shorter rows in arrays of their own.  Lengths around the switch and around stage ends, a row
    start that is not 16-byte aligned, more rows than resident CTAs (the ring wraps, stages are held and
    handed back many times), rows that take the second look / the slow path with the aliased arrays."""
    import paper_1702_08734_b200 as fs
    rng = np.random.default_rng(n)
    nr = 1500
    big = rng.random((nr, n + 3), dtype=np.float32)
    big[3, :] = np.sort(big[3, :])                      # ascending: the head misleads the sample
    big[4, :] = np.sort(big[4, :])[::-1]                # descending
    big[5, :] = 0.25                                    # constant: everything ties
    big[6, :] = np.floor(big[6, :] * 4)                 # four distinct values
    big[7, :n // 2] += 2.0                              # the small values come late
    big[8, ::3] = 0.0                                   # +-0, infinities and NaN in rows of this class
    big[8, 1::3] = -0.0
    big[9, ::5] = np.inf
    big[10, ::4] = -np.inf
    big[11, :] = np.inf
    big[12, 100:1500] = np.nan
    big[13, :] = np.nan
    t = torch.from_numpy(big).cuda()
    for off in (0, 1):
        view = t[:, off:off + n]
        host = np.ascontiguousarray(big[:, off:off + n])
        for k in (257, 1024):
            gv, gi = fs.kselect(view, k)
            torch.cuda.synchronize()
            ev, ei = oracle.kselect(host, k)
            assert np.array_equal(gi.cpu().numpy(), ei), (n, off, k)
            assert np.array_equal(gv.cpu().numpy().view(np.uint32), ev.view(np.uint32)), (n, off, k)


@pytest.mark.parametrize("k", [2, 100, 300, 1024])
def test_rows_with_many_nans(k):
    """NaN sorts last but passes every bound (the filters test "less than or unordered"): a row whose
    candidates reach k only through NaNs must not be answered from them.  Blocks of NaN in the sampled head,
    NaN scattered through the row, rows with fewer than k real values (there NaNs do belong in the output),
    at row lengths of every class, and as long rows (A4)."""
    rng = np.random.default_rng(k)
    for n in (700, 5000, 8191, 16384, 40000):
        rows = rng.random((12, n), dtype=np.float32)
        rows[0, 100:100 + n // 6] = np.nan          # a block inside the head the scout samples
        rows[1, : n // 2] = np.nan                  # the whole head
        rows[2, ::3] = np.nan                       # scattered
        rows[3, 10:] = np.nan                       # ten real values
        rows[4, : n - 1500] = np.nan                # 1 500 real values at the end
        rows[5, :] = np.nan
        rows[6, n // 3:] = np.nan                   # NaN tail
        rows[7, ::2] = np.inf
        rows[7, 1::4] = np.nan
        rows = np.concatenate([rows, rng.random((300, n), dtype=np.float32)])   # and a GPU's worth of plain rows
        assert_exact(rows, k)
    n = 1 << 19
    long = rng.random((4, n), dtype=np.float32)
    long[0, 1000:200000] = np.nan
    long[1, ::3] = np.nan
    long[2, 700:] = np.nan
    long[3, : n - 5000] = np.nan
    assert_exact(long, k)


def assert_exact_largest(rows_np, k, n=None):
    import paper_1702_08734_b200 as fs
    ev, ei = oracle.kselect(rows_np, k, n=n, largest=True)
    gv, gi = fs.kselect(torch.from_numpy(rows_np).cuda(), k, n=n, largest=True)
    torch.cuda.synchronize()
    gv, gi = gv.cpu().numpy(), gi.cpu().numpy()
    bad = np.nonzero((gi != ei).any(1) | (gv.view(np.uint32) != ev.view(np.uint32)).any(1))[0]
    assert bad.size == 0, "rows %s differ (largest, k=%d); first: got %s want %s" % (
        bad[:5], k, gi[bad[0]][:8], ei[bad[0]][:8])


@pytest.mark.parametrize("k", [1, 2, 32, 100, 256, 257, 1024])
def test_largest_variant(k):
    """fs_kselect_largest ("other comparators") on every path of the selection: batch rows of cfg2's
    shape with duplicated runs, ragged short rows with padding, special values, rows that mislead the
    sample (second filter pass / slow path), and long rows (A4)."""
    dup, _ = datagen.kselect_dup_rows(0, 10000)
    sel = list(np.nonzero(dup)[0][:4]) + [0, 1]
    assert_exact_largest(np.concatenate([datagen.kselect_rows(int(r), 1, 16384) for r in sel]), k)
    assert_exact_largest(datagen.kselect_rows(3, 21, 2003, duplicates=False), k)
    rng = np.random.default_rng(k)
    small = rng.integers(-3, 4, size=(5, 40)).astype(np.float32)
    for n in (0, 1, 5, 40):
        assert_exact_largest(small, k, n=n)
    sp = rng.standard_normal((6, 700)).astype(np.float32)
    sp[0, ::3] = 0.0
    sp[0, 1::3] = -0.0
    sp[1, ::5] = np.inf
    sp[2, ::4] = -np.inf
    sp[3, :] = -np.inf
    sp[4, 10:20] = np.nan
    sp[5, :] = np.nan
    assert_exact_largest(sp, k)
    n = 16384
    asc = np.sort(rng.random(n, dtype=np.float32))
    late = rng.random(n, dtype=np.float32)
    late[-3000:] += 1.0
    few = rng.integers(0, 3, n).astype(np.float32)
    rows = np.stack([asc, asc[::-1].copy(), late, few, np.zeros(n, np.float32)])
    assert_exact_largest(np.concatenate([rows, datagen.kselect_rows(9, 300, n, duplicates=False)[:, :n]]), k)
    n = 1 << 19
    a = np.arange(n, dtype=np.float32)
    lr = datagen.kselect_rows(77, 2, n, duplicates=False)
    assert_exact_largest(np.concatenate([lr, np.stack([a, a[::-1].copy(), (np.arange(n) % 5).astype(np.float32)])]), k)


def test_host_entry_point_and_errors():
    import paper_1702_08734_b200 as fs
    rows = datagen.kselect_rows(7, 5, 3000)
    v, i = fs.kselect_host(rows, 17)
    ev, ei = oracle.kselect(rows, 17)
    assert np.array_equal(i, ei) and np.array_equal(v.view(np.uint32), ev.view(np.uint32))
    t = torch.from_numpy(rows).cuda()
    with pytest.raises(fs.FsError):
        fs.kselect(t, 0)
    with pytest.raises(fs.FsError):
        fs.kselect(t, 1025)
    assert fs.kselect(t[:0], 5)[0].shape == (0, 5)
