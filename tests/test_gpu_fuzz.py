"""GPU parity on seeded random shapes and adversarial row contents: fs_kselect (both comparators) and
fs_flat_l2_knn (integer data, with and without a prepared database) against the oracle, bit for bit.
The fixed parity tests pick their shapes by hand; these pick them at random (sizes around every class
boundary, strides, misaligned starts, every k class) so that a path nobody thought of meets the oracle too."""
import numpy as np
import pytest
import torch

import oracle

pytestmark = pytest.mark.gpu


def _row(n, rng):
    t = int(rng.integers(0, 14))
    x = rng.random(n, dtype=np.float32)
    if t == 1:
        x = np.sort(x)
    elif t == 2:
        x = np.sort(x)[::-1].copy()
    elif t == 3:
        x[:] = rng.random()
    elif t == 4:
        x = np.floor(x * rng.integers(2, 50)).astype(np.float32)
    elif t == 5:
        x = (x * 1e38).astype(np.float32) * rng.choice([-1, 1], n).astype(np.float32)
    elif t == 6:
        x = (x * 1e-40).astype(np.float32)          # denormals
    elif t in (7, 8, 9):
        m = rng.random(n) < rng.random()
        x[m] = (np.inf, -np.inf, np.nan)[t - 7]
    elif t == 10:
        x[:] = 1.0
        idx = rng.integers(0, n, max(1, n // 50))
        x[idx] = rng.random(idx.size)
    elif t == 11:
        x = np.repeat(rng.random(n // 64 + 1, dtype=np.float32), 64)[:n].copy()
    elif t == 12:
        x = x + 1.0
        x[rng.integers(0, n):] -= 1.0               # the small values come late
    elif t == 13:
        x = np.where(rng.random(n) < 0.5, 0.0, -0.0).astype(np.float32)
        x[rng.integers(0, n, 3)] = -1.0
    return x


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_kselect_random_shapes_and_contents(seed):
    import paper_1702_08734_b200 as fs
    rng = np.random.default_rng(seed)
    for case in range(60):
        n = int(rng.choice([rng.integers(1, 300), rng.integers(300, 9000), rng.integers(9000, 70000)]))
        nr = int(rng.integers(1, 40)) if n > 9000 else int(rng.integers(1, 500))
        k = int(rng.choice([1, 2, rng.integers(1, 33), rng.integers(33, 257), rng.integers(257, 1025), 1024]))
        pad, off = int(rng.integers(0, 5)), int(rng.integers(0, 4))
        rows = np.stack([_row(n + pad + off, rng) for _ in range(nr)])
        view = torch.from_numpy(rows).cuda()[:, off:off + n]
        host = np.ascontiguousarray(rows[:, off:off + n])
        largest = bool(rng.integers(0, 2))
        gv, gi = fs.kselect(view, k, largest=largest)
        torch.cuda.synchronize()
        ev, ei = oracle.kselect(host, k, largest=largest)
        what = (seed, case, n, nr, k, off, largest)
        assert np.array_equal(gi.cpu().numpy(), ei), what
        assert np.array_equal(gv.cpu().numpy().view(np.uint32), ev.view(np.uint32)), what


@pytest.mark.parametrize("seed", [0, 1])
def test_flat_random_shapes_integer_data(seed):
    import paper_1702_08734_b200 as fs
    rng = np.random.default_rng(100 + seed)
    for case in range(40):
        d = int(rng.choice([rng.integers(1, 40), 4 * rng.integers(8, 33), 4 * rng.integers(8, 33), rng.integers(129, 200)]))
        nb = int(rng.choice([rng.integers(1, 300), rng.integers(300, 9000), rng.integers(9000, 50000)]))
        nq = int(rng.choice([rng.integers(1, 10), rng.integers(10, 200)]))
        k = int(rng.choice([1, rng.integers(1, 13), rng.integers(13, 65), rng.integers(65, 300), rng.integers(300, 1025)]))
        hi = int(rng.choice([2, 4, 16, 200]))
        xb = rng.integers(0, hi, size=(nb, d)).astype(np.float32)
        xq = rng.integers(0, hi, size=(nq, d)).astype(np.float32)
        if nb > 50:
            xb[rng.integers(0, nb, 30)] = xb[rng.integers(0, nb, 30)]   # exact duplicates: ties by id
        b, q = torch.from_numpy(xb).cuda(), torch.from_numpy(xq).cuda()
        prep = fs.flat_prepare(b) if case % 2 else None
        gd, gi = fs.flat_l2_knn(q, b, k, prep=prep)
        torch.cuda.synchronize()
        od, oi = oracle.flat_l2_knn(xq, xb, k)
        what = (seed, case, nq, nb, d, k, hi, prep is not None)
        assert np.array_equal(gi.cpu().numpy(), oi), what
        assert np.array_equal(gd.cpu().numpy().view(np.uint32), od.view(np.uint32)), what
