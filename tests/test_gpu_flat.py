"""GPU parity: fs_flat_l2_knn (through the C ABI) vs the exact-search oracle.

Acceptance (BASELINE.json north_star): for every returned
(dist, id): |dist - D(j,id)| <= 1e-4 (||x_j||^2 + ||y_id||^2); D(j,id) <= oracle's
k-th distance + that tolerance; ids distinct and in range; distances ascending;
equal returned distances have ascending ids.  On integer-valued data (cfg3)
fp32 arithmetic is exact and the result must equal the oracle bit for bit.
"""
import numpy as np
import pytest
import torch

import datagen
import oracle

pytestmark = pytest.mark.gpu

TOL = 1e-4


def run(xq, xb, k):
    import paper_1702_08734_b200 as fs
    d, i = fs.flat_l2_knn(torch.from_numpy(xq).cuda(), torch.from_numpy(xb).cuda(), k)
    torch.cuda.synchronize()
    return d.cpu().numpy(), i.cpu().numpy()


def check_acceptance(xq, xb, k, gd, gi, od64):
    nq, nb = xq.shape[0], xb.shape[0]
    kk = min(k, nb)
    xn = (xq.astype(np.float64) ** 2).sum(1)
    yn = (xb.astype(np.float64) ** 2).sum(1)
    assert np.all(gi[:, kk:] == -1) and np.all(np.isposinf(gd[:, kk:]))
    ids = gi[:, :kk]
    assert ids.min() >= 0 and ids.max() < nb
    assert all(len(set(r.tolist())) == kk for r in ids), "duplicate ids"
    exact = oracle.pair_l2(xq, xb, ids)
    tol = TOL * (xn[:, None] + yn[ids])
    assert np.all(np.abs(gd[:, :kk].astype(np.float64) - exact) <= tol), "distance off"
    assert np.all(exact <= od64[:, kk - 1:kk] + tol), "returned id is not a k-NN within tolerance"
    dd = np.diff(gd[:, :kk], axis=1)
    assert np.all(dd >= 0), "not ascending"
    same = dd == 0
    assert np.all(np.diff(ids, axis=1)[same] > 0), "ties not by ascending id"


def test_cfg1_tiny_full():
    """BASELINE.json configs[0]: nb=8192, nq=64, d=64, ~N(0,1), seed 0, k=10."""
    xb = datagen.gaussian_vectors(0, 8192, 64)
    xq = datagen.gaussian_vectors(8192, 64, 64)
    od, oi, od64 = oracle.flat_l2_knn(xq, xb, 10, want64=True)
    gd, gi = run(xq, xb, 10)
    check_acceptance(xq, xb, 10, gd, gi, od64)
    assert (gi == oi).mean() > 0.999  # real-valued data: ids agree except at rounding near-ties


@pytest.mark.parametrize("nq,nb,d,k", [
    (1, 1, 1, 1), (3, 5, 2, 3), (65, 129, 3, 7), (70, 1000, 17, 32), (130, 3001, 64, 33),
    (64, 2500, 128, 100), (33, 777, 96, 128), (17, 5000, 100, 1024), (200, 4099, 24, 1),
    (5, 300, 130, 400),
    # d % 32 != 0 on the tensor-core engine: the last 32-column stage is partly zero-filled by TMA
    (40, 3000, 36, 10), (128, 2000, 68, 50), (260, 9000, 100, 10), (33, 4000, 124, 1),
])
def test_shapes_real_valued(nq, nb, d, k):
    rng = np.random.default_rng(nq * 7 + nb)
    xb = rng.standard_normal((nb, d)).astype(np.float32)
    xq = rng.standard_normal((nq, d)).astype(np.float32)
    _, _, od64 = oracle.flat_l2_knn(xq, xb, k, want64=True)
    gd, gi = run(xq, xb, k)
    check_acceptance(xq, xb, k, gd, gi, od64)


def test_misaligned_operands():
    """Operands that start 4 bytes off a 16-byte boundary: TMA cannot read them in place, the engine
    works on truncated copies; real-valued data so that the lo planes are read too."""
    import paper_1702_08734_b200 as fs
    rng = np.random.default_rng(5)
    nq, nb, d, k = 70, 6000, 96, 10
    xb = rng.standard_normal((nb, d)).astype(np.float32)
    xq = rng.standard_normal((nq, d)).astype(np.float32)
    bb = torch.empty(nb * d + 1, dtype=torch.float32, device="cuda")
    qq = torch.empty(nq * d + 1, dtype=torch.float32, device="cuda")
    tb, tq = bb[1:].view(nb, d), qq[1:].view(nq, d)
    tb.copy_(torch.from_numpy(xb))
    tq.copy_(torch.from_numpy(xq))
    assert tb.data_ptr() % 16 == 4 and tq.data_ptr() % 16 == 4
    gd, gi = fs.flat_l2_knn(tq, tb, k)
    torch.cuda.synchronize()
    _, _, od64 = oracle.flat_l2_knn(xq, xb, k, want64=True)
    check_acceptance(xq, xb, k, gd.cpu().numpy(), gi.cpu().numpy(), od64)


@pytest.mark.parametrize("d", [36, 100])
def test_partial_last_stage_integer_data_bit_exact(d):
    """d % 32 != 0 through the tensor-core engine (zero-filled tail of the last stage): small-integer data,
    where every product and partial sum is an exact fp32 integer, must equal the oracle bit for bit."""
    import paper_1702_08734_b200 as fs
    assert "d % 4" in fs.flat_engine()
    rng = np.random.default_rng(d)
    xb = rng.integers(0, 256, (20000, d)).astype(np.float32)
    xq = rng.integers(0, 256, (300, d)).astype(np.float32)
    xb[777] = xq[5]  # an exact duplicate: distance 0
    for k in (1, 10, 100):
        od, oi = oracle.flat_l2_knn(xq, xb, k)
        gd, gi = run(xq, xb, k)
        assert np.array_equal(gi, oi) and np.array_equal(gd, od)


@pytest.mark.parametrize("k", [1, 10, 100])
def test_cfg3_shaped_integer_data_bit_exact(k):
    """cfg3 recipe at reduced size: integer data -> bit-exact ids and distances,
    exact ties resolved by lower id (many with few distinct values)."""
    xb = datagen.sift_like(0, 20000)
    xq = datagen.sift_like(1_000_000, 150)
    xb[5000:5040] = xb[100:140]  # exact duplicates -> exact ties
    od, oi = oracle.flat_l2_knn(xq, xb, k)
    gd, gi = run(xq, xb, k)
    assert np.array_equal(gi, oi)
    assert np.array_equal(gd.view(np.uint32), od.view(np.uint32))


@pytest.mark.parametrize("k", [2, 10, 13, 16, 40, 100, 1024])
def test_sampled_bound_integer_data_bit_exact(k):
    """Databases of >= 32 768 rows take the sampled bound of the tensor-core engine (DESIGN 5.2): a strided
    sample is searched first and its c-th distance bounds every queue.  Integer data: bit-exact.  The second
    half of the queries has its nearest rows planted exactly ON the sample positions, so the sampled bound is
    too tight for them and they must come out of the re-run (B4 sees fewer than k keys)."""
    nb, nq = 40000, 300
    xb = datagen.sift_like(0, nb)
    xq = datagen.sift_like(1_000_000, nq)
    stride = nb // 4096                       # ns = 4096 for this nb (flat_tc_plan)
    rng = np.random.default_rng(k)
    for q in range(nq // 2, nq):              # 160 near-copies of the query at sample positions
        pos = rng.choice(4096, 160, replace=False) * stride
        xb[pos] = np.clip(xq[q][None, :] + rng.integers(-2, 3, size=(160, xb.shape[1])), 0, 255).astype(np.float32)
    od, oi = oracle.flat_l2_knn(xq, xb, k)
    gd, gi = run(xq, xb, k)
    assert np.array_equal(gi, oi)
    assert np.array_equal(gd.view(np.uint32), od.view(np.uint32))


def test_sampled_bound_real_valued():
    xb = datagen.gaussian_vectors(0, 50000, 96)
    xq = datagen.gaussian_vectors(50000, 200, 96)
    for k in (5, 100):
        _, oi, od64 = oracle.flat_l2_knn(xq, xb, k, want64=True)
        gd, gi = run(xq, xb, k)
        check_acceptance(xq, xb, k, gd, gi, od64)
        assert (gi == oi).mean() > 0.999


def test_handworked_and_duplicates():
    xb = np.array([[0, 0], [3, 4], [6, 8], [3, 4], [-3, 4]], np.float32)
    xq = np.array([[0, 0], [3, 4]], np.float32)
    gd, gi = run(xq, xb, 3)
    assert gi.tolist() == [[0, 1, 3], [1, 3, 0]] and gd.tolist() == [[0, 25, 25], [0, 0, 25]]
    gd, gi = run(xq, xb, 7)  # k > nb pads
    assert gi[:, 5:].tolist() == [[-1, -1], [-1, -1]] and np.all(np.isposinf(gd[:, 5:]))


def test_empty_and_errors():
    import paper_1702_08734_b200 as fs
    xq = torch.zeros((4, 8), device="cuda")
    d, i = fs.flat_l2_knn(xq, torch.zeros((0, 8), device="cuda"), 3)
    assert np.all(i.cpu().numpy() == -1) and np.all(np.isposinf(d.cpu().numpy()))
    d, i = fs.flat_l2_knn(xq[:0], torch.zeros((5, 8), device="cuda"), 3)
    assert d.shape == (0, 3)
    with pytest.raises(fs.FsError):
        fs.flat_l2_knn(xq, torch.zeros((5, 8), device="cuda"), 2000)


def test_host_entry_point():
    import paper_1702_08734_b200 as fs
    xb = datagen.sift_like(0, 3000)
    xq = datagen.sift_like(1_000_000, 20)
    gd, gi = fs.flat_l2_knn_host(xq, xb, 10)
    od, oi = oracle.flat_l2_knn(xq, xb, 10)
    assert np.array_equal(gi, oi) and np.array_equal(gd, od)


def test_mma_ignores_low_mantissa_bits():
    """The tensor-core engine reads the caller's fp32 arrays as the TF32 hi plane (DESIGN 5.2): tcgen05.mma
    kind::tf32 must ignore the 13 low mantissa bits.  FS_TC_PLANES=1 makes the library feed explicitly
    truncated copies instead; both runs must agree bit for bit on real-valued data."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = (
        "import sys, numpy as np, torch; sys.path.insert(0, %r)\n"
        "import paper_1702_08734_b200 as fs\n"
        "from datagen import gen_torch as gt\n"
        "d, i = fs.flat_l2_knn(gt.gaussian_vectors(50000, 300, 128), gt.gaussian_vectors(0, 50000, 128), 10)\n"
        "torch.cuda.synchronize()\n"
        "sys.stdout.write(d.cpu().numpy().tobytes().hex() + i.cpu().numpy().tobytes().hex())\n" % root)
    outs = []
    for planes in ("0", "1"):
        env = dict(os.environ, FS_TC_PLANES=planes)
        r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        outs.append(r.stdout)
    assert outs[0] == outs[1] and len(outs[0]) > 0


def _both(xq, xb, k, view_off=0):
    """(unprepared, prepared) results of the same search; xb may be a column-offset view start (misaligned)."""
    import paper_1702_08734_b200 as fs
    q = torch.from_numpy(xq).cuda()
    if view_off:
        flat = torch.zeros(xb.size + view_off, dtype=torch.float32, device="cuda")
        flat[view_off:] = torch.from_numpy(xb).cuda().reshape(-1)
        b = flat[view_off:].view(xb.shape)
    else:
        b = torch.from_numpy(xb).cuda()
    d0, i0 = fs.flat_l2_knn(q, b, k)
    prep = fs.flat_prepare(b)
    d1, i1 = fs.flat_l2_knn(q, b, k, prep=prep)
    d2, i2 = fs.flat_l2_knn(q, b, k, prep=prep)  # the block is only read: a second call sees the same
    torch.cuda.synchronize()
    assert torch.equal(d1, d2) and torch.equal(i1, i2)
    return (d0.cpu().numpy(), i0.cpu().numpy()), (d1.cpu().numpy(), i1.cpu().numpy())


@pytest.mark.parametrize("k", [1, 10, 100])
def test_prepared_database_integer_data_bit_exact(k):
    """fs_flat_prepare + fs_flat_l2_knn_prepared (the ||y||^2 of Eq. 2 computed once): the oracle's
    result bit for bit on integer data, on a database large enough for the sampled bound."""
    xb = datagen.sift_like(0, 40000)
    xq = datagen.sift_like(1_000_000, 150)
    xb[5000:5040] = xb[100:140]
    od, oi = oracle.flat_l2_knn(xq, xb, k)
    (d0, i0), (d1, i1) = _both(xq, xb, k)
    assert np.array_equal(i1, oi) and np.array_equal(d1.view(np.uint32), od.view(np.uint32))
    assert np.array_equal(i0, i1) and np.array_equal(d0.view(np.uint32), d1.view(np.uint32))


@pytest.mark.parametrize("case", ["real", "int_db_real_q", "real_db_int_q", "ffma_d30", "ffma_d200", "misaligned"])
def test_prepared_database_equals_the_plain_call(case):
    """Same bits as fs_flat_l2_knn in every operand-split situation: both sides real-valued (3xTF32), only
    the queries (the database's lo plane is zeros but is read), only the database, dimensions of the FFMA
    engine (the block holds the norms only), a database TMA cannot read in place (the block is not used)."""
    rng = np.random.default_rng(7)
    d = {"ffma_d30": 30, "ffma_d200": 200}.get(case, 96)
    nb, nq = 20000, 70
    xb = rng.standard_normal((nb, d)).astype(np.float32)
    xq = rng.standard_normal((nq, d)).astype(np.float32)
    if case == "int_db_real_q":
        xb = np.rint(xb * 8).astype(np.float32)
    if case == "real_db_int_q":
        xq = np.rint(xq * 8).astype(np.float32)
    for k in (1, 10, 100):
        (d0, i0), (d1, i1) = _both(xq, xb, k, view_off=1 if case == "misaligned" else 0)
        assert np.array_equal(i0, i1) and np.array_equal(d0.view(np.uint32), d1.view(np.uint32)), (case, k)
    _, _, od64 = oracle.flat_l2_knn(xq, xb, 10, want64=True)
    (_, _), (d1, i1) = _both(xq, xb, 10)
    check_acceptance(xq, xb, 10, d1, i1, od64)


def test_prepared_database_errors_and_empty():
    import paper_1702_08734_b200 as fs
    xb = torch.zeros((100, 64), device="cuda")
    xq = torch.zeros((4, 64), device="cuda")
    prep = fs.flat_prepare(xb)
    assert prep.numel() == fs.lib().fs_flat_prepare_bytes(100, 64) > 100 * 4
    with pytest.raises(fs.FsError):
        fs.flat_l2_knn(xq, xb, 3, prep=prep[:256])          # too small
    with pytest.raises(fs.FsError):
        fs.flat_l2_knn(xq, xb, 3, prep=prep[16:])           # misaligned (and too small)
    with pytest.raises(fs.FsError):
        fs.flat_prepare(xb, prep=torch.empty(64, dtype=torch.uint8, device="cuda"))
    e = torch.zeros((0, 64), device="cuda")
    d, i = fs.flat_l2_knn(xq, e, 3, prep=fs.flat_prepare(e))
    assert np.all(i.cpu().numpy() == -1) and np.all(np.isposinf(d.cpu().numpy()))
    d, i = fs.flat_l2_knn(xq, xb, 3, prep=prep)             # all-zero data: every distance 0, ids 0..2
    assert i.cpu().numpy().tolist() == [[0, 1, 2]] * 4 and np.all(d.cpu().numpy() == 0)
