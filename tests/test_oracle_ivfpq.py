"""Pins for the IVFADC oracle (oracle.ivfpq_encode / ivfpq_search; Eq. (3)-(7),
(10), (11), Alg. 4 of PAPER.md)."""
import numpy as np
import pytest

import datagen
import oracle
from golden_io import load


def toy_quantizers():
    coarse = np.array([[0, 0], [100, 100]], np.float32)
    pq = np.tile((np.arange(256, dtype=np.float32) - 128.0)[None, :, None], (2, 1, 1))
    return coarse, pq


def random_index(rng, nlist=8, d=12, M=4, nb=600, integer=False):
    if integer:
        coarse = rng.integers(-20, 20, size=(nlist, d)).astype(np.float32)
        pq = rng.integers(-6, 7, size=(M, 256, d // M)).astype(np.float32)
        xb = rng.integers(-25, 25, size=(nb, d)).astype(np.float32)
    else:
        coarse = rng.standard_normal((nlist, d)).astype(np.float32) * 3
        pq = rng.standard_normal((M, 256, d // M)).astype(np.float32)
        xb = (coarse[rng.integers(0, nlist, nb)] + rng.standard_normal((nb, d))).astype(np.float32)
    lst, codes = oracle.ivfpq_encode(coarse, pq, xb)
    offsets, lcodes, lids = oracle.build_lists(lst, codes, np.arange(nb), nlist)
    return coarse, pq, xb, lst, codes, offsets, lcodes, lids


def test_handworked_example():
    g = load("ivfpq_handworked.txt")
    coarse, pq = toy_quantizers()
    y = g["y"].astype(np.float32).reshape(-1, 2)
    lst, codes = oracle.ivfpq_encode(coarse, pq, y)
    assert lst.tolist() == g["lists"].tolist()
    assert codes.reshape(-1).tolist() == g["codes"].tolist()
    x = np.zeros((3, 2), np.float32)
    assert oracle.adc_reconstruct(coarse, pq, x, lst, codes).tolist() == g["dist"].tolist()
    offsets, lcodes, lids = oracle.build_lists(lst, codes, np.arange(3), 2)
    assert offsets.tolist() == [0, 2, 3] and lids.tolist() == [0, 2, 1]
    r1 = oracle.ivfpq_search(coarse, pq, offsets, lcodes, lids, x[:1], nprobe=1, k=3)
    assert r1["probed"][0].tolist() == [0]
    assert r1["ids"][0].tolist() == g["np1_ids"].tolist()
    assert r1["dist"][0, :2].tolist() == [4.0, 13.0] and np.isposinf(r1["dist"][0, 2])
    r2 = oracle.ivfpq_search(coarse, pq, offsets, lcodes, lids, x[:1], nprobe=2, k=3)
    assert r2["ids"][0].tolist() == g["np2_ids"].tolist()
    assert r2["dist"][0].tolist() == g["np2_dist"].tolist()
    assert r2["probed"][0].tolist() == [0, 1] and r2["coarse64"][0].tolist() == [0.0, 20000.0]


def test_handworked_margins():
    """Pins the best/second-best margins of oracle.ivfpq_encode (the outputs the GPU parity
    tests use to excuse near-ties) to values worked by hand in ivfpq_handworked.txt."""
    g = load("ivfpq_handworked.txt")
    coarse, pq = toy_quantizers()
    y = g["y"].astype(np.float32).reshape(-1, 2)
    lst, codes, cm, km = oracle.ivfpq_encode(coarse, pq, y, margins=True)
    assert cm[0] == g["coarse_margin_y0_num"][0] / g["coarse_margin_y0_den"][0]
    assert cm[2] == g["coarse_margin_y2_num"][0] / g["coarse_margin_y2_den"][0]
    assert km[0].tolist() == g["code_margin_y0"].tolist()
    assert km[2].tolist() == g["code_margin_y2"].tolist()      # exact codeword tie -> margin 0
    # y1 = (101.4, 99.6) is not exact in fp32: residual ~(1.4, -0.4); sub-quantizer 0: best codeword 1
    # at 0.4^2, second codeword 2 at 0.6^2 -> (0.36 - 0.16) / 0.36; sub-quantizer 1: 0.4^2 vs 0.6^2 too
    assert np.allclose(km[1], [(0.36 - 0.16) / 0.36] * 2, rtol=0, atol=2e-5)
    assert abs(cm[1] - (20202.12 - 2.12) / 20202.12) < 1e-9
    e = g["extra"].astype(np.float32).reshape(-1, 2)
    el, _, ecm, ekm = oracle.ivfpq_encode(coarse, pq, e, margins=True)
    assert el.tolist() == g["extra_lists"].tolist()            # equidistant -> lower centroid
    assert ecm.tolist() == g["extra_coarse_margin"].tolist()   # equidistant -> 0, on a centroid -> 1


def test_margins_against_sorted_distances():
    """Margins are (second - best) / second of the sorted distance lists (numpy, independent of
    the oracle's running best/second update), in [0, 1], and 0 exactly where two candidates tie."""
    rng = np.random.default_rng(11)
    nlist, d, M, n = 7, 8, 4, 300
    coarse = rng.integers(-3, 4, size=(nlist, d)).astype(np.float32)   # small integers: exact ties occur
    pq = rng.integers(-2, 3, size=(M, 256, d // M)).astype(np.float32)
    y = rng.integers(-4, 5, size=(n, d)).astype(np.float32)
    lst, codes, cm, km = oracle.ivfpq_encode(coarse, pq, y, margins=True)
    dc = ((y[:, None, :].astype(np.float64) - coarse[None]) ** 2).sum(-1)
    s = np.sort(dc, axis=1)
    want = (s[:, 1] - s[:, 0]) / np.maximum(s[:, 1], 1e-300)
    assert np.array_equal(cm, want) and (cm == 0).any() and np.all((cm >= 0) & (cm <= 1))
    assert np.array_equal(lst, dc.argmin(1))
    r = (y.astype(np.float64) - coarse[lst]).reshape(n, M, d // M)
    ds = ((r[:, :, None, :] - pq[None].astype(np.float64)) ** 2).sum(-1)   # [n, M, 256]
    s = np.sort(ds, axis=2)
    want = (s[:, :, 1] - s[:, :, 0]) / np.maximum(s[:, :, 1], 1e-300)
    assert np.array_equal(km, want) and np.all((km >= 0) & (km <= 1))
    assert np.array_equal(codes, ds.argmin(2))


def test_lut_identity_eq10_and_eq11():
    """Reconstruction distance (Eq. 7) == sum of table look-ups (Eq. 10) ==
    term1 + term2 - 2 term3 (Eq. 11), to 1e-12 relative."""
    rng = np.random.default_rng(2)
    coarse, pq, xb, lst, codes, *_ = random_index(rng, nlist=5, d=24, M=8, nb=400)
    for L in range(5):
        x = rng.standard_normal((1, 24)).astype(np.float32)
        cs = codes[rng.integers(0, 400, 50)]
        rec = oracle.adc_reconstruct(coarse, pq, np.repeat(x, 50, 0), np.full(50, L), cs)
        lut, tables = oracle.adc_lut_sum(coarse, pq, x[0], L, cs, want_tables=True)
        eq11 = oracle.adc_eq11(coarse, pq, x[0], L, cs)
        assert np.max(np.abs(rec - lut) / rec) < 1e-12
        assert np.max(np.abs(rec - eq11) / rec) < 1e-12
        # a table entry is itself a squared distance between sub-vectors
        m, j = 3, 77
        sub = slice(m * 3, m * 3 + 3)
        ref = np.sum((x[0, sub].astype(np.float64) - coarse[L, sub] - pq[m, j]) ** 2)
        assert abs(tables[m, j] - ref) < 1e-12 * max(1.0, ref)


def test_encode_against_numpy_bruteforce():
    rng = np.random.default_rng(4)
    coarse, pq, xb, lst, codes, *_ = random_index(rng, integer=True)
    d, M = 12, 4
    D = ((xb[:, None, :].astype(np.float64) - coarse[None]) ** 2).sum(-1)
    assert np.array_equal(lst, np.argmin(D, axis=1))  # argmin takes the first minimum
    res = xb.astype(np.float64) - coarse[lst]
    for m in range(M):
        sub = res[:, m * 3:(m + 1) * 3]
        Dm = ((sub[:, None, :] - pq[m][None].astype(np.float64)) ** 2).sum(-1)
        assert np.array_equal(codes[:, m], np.argmin(Dm, axis=1))


def test_exhaustive_limit_equals_bruteforce_adc():
    """nprobe = nlist makes Eq. (6) equal Eq. (4): compare with an ADC
    scan over all vectors that ignores the lists."""
    rng = np.random.default_rng(6)
    coarse, pq, xb, lst, codes, offsets, lcodes, lids = random_index(rng, integer=True)
    xq = rng.integers(-25, 25, size=(7, 12)).astype(np.float32)
    r = oracle.ivfpq_search(coarse, pq, offsets, lcodes, lids, xq, nprobe=8, k=20)
    for j in range(7):
        recon = coarse[lst].astype(np.float64) + np.concatenate(
            [pq[m][codes[:, m]] for m in range(4)], axis=1)
        dist = ((xq[j].astype(np.float64) - recon) ** 2).sum(1)
        order = np.lexsort((np.arange(600), dist))[:20]
        assert r["ids"][j].tolist() == order.tolist()
        assert np.array_equal(r["dist64"][j], dist[order])


def test_lossless_limit_equals_exact_search():
    """If every database vector is exactly c_L + a codeword combination then
    q(y) = y and IVFPQ with nprobe = nlist equals the exact-search oracle."""
    rng = np.random.default_rng(8)
    nlist, d, M = 4, 8, 4
    coarse = (rng.integers(-4, 5, size=(nlist, d)) * 64).astype(np.float32)  # far apart
    pq = np.zeros((M, 256, 2), np.float32)
    pq[:, :, 0] = (np.arange(256) % 16) - 8
    pq[:, :, 1] = (np.arange(256) // 16) - 8
    nb = 500
    L = rng.integers(0, nlist, nb)
    c = rng.integers(0, 256, size=(nb, M))
    xb = coarse[L] + np.concatenate([pq[m][c[:, m]] for m in range(M)], axis=1)
    lst, codes = oracle.ivfpq_encode(coarse, pq, xb)
    recon = coarse[lst] + np.concatenate([pq[m][codes[:, m]] for m in range(M)], axis=1)
    assert np.array_equal(recon, xb)
    offsets, lcodes, lids = oracle.build_lists(lst, codes, np.arange(nb), nlist)
    xq = rng.integers(-300, 300, size=(6, d)).astype(np.float32)
    r = oracle.ivfpq_search(coarse, pq, offsets, lcodes, lids, xq, nprobe=nlist, k=15)
    dist, ids = oracle.flat_l2_knn(xq, xb, 15)
    assert np.array_equal(r["ids"], ids) and np.array_equal(r["dist"], dist)


def test_degenerate_quantizers():
    rng = np.random.default_rng(10)
    # nlist = 1 with a zero centroid -> plain PQ-ADC
    d, M = 8, 8  # M = d: per-dimension scalar quantisation
    coarse = np.zeros((1, d), np.float32)
    pq = np.tile((np.arange(256, dtype=np.float32) / 8.0 - 16.0)[None, :, None], (M, 1, 1))
    xb = (rng.standard_normal((300, d)) * 4).astype(np.float32)
    lst, codes = oracle.ivfpq_encode(coarse, pq, xb)
    assert np.all(lst == 0)
    grid = pq[0, :, 0].astype(np.float64)
    expect = np.argmin(np.abs(xb.astype(np.float64)[:, :, None] - grid[None, None, :]), axis=2)
    assert np.array_equal(codes, expect)


def test_monotone_in_nprobe_and_probe_order():
    rng = np.random.default_rng(12)
    coarse, pq, xb, lst, codes, offsets, lcodes, lids = random_index(rng, nlist=16, nb=1500)
    xq = rng.standard_normal((10, 12)).astype(np.float32) * 3
    prev = None
    for nprobe in (1, 2, 4, 16):
        r = oracle.ivfpq_search(coarse, pq, offsets, lcodes, lids, xq, nprobe=nprobe, k=10)
        assert np.all(np.diff(r["coarse64"], axis=1) >= 0)
        full = ((xq[:, None, :].astype(np.float64) - coarse[None]) ** 2).sum(-1)
        assert np.array_equal(r["probed"], np.argsort(full, axis=1, kind="stable")[:, :nprobe])
        # every returned id lives in a probed list
        for j in range(10):
            got = r["ids"][j][r["ids"][j] >= 0]
            assert np.all(np.isin(lst[got], r["probed"][j]))
        if prev is not None:  # k-th distance non-increasing in nprobe
            assert np.all(r["dist64"][:, -1] <= prev[:, -1])
        prev = r["dist64"]
    # fixed probe lists reproduce the same step 2-3
    r2 = oracle.ivfpq_search(coarse, pq, offsets, lcodes, lids, xq, nprobe=16, k=10,
                             probed_in=r["probed"])
    assert np.array_equal(r2["ids"], r["ids"])


def test_empty_lists_and_padding():
    coarse, pq = toy_quantizers()
    y = np.array([[3, -2], [2.5, 0]], np.float32)  # both in list 0; list 1 empty
    lst, codes = oracle.ivfpq_encode(coarse, pq, y)
    offsets, lcodes, lids = oracle.build_lists(lst, codes, np.array([10, 11]), 2)
    r = oracle.ivfpq_search(coarse, pq, offsets, lcodes, lids, np.array([[99, 99]], np.float32),
                            nprobe=1, k=2)
    assert r["probed"][0].tolist() == [1] and r["ids"][0].tolist() == [-1, -1]
    r = oracle.ivfpq_search(coarse, pq, offsets, lcodes, lids, np.array([[99, 99]], np.float32),
                            nprobe=2, k=3)
    # (99-2)^2 + 99^2 = 19210 (id 11) < (99-3)^2 + (99+2)^2 = 19417 (id 10)
    assert r["ids"][0].tolist() == [11, 10, -1] and r["dist"][0, :2].tolist() == [19210.0, 19417.0]


def test_cost_identities():
    """P:L290-293 and P:L311, as arithmetic on the configs' numbers."""
    d, b, tau = 96, 16, 64
    assert 256 * d == 24576  # table MACs per (query, list) pair
    assert tau * d * 256 == 64 * 24576  # from scratch
    assert 256 * d + tau * b * 256 < tau * d * 256  # Eq. (11) decomposition is cheaper
