"""Pins for the exact-search oracle (oracle.flat_l2_knn, Eq. (1), D squared P:L52)."""
import numpy as np
import pytest

import datagen
import oracle
from golden_io import load


def test_handworked_example():
    g = load("flat_handworked.txt")
    xb = g["xb"].astype(np.float32).reshape(-1, 2)
    xq = g["xq"].astype(np.float32).reshape(-1, 2)
    full = oracle.pair_l2(xq, xb, np.tile(np.arange(5), (2, 1)))
    assert full[0].tolist() == g["D0"].tolist() and full[1].tolist() == g["D1"].tolist()
    dist, ids = oracle.flat_l2_knn(xq, xb, 3)
    assert dist[0].tolist() == g["k3_dist0"].tolist() and ids[0].tolist() == g["k3_ids0"].tolist()
    assert dist[1].tolist() == g["k3_dist1"].tolist() and ids[1].tolist() == g["k3_ids1"].tolist()


def test_bruteforce_independent():
    """Against an independent implementation: Eq. (2) expansion in numpy double + lexsort."""
    rng = np.random.default_rng(5)
    for nb, d in [(1, 1), (7, 3), (32, 4), (200, 17)]:
        xb = rng.integers(-3, 4, size=(nb, d)).astype(np.float32)  # exact, many ties
        xq = rng.integers(-3, 4, size=(9, d)).astype(np.float32)
        for k in {1, min(3, nb), nb}:
            dist, ids, d64 = oracle.flat_l2_knn(xq, xb, k, want64=True)
            q, b = xq.astype(np.float64), xb.astype(np.float64)
            D = (q * q).sum(1)[:, None] + (b * b).sum(1)[None, :] - 2.0 * q @ b.T  # Eq. (2)
            for j in range(9):
                order = np.lexsort((np.arange(nb), D[j]))[:k]
                assert ids[j].tolist() == order.tolist()
                assert np.array_equal(d64[j], D[j][order])


def test_eq2_equals_direct_form_in_double():
    """Eq. (2) P:L54 vs the direct form on real-valued data, 1e-12 relative."""
    xb = datagen.gaussian_vectors(0, 500, 64)
    xq = datagen.gaussian_vectors(500, 20, 64)
    ids = np.tile(np.arange(500), (20, 1))
    direct = oracle.pair_l2(xq, xb, ids)
    q, b = xq.astype(np.float64), xb.astype(np.float64)
    D = (q * q).sum(1)[:, None] + (b * b).sum(1)[None, :] - 2.0 * q @ b.T
    assert np.max(np.abs(D - direct) / direct) < 1e-12


def test_identities():
    rng = np.random.default_rng(9)
    xb = rng.standard_normal((300, 8)).astype(np.float32)
    xb[17] = xb[250]  # duplicates: a query equal to a database vector -> 0, lowest id first
    dist, ids = oracle.flat_l2_knn(xb[250:251], xb, 2)
    assert dist[0].tolist() == [0.0, 0.0] and ids[0].tolist() == [17, 250]
    # k = nb returns a permutation of all ids, ascending distances
    dist, ids = oracle.flat_l2_knn(xb[:4], xb, 300)
    assert all(sorted(r.tolist()) == list(range(300)) for r in ids)
    assert np.all(np.diff(dist, axis=1) >= 0)
    # d = 1 reduces to sorting (x - y)^2
    y = rng.integers(-50, 50, size=(64, 1)).astype(np.float32)
    dist, ids = oracle.flat_l2_knn(np.array([[0.5]], np.float32), y, 64)
    key = (0.5 - y[:, 0].astype(np.float64)) ** 2
    assert ids[0].tolist() == np.lexsort((np.arange(64), key)).tolist()
    # permuting dimensions / translating by an exactly representable offset keeps ids
    xi = rng.integers(-8, 8, size=(100, 6)).astype(np.float32)
    qi = rng.integers(-8, 8, size=(5, 6)).astype(np.float32)
    _, ids0 = oracle.flat_l2_knn(qi, xi, 10)
    perm = rng.permutation(6)
    _, ids1 = oracle.flat_l2_knn(qi[:, perm], xi[:, perm], 10)
    _, ids2 = oracle.flat_l2_knn(qi + 16.0, xi + 16.0, 10)
    assert np.array_equal(ids0, ids1) and np.array_equal(ids0, ids2)


def test_padding_when_k_exceeds_nb():
    xb = np.array([[1.0], [0.0]], np.float32)
    dist, ids = oracle.flat_l2_knn(np.array([[0.0]], np.float32), xb, 4)
    assert ids[0].tolist() == [1, 0, -1, -1]
    assert dist[0, :2].tolist() == [0.0, 1.0] and np.all(np.isposinf(dist[0, 2:]))


def test_sift_like_data_is_integer_exact():
    """cfg3's data are integers in [0,255], d=128: ||x||^2+||y||^2 < 2^24, so every
    term of Eq. (2) is an exact fp32 integer and the oracle's
    double result is an integer representable in fp32."""
    xb = datagen.sift_like(0, 2000)
    xq = datagen.sift_like(1_000_000, 8)
    assert xb.min() >= 0 and xb.max() <= 255 and np.all(xb == np.rint(xb))
    assert (xb.astype(np.float64) ** 2).sum(1).max() * 2 < 2 ** 24
    dist, ids, d64 = oracle.flat_l2_knn(xq, xb, 10, want64=True)
    assert np.all(d64 == np.rint(d64)) and np.all(dist.astype(np.float64) == d64)
