"""Pins for the k-means oracle (oracle.kmeans_step; section 6.2 of PAPER.md)."""
import numpy as np

import datagen
import oracle
from golden_io import load


def test_handworked_step():
    g = load("kmeans_handworked.txt")
    x = g["points"].astype(np.float32)[:, None]
    c = g["centroids"].astype(np.float32)[:, None]
    seed, it = 5, 3
    out, assign, mg = oracle.kmeans_step(x, c, seed=seed, it=it, margins=True)
    assert assign.tolist() == g["assign"].tolist()          # the tie at 2.5 goes to the lower centroid
    assert out[0, 0] == np.float32(g["new_c0"][0]) and out[1, 0] == np.float32(g["new_c1"][0])
    assert np.array_equal(mg, g["margin_num"] / g["margin_den"])
    # empty cluster: the stated hashed re-seed, recomputed with datagen's own splitmix64 finaliser
    U = np.uint64
    with np.errstate(over="ignore"):
        a = datagen.mix64(U(seed) + U(0x9E3779B97F4A7C15) * U(it + 1))
        src = int(datagen.mix64(a + U(2)) % U(len(x)))
    assert out[2, 0] == x[src, 0]


def test_two_blobs_converge_in_one_step():
    """Two well-separated blobs, one initial centroid near each: one Lloyd step lands on the blob means
    (computed here independently in double); a second step changes nothing."""
    rng = np.random.default_rng(0)
    a = rng.standard_normal((300, 5)).astype(np.float32)
    b = (rng.standard_normal((200, 5)) + 50.0).astype(np.float32)
    x = np.concatenate([a, b])[rng.permutation(500)]
    near_a = (x.astype(np.float64) ** 2).sum(1) < 25.0 ** 2 * 5
    c0 = np.array([[1.0] * 5, [45.0] * 5], np.float32)
    out, assign = oracle.kmeans_step(x, c0)
    assert np.array_equal(assign == 0, near_a)
    want = np.stack([x[near_a].astype(np.float64).mean(0), x[~near_a].astype(np.float64).mean(0)])
    assert np.allclose(out, want, rtol=1e-6, atol=1e-6)
    out2, assign2 = oracle.kmeans_step(x, out)
    assert np.array_equal(assign2, assign) and np.array_equal(out2, out)


def test_step_against_numpy_and_objective_decreases():
    """Assignment = numpy argmin of the squared distances (first minimum = lower centroid), and the
    k-means objective never increases over Lloyd steps (a textbook invariant)."""
    x = datagen.deep_like(0, 800, d=16)
    c = x[::100].copy()
    prev = np.inf
    for it in range(4):
        d2 = ((x[:, None, :].astype(np.float64) - c[None].astype(np.float64)) ** 2).sum(-1)
        out, assign = oracle.kmeans_step(x, c, seed=1, it=it)
        assert np.array_equal(assign, d2.argmin(1))
        obj = d2.min(1).sum()
        assert obj <= prev * (1 + 1e-12)
        prev = obj
        c = out
