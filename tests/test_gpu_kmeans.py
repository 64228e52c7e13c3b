"""GPU parity of fs_kmeans (through the C ABI) with oracle.kmeans_step (section 6.2):
one Lloyd iteration from identical initial centroids; several iterations; determinism; empty clusters."""
import numpy as np
import pytest
import torch

import datagen
import oracle

pytestmark = pytest.mark.gpu


def fsmod():
    import paper_1702_08734_b200 as fs
    return fs


def one_step(x, c0, seed=0):
    fs = fsmod()
    gc, ga = fs.kmeans(torch.from_numpy(x).cuda(), c0.shape[0], 1, seed=seed, centroids=torch.from_numpy(c0).cuda(),
                       want_assign=True)
    torch.cuda.synchronize()
    return gc.cpu().numpy(), ga.cpu().numpy()


@pytest.mark.parametrize("d,K,n", [(96, 64, 20000), (6, 256, 30000), (128, 300, 9000), (12, 256, 5000), (50, 7, 1000)])
def test_one_step_matches_oracle(d, K, n):
    """d = 96 / 128 take the tensor-core assignment, the others the FFMA engine; dsub-sized d as in PQ training."""
    x = datagen.deep_like(0, n, d=d) if d >= 32 else datagen.gaussian_vectors(0, n, d)
    c0 = x[(np.arange(K) * n) // K].copy()
    gc, ga = one_step(x, c0)
    oc, oa, mg = oracle.kmeans_step(x, c0, margins=True)
    bad = (ga != oa) & (mg >= 1e-5)
    assert not bad.any(), "assignment differs beyond near-ties at %s" % np.nonzero(bad)[0][:5]
    if np.array_equal(ga, oa):
        scale = np.abs(oc).max()
        assert np.all(np.abs(gc - oc) <= 1e-5 * scale), "centroids differ from the oracle's means"
    else:  # near-ties moved a few points: compare the clusters nobody moved in or out of
        moved = np.zeros(K, bool)
        moved[ga[ga != oa]] = True
        moved[oa[ga != oa]] = True
        assert moved.sum() <= max(2, K // 20)
        assert np.all(np.abs(gc[~moved] - oc[~moved]) <= 1e-5 * np.abs(oc).max())


def test_init_iterations_determinism_and_empty_clusters():
    fs = fsmod()
    n, d, K = 12000, 96, 50
    x = datagen.deep_like(0, n, d=d)
    tx = torch.from_numpy(x).cuda()
    # init: evenly strided points, then the same steps as the oracle
    c = x[(np.arange(K) * n) // K].copy()
    for it in range(3):
        c, _ = oracle.kmeans_step(x, c, seed=9, it=it)
    g1 = fs.kmeans(tx, K, 3, seed=9).cpu().numpy()
    assert np.all(np.abs(g1 - c) <= 3e-5 * np.abs(c).max())      # three steps: rounding of the means feeds back
    g2 = fs.kmeans(tx, K, 3, seed=9).cpu().numpy()
    assert np.array_equal(g1.view(np.uint32), g2.view(np.uint32))  # deterministic update: bit-identical runs
    # empty clusters: two centroids far from every point are re-seeded by the stated rule
    c0 = x[:K].copy()
    c0[3] += 100.0
    c0[17] -= 100.0
    gc, ga = one_step(x, c0, seed=4)
    oc, oa = oracle.kmeans_step(x, c0, seed=4, it=0)
    assert not (ga == 3).any() and not (ga == 17).any()
    assert np.array_equal(gc[3], oc[3]) and np.array_equal(gc[17], oc[17])
    assert fs.kmeans(tx, K, 0, seed=1).shape == (K, d)             # niter = 0: the initial points


def test_trained_index_is_reproducible():
    """fs_ivfpq_train twice on the same sample: bit-identical quantizers (round 1 used float atomics)."""
    fs = fsmod()
    xb = torch.from_numpy(datagen.deep_like(0, 8000)).cuda()
    qs = []
    for _ in range(2):
        ix = fs.IvfPq(96, 40, 16)
        ix.train(xb, niter=3, seed=2)
        qs.append([t.cpu().numpy() for t in ix.get_quantizers()])
        ix.close()
    assert np.array_equal(qs[0][0].view(np.uint32), qs[1][0].view(np.uint32))
    assert np.array_equal(qs[0][1].view(np.uint32), qs[1][1].view(np.uint32))
