"""GPU parity of the shard-merge path: the database cut into contiguous id
shards, each searched on its own through the C ABI, the partial lists joined by fs_merge_topk.  One GPU
runs the shards one after another (the exchange step is covered by tests/test_multirank.py over gloo)."""
import numpy as np
import pytest
import torch

import datagen
import oracle

pytestmark = pytest.mark.gpu


def fsmod():
    import paper_1702_08734_b200 as fs
    return fs


def test_merge_topk_against_oracle():
    """Lists as shards produce them: sorted by (distance, id), shard g's ids below shard g + 1's (fs.h:
    that order is what makes ties at the k-th place exact); many exact ties, padding at the tails."""
    fs = fsmod()
    rng = np.random.default_rng(3)
    for nq, G, kk in ((5, 1, 7), (33, 2, 10), (64, 8, 100), (3, 3, 1024), (17, 5, 33)):
        d = rng.integers(0, 50, size=(nq, G, kk)).astype(np.float32)
        i = np.empty((nq, G, kk), np.int64)
        for q in range(nq):
            for g in range(G):
                ids = np.sort(rng.choice(10 * kk, kk, replace=False)) + g * 10 * kk   # shard g: ids in [g 10 kk, (g + 1) 10 kk)
                o = np.lexsort((ids, d[q, g]))
                d[q, g], i[q, g] = d[q, g][o], ids[o]
        pad = rng.integers(0, 3, size=(nq, G))
        for q in range(nq):
            for g in range(G):
                if pad[q, g]:
                    i[q, g, -pad[q, g]:] = -1
                    d[q, g, -pad[q, g]:] = np.inf
        gd, gi = fs.merge_topk(torch.from_numpy(d).cuda(), torch.from_numpy(i).cuda())
        od, oi = oracle.merge_topk(d, i, kk)
        assert np.array_equal(gi.cpu().numpy(), oi)
        assert np.array_equal(gd.cpu().numpy(), od)
    # ids in no particular order, distinct distances: the order of the lists does not matter
    d = rng.permutation(4 * 3 * 20).reshape(4, 3, 20).astype(np.float32)
    d.sort(axis=2)
    i = rng.permutation(10**6)[:4 * 3 * 20].reshape(4, 3, 20).astype(np.int64) + (1 << 40)
    gd, gi = fs.merge_topk(torch.from_numpy(d).cuda(), torch.from_numpy(i).cuda())
    od, oi = oracle.merge_topk(d, i, 20)
    assert np.array_equal(gi.cpu().numpy(), oi) and np.array_equal(gd.cpu().numpy(), od)


@pytest.mark.parametrize("G,k", [(2, 10), (3, 100), (8, 1)])
def test_flat_shards_equal_unsharded(G, k):
    """Integer-valued data (exact arithmetic, many ties): G shards + merge == one search, bit for bit,
    and == the oracle."""
    from paper_1702_08734_b200 import multirank as mr
    fs = fsmod()
    nb, nq = 50_000, 300
    xb = datagen.sift_like(0, nb)
    xb[30_000:30_050] = xb[10:60]          # duplicates in different shards: ties across shards
    xq = datagen.sift_like(10**6, nq)
    tb, tq = torch.from_numpy(xb).cuda(), torch.from_numpy(xq).cuda()
    wd, wi = fs.flat_l2_knn(tq, tb, k)
    parts_d, parts_i = [], []
    for g in range(G):
        first, n = mr.shard_range(g, G, nb)
        d, i = fs.flat_l2_knn(tq, tb[first:first + n].contiguous(), k)
        parts_d.append(d)
        parts_i.append(torch.where(i >= 0, i + first, i))
    md, mi = fs.merge_topk(torch.stack(parts_d, 1).contiguous(), torch.stack(parts_i, 1).contiguous())
    assert torch.equal(mi, wi) and torch.equal(md, wd)
    od, oi = oracle.flat_l2_knn(xq, xb, k)
    assert np.array_equal(mi.cpu().numpy(), oi) and np.array_equal(md.cpu().numpy(), od)


def test_ivfpq_shards_equal_unsharded():
    """IVFPQ: every shard holds all lists over its own vectors and the same quantizers; the
    merged result equals the single index's (same ADC distances: equal codes, equal tables)."""
    from paper_1702_08734_b200 import multirank as mr
    fs = fsmod()
    d, nlist, M, nb, nq, nprobe, k, G = 96, 64, 16, 40_000, 200, 8, 50, 3
    xb = datagen.deep_like(0, nb)
    xq = datagen.deep_like(10**8, nq)
    whole = fs.IvfPq(d, nlist, M)
    whole.train(torch.from_numpy(xb[:10_000]).cuda(), niter=4, seed=1)
    coarse, pq = whole.get_quantizers()
    whole.add(torch.from_numpy(xb).cuda())
    tq = torch.from_numpy(xq).cuda()
    wd, wi = whole.search(tq, nprobe, k)
    parts_d, parts_i = [], []
    for g in range(G):
        first, n = mr.shard_range(g, G, nb)
        ix = fs.IvfPq(d, nlist, M)
        ix.set_quantizers(coarse, pq)
        ix.add(torch.from_numpy(xb[first:first + n]).cuda(),
               torch.arange(first, first + n, dtype=torch.int64, device="cuda"))   # global ids
        dd, ii = ix.search(tq, nprobe, k)
        parts_d.append(dd)
        parts_i.append(ii)
        ix.close()
    md, mi = fs.merge_topk(torch.stack(parts_d, 1).contiguous(), torch.stack(parts_i, 1).contiguous())
    assert torch.equal(mi, wi) and torch.equal(md, wd)
    whole.close()
