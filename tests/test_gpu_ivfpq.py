"""GPU parity: fs_ivfpq_add / fs_ivfpq_search (through the C ABI) vs the IVFADC oracle.

Acceptance (BASELINE.json north_star, reading C-12):
  add     list number and code of every vector equal the oracle's, except where the
          oracle's best and second-best (coarse or sub-quantizer) distances differ by
          < 1e-5 relative; every id stored exactly once; lists keep append order.
  search  probed lists identical to the oracle's except at coarse near-ties; every
          returned (dist, id) has id in a probed list, |dist - ADC| <= 1e-3 ADC, and
          ADC <= (1 + 1e-3) * the oracle's k-th ADC distance over the same lists;
          ascending, distinct ids, exact ties in ascending id order.
Both sides use the same quantizer arrays (reading C-11).
"""
import numpy as np
import pytest
import torch

import datagen
import oracle

pytestmark = pytest.mark.gpu

RTOL = 1e-3


def fsmod():
    import paper_1702_08734_b200 as fs
    return fs


def make_index(d, nlist, M, coarse, pq):
    fs = fsmod()
    ix = fs.IvfPq(d, nlist, M)
    ix.set_quantizers(torch.from_numpy(coarse).cuda(), torch.from_numpy(pq).cuda())
    return ix


def check_add(ix, coarse, pq, xb, ids=None):
    nb = xb.shape[0]
    nlist, M = coarse.shape[0], pq.shape[0]
    ids = np.arange(nb, dtype=np.int64) if ids is None else ids
    offs, codes, lids = (t.cpu().numpy() for t in ix.export())
    assert offs[0] == 0 and offs[-1] == nb and np.all(np.diff(offs) >= 0)
    # every id exactly once
    assert np.array_equal(np.sort(lids), np.sort(ids))
    pos_of = np.empty(nb, np.int64)
    order = np.argsort(ids, kind="stable")
    rank = np.empty(nb, np.int64)
    rank[order] = np.arange(nb)
    where = {int(i): p for p, i in enumerate(lids)}
    pos_of = np.array([where[int(i)] for i in ids])
    glist = np.searchsorted(offs, pos_of, side="right") - 1
    gcodes = codes[pos_of]
    olist, ocodes, cm, km = oracle.ivfpq_encode(coarse, pq, xb, margins=True)
    bad_list = (glist != olist) & (cm >= 1e-5)
    assert not bad_list.any(), "coarse assignment differs at %s" % np.nonzero(bad_list)[0][:5]
    same = glist == olist
    bad_code = (gcodes != ocodes) & (km >= 1e-5) & same[:, None]
    assert not bad_code.any(), "codes differ at %s" % np.argwhere(bad_code)[:5]
    assert same.mean() > 0.999 and (gcodes == ocodes)[same].mean() > 0.999
    # append order: arrival order inside every list
    arrival = rank[np.array([np.nonzero(ids == i)[0][0] for i in lids])] if nb <= 2000 else None
    if arrival is not None:
        for L in range(nlist):
            seg = arrival[offs[L]:offs[L + 1]]
            assert np.all(np.diff(seg) > 0), "list %d lost append order" % L
    return offs, codes, lids


def verify_search(coarse, pq, offs, codes, lids, xq, nprobe, k, gd, gi, gp):
    """The acceptance predicates of the header on GPU outputs (gd, gi, gp) for the queries xq.

    (offs, codes, lids) is the GPU-built inverted file in CSR form on the host; for the big
    configs it is the sub-index of the lists these queries probe (every other list empty).
    Look-ups go through one sort of lids, so 10^8-entry files are fine."""
    nq = xq.shape[0]
    # (1) probed lists vs the oracle's own coarse step (Eq. 5)
    o1 = oracle.ivfpq_search(coarse, pq, offs, codes, lids, xq, nprobe, k)
    xn = (xq.astype(np.float64) ** 2).sum(1)
    cn = (coarse.astype(np.float64) ** 2).sum(1)
    for q in range(nq):
        assert len(set(gp[q].tolist())) == nprobe, "probed lists repeat"
        if np.array_equal(gp[q], o1["probed"][q]):
            continue
        kth = o1["coarse64"][q, -1]
        for L in set(gp[q].tolist()) ^ set(o1["probed"][q].tolist()):
            dL = ((xq[q].astype(np.float64) - coarse[L]) ** 2).sum()
            assert abs(dL - kth) <= 1e-4 * (xn[q] + cn[L]), "probed list %d of query %d is no near-tie" % (L, q)
    # (2) steps 2-3 over the lists the GPU probed
    o = oracle.ivfpq_search(coarse, pq, offs, codes, lids, xq, nprobe, k, probed_in=gp)
    order = np.argsort(lids, kind="stable")
    sorted_ids = lids[order]
    n_exact = 0
    for q in range(nq):
        valid = gi[q] >= 0
        nv = int(valid.sum())
        assert nv == int((o["ids"][q] >= 0).sum()), "wrong number of results"
        assert np.all(gi[q, nv:] == -1) and np.all(np.isposinf(gd[q, nv:]))
        if nv == 0:
            continue
        ids = gi[q, :nv]
        assert len(set(ids.tolist())) == nv, "duplicate ids"
        at = np.searchsorted(sorted_ids, ids)
        assert np.all(at < len(sorted_ids)) and np.array_equal(sorted_ids[np.minimum(at, len(sorted_ids) - 1)], ids), \
            "id not stored in the (probed part of the) inverted file"
        pos = order[at]
        list_of = np.searchsorted(offs, pos, side="right") - 1
        assert np.isin(list_of, gp[q]).all(), "id outside the probed lists"
        adc = oracle.adc_reconstruct(coarse, pq, np.repeat(xq[q:q + 1], nv, 0), list_of, codes[pos])
        assert np.all(np.abs(gd[q, :nv] - adc) <= RTOL * adc + 1e-30), "ADC distance off"
        kth = o["dist64"][q, nv - 1]
        assert np.all(adc <= (1 + RTOL) * kth + 1e-30), "returned id is not in the top-k within tolerance"
        dd = np.diff(gd[q, :nv])
        assert np.all(dd >= 0), "not ascending"
        assert np.all(np.diff(ids)[dd == 0] > 0), "exact ties not in ascending id order"
        n_exact += int(np.array_equal(ids, o["ids"][q, :nv]))
    assert n_exact >= 0.9 * nq, "only %d of %d queries match the oracle id for id" % (n_exact, nq)
    return n_exact


def check_search(ix, coarse, pq, offs, codes, lids, xq, nprobe, k):
    gd, gi, gp = ix.search(torch.from_numpy(xq).cuda(), nprobe, k, want_probed=True)
    torch.cuda.synchronize()
    gd, gi, gp = gd.cpu().numpy(), gi.cpu().numpy(), gp.cpu().numpy()
    verify_search(coarse, pq, offs, codes, lids, xq, nprobe, k, gd, gi, gp)
    return gd, gi, gp


def test_handworked_example():
    """tests/golden/ivfpq_handworked.txt through the GPU path (d=2, M=2, dsub=1)."""
    from golden_io import load
    g = load("ivfpq_handworked.txt")
    coarse = np.array([[0, 0], [100, 100]], np.float32)
    pq = np.tile((np.arange(256, dtype=np.float32) - 128.0)[None, :, None], (2, 1, 1)).copy()
    y = g["y"].astype(np.float32).reshape(-1, 2)
    ix = make_index(2, 2, 2, coarse, pq)
    ix.add(torch.from_numpy(y).cuda())
    offs, codes, lids = (t.cpu().numpy() for t in ix.export())
    assert offs.tolist() == [0, 2, 3] and lids.tolist() == [0, 2, 1]
    assert codes[np.argsort(lids)].reshape(-1).tolist() == g["codes"].tolist()
    x = torch.zeros((1, 2), device="cuda")
    d1, i1 = ix.search(x, 1, 3)
    assert i1.cpu().numpy()[0].tolist() == g["np1_ids"].tolist()
    assert d1.cpu().numpy()[0, :2].tolist() == [4.0, 13.0] and np.isposinf(d1.cpu().numpy()[0, 2])
    d2, i2, p2 = ix.search(x, 2, 3, want_probed=True)
    assert i2.cpu().numpy()[0].tolist() == g["np2_ids"].tolist()
    assert d2.cpu().numpy()[0].tolist() == g["np2_dist"].tolist()
    assert p2.cpu().numpy()[0].tolist() == [0, 1]
    ix.close()


@pytest.mark.parametrize("M,nlist", [(8, 64), (16, 100), (4, 1), (24, 7)])
def test_tiny_config_trained_quantizers(M, nlist):
    """SURVEY C-12 tiny config at reduced size: d=96 deep-like data, quantizers trained
    by fs_ivfpq_train (off the parity path) and shared with the oracle."""
    fs = fsmod()
    d, nb, nq = 96, 20000, 60
    xb = datagen.deep_like(0, nb)
    xq = datagen.deep_like(10**8, nq)
    ix = fs.IvfPq(d, nlist, M)
    ix.train(torch.from_numpy(xb[:8000]).cuda(), niter=4, seed=1)
    coarse, pq = (t.cpu().numpy() for t in ix.get_quantizers())
    assert np.isfinite(coarse).all() and np.isfinite(pq).all()
    half = nb // 2 + 13
    ix.add(torch.from_numpy(xb[:half]).cuda())     # two adds: staging keeps arrival order
    ix.add(torch.from_numpy(xb[half:]).cuda())
    assert ix.ntotal == nb
    offs, codes, lids = check_add(ix, coarse, pq, xb)
    for nprobe in sorted({1, min(8, nlist), nlist}):
        for k in (1, 100):
            check_search(ix, coarse, pq, offs, codes, lids, xq, nprobe, k)
    assert ix.last_scanned_codes > 0
    ix.close()


def test_search_between_adds_and_custom_ids():
    """Finalise, add more, search again (re-finalise merges old lists and new vectors);
    caller-supplied int64 ids; k > number of candidates pads."""
    rng = np.random.default_rng(5)
    d, nlist, M, nb = 32, 9, 8, 1500
    coarse = rng.standard_normal((nlist, d)).astype(np.float32)
    pq = (0.3 * rng.standard_normal((M, 256, d // M))).astype(np.float32)
    xb = (coarse[rng.integers(0, nlist, nb)] + 0.3 * rng.standard_normal((nb, d))).astype(np.float32)
    xq = (coarse[rng.integers(0, nlist, 40)] + 0.3 * rng.standard_normal((40, d))).astype(np.float32)
    ids = (np.arange(nb, dtype=np.int64) * 7919 + (1 << 40))
    ix = make_index(d, nlist, M, coarse, pq)
    ix.add(torch.from_numpy(xb[:700]).cuda(), torch.from_numpy(ids[:700]).cuda())
    offs, codes, lids = check_add(ix, coarse, pq, xb[:700], ids[:700])
    check_search(ix, coarse, pq, offs, codes, lids, xq, 3, 10)
    ix.add(torch.from_numpy(xb[700:]).cuda(), torch.from_numpy(ids[700:]).cuda())
    offs, codes, lids = check_add(ix, coarse, pq, xb, ids)
    for nprobe, k in ((1, 1), (3, 10), (9, 1024), (2, 300)):
        check_search(ix, coarse, pq, offs, codes, lids, xq, nprobe, k)
    ix.close()


def test_exact_ties_and_lossless_limit():
    """Vectors that are exactly centroid + codewords (integers): ADC distances are exact
    in fp32, identical codes give exactly equal distances -> results equal the oracle
    bit for bit, ties by ascending id; and with nprobe = nlist they equal exact search."""
    rng = np.random.default_rng(11)
    d, nlist, M, nb = 16, 4, 4, 900
    coarse = (rng.integers(-3, 4, size=(nlist, d)) * 40).astype(np.float32)
    pq = rng.integers(-8, 9, size=(M, 256, d // M)).astype(np.float32)
    for m in range(M):  # distinct codewords so that encoding is unambiguous
        pq[m, :, 0] = np.arange(256) - 128
    L = rng.integers(0, nlist, nb)
    cw = rng.integers(0, 256, size=(nb, M))
    cw[300:330] = cw[0:30]
    L[300:330] = L[0:30]   # exact duplicates -> exact ties
    xb = coarse[L] + np.concatenate([pq[m, cw[:, m]] for m in range(M)], axis=1)
    xb = xb.astype(np.float32)
    xq = xb[rng.integers(0, nb, 25)] + rng.integers(-2, 3, size=(25, d)).astype(np.float32)
    ix = make_index(d, nlist, M, coarse, pq)
    ix.add(torch.from_numpy(xb).cuda())
    offs, codes, lids = (t.cpu().numpy() for t in ix.export())
    for nprobe, k in ((nlist, 20), (2, 50), (nlist, 1)):
        gd, gi, gp = ix.search(torch.from_numpy(xq).cuda(), nprobe, k, want_probed=True)
        o = oracle.ivfpq_search(coarse, pq, offs, codes, lids, xq, nprobe, k, probed_in=gp.cpu().numpy())
        assert np.array_equal(gi.cpu().numpy(), o["ids"])
        assert np.array_equal(gd.cpu().numpy(), o["dist"])
    fd, fi = oracle.flat_l2_knn(xq, xb, 20)
    gd, gi = ix.search(torch.from_numpy(xq).cuda(), nlist, 20)
    assert np.array_equal(gi.cpu().numpy(), fi) and np.array_equal(gd.cpu().numpy(), fd)
    ix.close()


def test_empty_index_empty_lists_errors_and_host_entry():
    fs = fsmod()
    rng = np.random.default_rng(3)
    d, nlist, M = 8, 5, 2
    coarse = rng.standard_normal((nlist, d)).astype(np.float32) * 5
    pq = rng.standard_normal((M, 256, d // M)).astype(np.float32)
    ix = fs.IvfPq(d, nlist, M)
    xq = torch.from_numpy(rng.standard_normal((3, d)).astype(np.float32)).cuda()
    with pytest.raises(fs.FsError):
        ix.search(xq, 1, 1)            # no quantizers: FS_ESTATE
    ix.set_quantizers(torch.from_numpy(coarse).cuda(), torch.from_numpy(pq).cuda())
    dd, ii = ix.search(xq, 2, 4)       # empty index: padding only
    assert np.all(ii.cpu().numpy() == -1) and np.all(np.isposinf(dd.cpu().numpy()))
    xb = (coarse[[0, 0, 3]] + 0.01).astype(np.float32)   # lists 1, 2, 4 stay empty
    ix.add(torch.from_numpy(xb).cuda())
    dd, ii, pp = ix.search(xq, nlist, 4, want_probed=True)
    assert sorted(ii.cpu().numpy()[0, :3].tolist()) == [0, 1, 2] and ii.cpu().numpy()[0, 3] == -1
    assert sorted(pp.cpu().numpy()[0].tolist()) == list(range(nlist))
    with pytest.raises(fs.FsError):
        ix.search(xq, nlist + 1, 1)
    with pytest.raises(fs.FsError):
        ix.search(xq, 1, 2000)
    hd, hi = ix.search_host(xq.cpu().numpy(), nlist, 4)
    assert np.array_equal(hi, ii.cpu().numpy()) and np.array_equal(hd, dd.cpu().numpy())
    ix.close()


def test_many_lists_per_item_duplicates():
    """d = 96, M = 16 with >= 32 lists per (query, list group) and enough items: the shape at which
    the dispatch picks the grouped fixed-point scan (DESIGN 5.3).  A tenth of the database are
    exact duplicates of other vectors: identical codes in one list must come back with identical
    distances, in ascending id order (reading C-6)."""
    fs = fsmod()
    d, M, nlist, nb, nq, nprobe, k = 96, 16, 64, 60000, 1400, 32, 100
    xb = datagen.deep_like(0, nb).copy()
    rng = np.random.default_rng(5)
    src = rng.integers(0, nb, nb // 10)
    dst = rng.integers(0, nb, nb // 10)
    xb[dst] = xb[src]
    xq = datagen.deep_like(10**8, nq)
    ix = fs.IvfPq(d, nlist, M)
    ix.train(torch.from_numpy(xb[:20000]).cuda(), niter=4, seed=2)
    coarse, pq = (t.cpu().numpy() for t in ix.get_quantizers())
    ix.add(torch.from_numpy(xb).cuda())
    offs, codes, lids = (t.cpu().numpy() for t in ix.export())
    # the whole batch goes through check_search: it is the launch configuration that reaches the
    # persistent kernel (>= 32 lists per item, >= 1 332 items)
    check_search(ix, coarse, pq, offs, codes, lids, xq, nprobe, k)
    bd, bi = ix.search(torch.from_numpy(xq).cuda(), nprobe, k)
    torch.cuda.synchronize()
    # duplicates: equal codes in the same list -> bitwise-equal distances
    pos_of = np.empty(nb, np.int64)
    pos_of[lids] = np.arange(nb)
    list_of = np.searchsorted(offs, np.arange(nb), side="right") - 1
    bi_h, bd_h = bi.cpu().numpy(), bd.cpu().numpy()
    checked = 0
    for q in range(0, nq, 7):
        ids = bi_h[q][bi_h[q] >= 0]
        p = pos_of[ids]
        key = [(int(list_of[x]), codes[x].tobytes()) for x in p]
        seen = {}
        for j, kk in enumerate(key):
            if kk in seen:
                assert bd_h[q, j] == bd_h[q, seen[kk]], "equal codes, different distances"
                checked += 1
            seen[kk] = j
    assert checked > 0
    ix.close()


@pytest.mark.parametrize("M", [8, 16])
def test_d128_shapes(M):
    """d = 128 (SIFT-like integer-valued data): dsub = 16 / 8, the other shapes with an unrolled
    table build."""
    fs = fsmod()
    d, nlist, nb, nq = 128, 32, 12000, 40
    xb = datagen.sift_like(0, nb)
    xq = datagen.sift_like(10**7, nq)
    ix = fs.IvfPq(d, nlist, M)
    ix.train(torch.from_numpy(xb[:6000]).cuda(), niter=4, seed=3)
    coarse, pq = (t.cpu().numpy() for t in ix.get_quantizers())
    ix.add(torch.from_numpy(xb).cuda())
    offs, codes, lids = check_add(ix, coarse, pq, xb)
    for nprobe, k in ((4, 10), (nlist, 100)):
        check_search(ix, coarse, pq, offs, codes, lids, xq, nprobe, k)
    ix.close()


def test_c1_large_nlist():
    """A coarse quantizer of 32 768 centroids with nprobe = 64: C1 goes through the distance matrix
    (DESIGN 5.3); tests/test_gpu_ivfpq_variants.py runs it again in passes of 512 queries, whose last
    pass (188 queries) takes the long-row k-selection plan."""
    fs = fsmod()
    d, M, nlist, nb, nq, nprobe, k = 96, 16, 32768, 50000, 700, 64, 10
    coarse = datagen.deep_like(5 * 10**7, nlist)
    rng = np.random.default_rng(11)
    pq = (0.05 * rng.standard_normal((M, 256, d // M))).astype(np.float32)
    xb = datagen.deep_like(0, nb)
    xq = datagen.deep_like(10**8, nq)
    ix = make_index(d, nlist, M, coarse, pq)
    ix.add(torch.from_numpy(xb).cuda())
    offs, codes, lids = (t.cpu().numpy() for t in ix.export())
    check_search(ix, coarse, pq, offs, codes, lids, xq, nprobe, k)
    ix.close()


@pytest.mark.parametrize("d,M,nlist,nq,nprobe,k", [
    (96, 16, 16, 300, 16, 5),      # nprobe = nlist = 16: the k-selection of C1 takes every column
    (96, 16, 17, 257, 17, 100),    # nlist not a multiple of 4: padded row stride of the distance matrix
    (96, 8, 33, 400, 33, 1),
    (64, 16, 40, 1000, 40, 10),
    (128, 16, 20, 260, 16, 7),
    (96, 16, 64, 3000, 48, 100),   # >= 32 lists per item and enough items: grouped fixed-point scan
])
def test_c1_matrix_and_scan_edge_shapes(d, M, nlist, nq, nprobe, k):
    """nq >= 256 and nprobe >= 16 on small coarse quantizers: C1 through the distance matrix, with the
    scan kernel the dispatch picks for the shape (DESIGN 5.3)."""
    rng = np.random.default_rng(nlist * 1000 + nq)
    coarse = rng.standard_normal((nlist, d)).astype(np.float32)
    pq = (0.2 * rng.standard_normal((M, 256, d // M))).astype(np.float32)
    nb = 5000
    xb = (coarse[rng.integers(0, nlist, nb)] + 0.3 * rng.standard_normal((nb, d))).astype(np.float32)
    xq = (coarse[rng.integers(0, nlist, nq)] + 0.3 * rng.standard_normal((nq, d))).astype(np.float32)
    ix = make_index(d, nlist, M, coarse, pq)
    ix.add(torch.from_numpy(xb).cuda())
    offs, codes, lids = (t.cpu().numpy() for t in ix.export())
    check_search(ix, coarse, pq, offs, codes, lids, xq, nprobe, k)
    ix.close()
