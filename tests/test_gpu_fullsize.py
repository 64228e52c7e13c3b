"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

The oracle cannot run the whole workloads in seconds, so (SURVEY 8c / the tier rules):
  cfg2  all 10 000 x 16 384 rows go through fs_kselect exactly as in bench.py; a seeded
        sample of rows (every duplicate-run pattern included) is compared bit for bit with
        the oracle; the 2^27-element row is checked against the oracle applied to the
        elements <= the k-th value (found with numpy's partition), which is the whole answer.
  cfg3  nb = 10^6, nq = 10^4, d = 128 integer data through fs_flat_l2_knn as in bench.py; a
        seeded sample of queries is compared bit for bit with the oracle.
  cfg4  nb = 10^8, nlist = 65 536, M = 16 and cfg5 nb = 10^9, nlist = 262 144, M = 8 are built in
        full (datagen.IVFPQ_CONFIGS) and checked as SURVEY C-12 says: (i) structure of the
        GPU-built inverted file (sum of lengths, every id exactly once, append order),
        (ii) the add path on >= 10 000 seeded ids regenerated on the CPU and re-encoded by the
        oracle, (iii) the whole 10^4-query batch is searched at every (nprobe, k) of
        BASELINE.json and the rows of a seeded 500 / 200-query subset of THAT output meet the
        oracle run over the GPU-built lists those queries probed (copied out with
        fs_ivfpq_export_lists).  A 2 * 10^6-vector index of the cfg4 shape stays as a quick case.
Inputs come from datagen's torch twin on the device (bit-identical to the numpy generator,
tests/test_datagen.py).
"""
import numpy as np
import pytest
import torch

import datagen
import oracle

pytestmark = pytest.mark.gpu


def fsmod():
    import paper_1702_08734_b200 as fs
    return fs


@pytest.mark.parametrize("k", [1, 32, 128, 1024])
def test_cfg2_full_batch_sampled_rows(k):
    from datagen import gen_torch as gt
    fs = fsmod()
    n_rows, n = 10_000, 16_384
    rows = gt.kselect_rows(0, n_rows, n)
    val, idx = fs.kselect(rows, k)
    torch.cuda.synchronize()
    dup, _ = datagen.kselect_dup_rows(0, n_rows)
    rng = np.random.default_rng(k)
    sample = np.unique(np.concatenate([np.nonzero(dup)[0][:24], rng.integers(0, n_rows, 72), [0, n_rows - 1]]))
    host = rows[torch.from_numpy(sample).cuda()].cpu().numpy()
    for j in range(3):  # device generator == numpy generator
        assert np.array_equal(host[j], datagen.kselect_rows(int(sample[j]), 1, n)[0])
    ev, ei = oracle.kselect(host, k)
    gv, gi = val[torch.from_numpy(sample).cuda()].cpu().numpy(), idx[torch.from_numpy(sample).cuda()].cpu().numpy()
    assert np.array_equal(gi, ei)
    assert np.array_equal(gv.view(np.uint32), ev.view(np.uint32))
    # properties on every row: ascending, values are the row's values at the indices
    v, i = val.cpu().numpy(), idx.cpu().numpy()
    assert np.all(np.diff(v, axis=1) >= 0)
    got = torch.gather(rows, 1, idx.long()).cpu().numpy()
    assert np.array_equal(got.view(np.uint32), v.view(np.uint32))
    eq = np.diff(v, axis=1) == 0
    assert np.all(np.diff(i, axis=1)[eq] > 0), "ties not by ascending index"


def test_cfg2_long_row():
    from datagen import gen_torch as gt
    fs = fsmod()
    n, k = 1 << 27, 1024
    row = gt.kselect_rows(10**6, 1, n, duplicates=False)
    val, idx = fs.kselect(row, k)
    torch.cuda.synchronize()
    host = row[0].cpu().numpy()
    kth = np.partition(host, k - 1)[k - 1]            # independent library routine
    cand = np.nonzero(host <= kth)[0]                 # every element that can be in the answer
    assert k <= cand.size < 4 * k
    ev, ei = oracle.kselect(host[cand][None, :], k)   # the oracle on the candidates = the answer
    assert np.array_equal(idx[0].cpu().numpy(), cand[ei[0]].astype(np.int32))
    assert np.array_equal(val[0].cpu().numpy().view(np.uint32), ev[0].view(np.uint32))


@pytest.mark.parametrize("kind", ["ascending", "descending", "constant"])
def test_cfg2_long_row_structured(kind):
    """The 2^27-element row when it is sorted or constant: the answer is known in closed form."""
    fs = fsmod()
    n, k = 1 << 27, 1024
    if kind == "constant":
        row = torch.full((1, n), 0.25, dtype=torch.float32, device="cuda")
        want_idx = np.arange(k)
        want_val = np.full(k, 0.25, np.float32)
    else:
        asc = torch.arange(n, dtype=torch.float32, device="cuda")  # exact up to 2^24, then runs of equal values
        row = (asc if kind == "ascending" else asc.flip(0))[None, :].contiguous()
        host = row[0].cpu().numpy()
        if kind == "ascending":
            want_idx = np.arange(k)
        else:  # the k smallest values sit at the end; equal values (runs above 2^24 only) keep index order
            want_idx = np.arange(n - 1, n - 1 - k, -1)
        want_val = host[want_idx]
    val, idx = fs.kselect(row, k)
    torch.cuda.synchronize()
    assert np.array_equal(idx[0].cpu().numpy(), want_idx.astype(np.int32))
    assert np.array_equal(val[0].cpu().numpy().view(np.uint32), want_val.view(np.uint32))


@pytest.mark.parametrize("k", [1, 10, 100])
def test_cfg3_full_sampled_queries(k):
    from datagen import gen_torch as gt
    fs = fsmod()
    nb, nq = 1_000_000, 10_000
    xb = gt.sift_like(0, nb)
    xq = gt.sift_like(nb, nq)
    gd, gi = fs.flat_l2_knn(xq, xb, k)
    torch.cuda.synchronize()
    rng = np.random.default_rng(100 + k)
    sample = np.unique(np.concatenate([rng.integers(0, nq, 14), [0, nq - 1]]))
    xb_h = xb.cpu().numpy()
    assert np.array_equal(xb_h[:64], datagen.sift_like(0, 64))
    od, oi = oracle.flat_l2_knn(xq[torch.from_numpy(sample).cuda()].cpu().numpy(), xb_h, k)
    s = torch.from_numpy(sample).cuda()
    assert np.array_equal(gi[s].cpu().numpy(), oi)                       # integer data: exact
    assert np.array_equal(gd[s].cpu().numpy().view(np.uint32), od.view(np.uint32))
    d_all, i_all = gd.cpu().numpy(), gi.cpu().numpy()
    assert np.all(np.diff(d_all, axis=1) >= 0) and i_all.min() >= 0 and i_all.max() < nb


def test_cfg3_k100_ten_runs_identical_bits():
    """The flat engine shares bounds between CTAs while they run (gbound / hbound, sampled bound, re-run of
    failed queries): whatever the interleaving, the output is one fixed answer.  Ten runs of cfg3 at k = 100
    on integer data and ten on real-valued data (3xTF32) must give identical bits."""
    from datagen import gen_torch as gt
    fs = fsmod()
    nb, nq, k = 1_000_000, 10_000, 100
    for gen in (gt.sift_like, lambda r0, n: gt.gaussian_vectors(r0, n, 128)):
        xb, xq = gen(0, nb), gen(nb, nq)
        d0, i0 = fs.flat_l2_knn(xq, xb, k)
        for _ in range(9):
            d1, i1 = fs.flat_l2_knn(xq, xb, k)
            assert torch.equal(i0, i1)
            assert torch.equal(d0.view(torch.int32), d1.view(torch.int32))
        del xb, xq


def test_cfg4_shaped_index():
    from datagen import gen_torch as gt
    from test_gpu_ivfpq import check_search
    fs = fsmod()
    d, M, nb, nlist, nq, k = 96, 16, 2_000_000, 2048, 2000, 100
    ix = fs.IvfPq(d, nlist, M)
    ix.train(gt.deep_like(0, 64 * nlist), niter=6, seed=0)
    chunk = 1 << 19
    for b in range(0, nb, chunk):
        ix.add(gt.deep_like(b, min(chunk, nb - b)))
    assert ix.ntotal == nb
    coarse, pq = (t.cpu().numpy() for t in ix.get_quantizers())
    offs, codes, lids = (t.cpu().numpy() for t in ix.export())
    # structure: every id exactly once, lists in append (= ascending id) order
    assert offs[0] == 0 and offs[-1] == nb and np.all(np.diff(offs) >= 0)
    assert np.array_equal(np.sort(lids), np.arange(nb))
    inner = np.ones(nb, bool)
    inner[offs[1:-1][offs[1:-1] < nb]] = False
    assert np.all(np.diff(lids)[inner[1:]] > 0)
    # sampled add path: the oracle re-encodes seeded ids from regenerated vectors
    rng = np.random.default_rng(7)
    sid = np.unique(rng.integers(0, nb, 3000))
    ys = np.concatenate([datagen.deep_like(int(i), 1) for i in sid[:400]])
    sid = sid[:400]
    olist, ocodes, cm, km = oracle.ivfpq_encode(coarse, pq, ys, margins=True)
    pos = np.empty(nb, np.int64)
    pos[lids] = np.arange(nb)
    glist = np.searchsorted(offs, pos[sid], side="right") - 1
    assert not ((glist != olist) & (cm >= 1e-5)).any()
    same = glist == olist
    assert not ((codes[pos[sid]] != ocodes) & (km >= 1e-5) & same[:, None]).any()
    # search: whole batch as bench.py runs it, oracle on a seeded subset over the GPU-built lists
    xq = gt.deep_like(10**8, nq)
    for nprobe in (16, 64):
        gd, gi = ix.search(xq, nprobe, k)
        torch.cuda.synchronize()
        sub = np.unique(rng.integers(0, nq, 24))
        xs = xq[torch.from_numpy(sub).cuda()].cpu().numpy()
        sd, si, _ = check_search(ix, coarse, pq, offs, codes, lids, xs, nprobe, k)
        # batch run vs subset run: the dispatch may pick different scan kernels for the two (float
        # tables / fixed-point tables, DESIGN 5.3), so near-ties may swap; everything else is equal
        bi_s = gi[torch.from_numpy(sub).cuda()].cpu().numpy()
        bd_s = gd[torch.from_numpy(sub).cuda()].cpu().numpy()
        assert np.allclose(bd_s, sd, rtol=1e-3, atol=0)
        assert (bi_s == si).mean() >= 0.98
    ix.close()


def _full_config(cfg):
    """SURVEY C-12 (i)-(iii) on BASELINE.json configs[3] / configs[4] at their stated size."""
    from datagen import gen_torch as gt
    from test_gpu_ivfpq import verify_search
    fs = fsmod()
    c = datagen.IVFPQ_CONFIGS[cfg]
    nb, d, nlist, M, nq = c["nb"], c["d"], c["nlist"], c["M"], c["nq"]
    ix = fs.IvfPq(d, nlist, M)
    ix.train(gt.deep_like(0, c["ntrain"]), niter=10, seed=0)
    chunk = 1 << 22
    for b in range(0, nb, chunk):
        ix.add(gt.deep_like(b, min(chunk, nb - b)))
    assert ix.ntotal == nb
    coarse, pq = (t.cpu().numpy() for t in ix.get_quantizers())
    assert np.isfinite(coarse).all() and np.isfinite(pq).all()
    offs_d, codes_d, lids_d = ix.export()
    torch.cuda.synchronize()

    # (i) structure, on the device copy of the inverted file
    offs = offs_d.cpu().numpy()
    assert offs[0] == 0 and offs[-1] == nb and np.all(np.diff(offs) >= 0)
    assert lids_d.numel() == nb and int(lids_d.sum().item()) == nb * (nb - 1) // 2
    x = lids_d.clone()
    while x.numel() > 1:                        # xor of all ids = xor of 0..nb-1
        if x.numel() & 1:
            x = torch.cat([x, x.new_zeros(1)])
        h = x.numel() // 2
        x = x[:h] ^ x[h:]
    want_xor = [nb - 1, 1, nb, 0][(nb - 1) % 4]  # xor of 0..m for m = nb - 1
    assert int(x.item()) == want_xor
    del x
    pos = torch.empty(nb, dtype=torch.int64, device="cuda")
    pos[lids_d] = torch.arange(nb, dtype=torch.int64, device="cuda")
    step = 1 << 26
    for a in range(0, nb, step):                # every id is stored, and nb slots in all: exactly once
        e = min(nb, a + step)
        assert torch.equal(lids_d[pos[a:e]], torch.arange(a, e, dtype=torch.int64, device="cuda"))
    asc = lids_d[1:] > lids_d[:-1]              # append order = ascending id inside every list
    inner = offs_d[1:-1]
    inner = inner[(inner > 0) & (inner < nb)]
    asc[inner - 1] = True
    assert bool(asc.all())
    del asc
    for L in datagen.unique_sample_ids(64, nlist, stream=10 * cfg + 5).tolist():   # sort-unique on sampled lists
        seg = lids_d[offs[L]:offs[L + 1]]
        assert torch.unique(seg).numel() == seg.numel()

    # (ii) sampled add path: regenerate seeded ids on the CPU, oracle steps 1-3 of Add
    sid = datagen.unique_sample_ids(c["add_check"], nb, stream=10 * cfg + 7)
    ys = datagen.deep_like(0, 0, ids=sid)
    for t in range(3):                          # device generator == numpy generator at these ids
        assert np.array_equal(ys[t], gt.deep_like(int(sid[t]), 1).cpu().numpy()[0])
    olist, ocodes, cm, km = oracle.ivfpq_encode(coarse, pq, ys, margins=True)
    p = pos[torch.from_numpy(sid).cuda()]
    glist = (torch.searchsorted(offs_d, p, right=True) - 1).cpu().numpy()
    gcodes = codes_d[p].cpu().numpy()
    assert not ((glist != olist) & (cm >= 1e-5)).any(), "coarse assignment differs beyond near-ties"
    same = glist == olist
    assert not ((gcodes != ocodes) & (km >= 1e-5) & same[:, None]).any(), "codes differ beyond near-ties"
    assert same.mean() > 0.999 and (gcodes == ocodes)[same].mean() > 0.999
    del pos, offs_d, codes_d, lids_d
    torch.cuda.empty_cache()

    # (iii) full batch at every (nprobe, k); the seeded subset of that output meets the oracle
    xq = gt.deep_like(nb, nq)
    sub = datagen.unique_sample_ids(c["check_queries"], nq, stream=10 * cfg + 6)
    xs = xq[torch.from_numpy(sub).cuda()].cpu().numpy()
    assert np.array_equal(xs[:2], datagen.deep_like(0, 0, ids=nb + sub[:2]))
    runs = []
    for nprobe, k in c["searches"]:
        gd, gi, gp = ix.search(xq, nprobe, k, want_probed=True)
        torch.cuda.synchronize()
        st = torch.from_numpy(sub).cuda()
        runs.append((nprobe, k, gd[st].cpu().numpy(), gi[st].cpu().numpy(), gp[st].cpu().numpy()))
        i_all = gi.cpu().numpy()
        assert i_all.max() < nb and np.all(np.diff(gd.cpu().numpy(), axis=1) >= 0)
    lists = np.unique(np.concatenate([r[4].reshape(-1) for r in runs]))
    so, sc, si = ix.export_lists(lists)
    offs_sub = np.zeros(nlist + 1, np.int64)    # CSR over all lists, the ones never probed empty
    lens = np.zeros(nlist, np.int64)
    lens[lists] = np.diff(so)
    np.cumsum(lens, out=offs_sub[1:])
    codes_sub, lids_sub = sc.cpu().numpy(), si.cpu().numpy()
    del sc, si
    for nprobe, k, gd, gi, gp in runs:
        verify_search(coarse, pq, offs_sub, codes_sub, lids_sub, xs, nprobe, k, gd, gi, gp)
    ix.close()


def test_cfg4_full():
    _full_config(4)


def test_cfg5_full():
    _full_config(5)
