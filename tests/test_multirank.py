"""N > 1 host logic on CPU: 2 ranks over gloo (the GPU runs use the same functions over nccl)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world_size, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world_size)
    from paper_1702_08734_b200 import multirank as mr
    import datagen
    r, w = mr.world()
    first, n = mr.rank_rows(r, 5)
    rows = datagen.kselect_rows(first, n, 64)           # this rank's rows, from the shared generator
    # ranges are disjoint and consecutive
    t = torch.tensor([first, n], dtype=torch.int64)
    got = [torch.zeros(2, dtype=torch.int64) for _ in range(w)]
    dist.all_gather(got, t)
    ranges = [(int(g[0]), int(g[1])) for g in got]
    mr.barrier()
    slow = mr.max_over_ranks(10.0 + 5.0 * r)            # rank 1 is the slow one
    val = mr.job_throughput(1000.0, slow, w)
    if r == 0:
        out.put((ranges, slow, val, float(rows[0, 0])))
    dist.destroy_process_group()


def test_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    ranges, slow, val, first_val = out.get()
    assert ranges == [(0, 5), (5, 5)]
    assert slow == 15.0                                   # max over ranks, not rank 0's own time
    assert abs(val - 2 * 1000.0 / 15e-3) < 1e-6           # all ranks' units over the slowest time
    import datagen
    assert first_val == float(datagen.kselect_rows(0, 1, 64)[0, 0])


def test_single_process_defaults():
    from paper_1702_08734_b200 import multirank as mr
    assert mr.world() == (0, 1)
    assert mr.max_over_ranks(3.5) == 3.5
    assert mr.rank_rows(3, 10_000) == (30_000, 10_000)


def _shard_worker(rank, world_size, port, out):
    """Database sharding over 2 gloo ranks, the ORACLE as the local search and as the merge: the host
    logic (shard ranges, id offsets, one all-gather, slot order) must reproduce the unsharded oracle."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world_size)
    import numpy as np
    import datagen
    import oracle
    from paper_1702_08734_b200 import multirank as mr
    nb, nq, k = 1001, 7, 12                              # odd sizes: uneven shards
    xb = datagen.sift_like(0, nb, d=32)                  # integer data: exact ties between shards occur
    xb[600:620] = xb[100:120]                            # duplicates across the shard boundary
    xq = datagen.sift_like(10**6, nq, d=32)
    first, n = mr.shard_range(rank, world_size, nb)

    def local():
        d, i = oracle.flat_l2_knn(xq, xb[first:first + n], k)
        return torch.from_numpy(d), torch.from_numpy(i)

    def merge(dg, ig):
        d, i = oracle.merge_topk(dg.numpy(), ig.numpy(), k)
        return torch.from_numpy(d), torch.from_numpy(i)

    md, mi = mr.sharded_search(local, merge, first)
    wd, wi = oracle.flat_l2_knn(xq, xb, k)
    ok = bool(np.array_equal(mi.numpy(), wi) and np.array_equal(md.numpy(), wd))
    # k larger than a shard: padding inside the partial lists must not reach the result
    def local_big():
        d, i = oracle.flat_l2_knn(xq, xb[first:first + 5], 8)
        return torch.from_numpy(d), torch.from_numpy(i)

    def merge_big(dg, ig):
        d, i = oracle.merge_topk(dg.numpy(), ig.numpy(), 8)
        return torch.from_numpy(d), torch.from_numpy(i)

    bd, bi = mr.sharded_search(local_big, merge_big, first)
    sub = np.concatenate([xb[s:s + 5] for s in (mr.shard_range(r, world_size, nb)[0] for r in range(world_size))])
    sub_ids = np.concatenate([np.arange(s, s + 5) for s in (mr.shard_range(r, world_size, nb)[0] for r in range(world_size))])
    wd2, wi2 = oracle.flat_l2_knn(xq, sub, 8)
    ok2 = bool(np.array_equal(bi.numpy(), sub_ids[wi2]) and np.array_equal(bd.numpy(), wd2))
    if rank == 0:
        out.put((ok, ok2, mr.shard_range(0, 2, nb), mr.shard_range(1, 2, nb)))
    dist.destroy_process_group()


def test_sharded_search_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(180)
        assert p.exitcode == 0
    ok, ok2, r0, r1 = out.get()
    assert ok, "sharded oracle search + merge differs from the unsharded oracle"
    assert ok2, "padding leaked through the merge"
    assert r0 == (0, 501) and r1 == (501, 500)


def test_oracle_merge_topk_pins():
    """oracle.merge_topk against its definition on hand-made lists: ties by lower id across shards,
    padding ignored, fewer than k candidates padded."""
    import numpy as np
    import oracle
    d = np.array([[[1.0, 2.0, 2.0], [0.5, 2.0, np.inf]]], np.float32)
    i = np.array([[[7, 3, 9], [40, 1, -1]]], np.int64)
    od, oi = oracle.merge_topk(d, i, 4)
    assert oi.tolist() == [[40, 7, 1, 3]] and od.tolist() == [[0.5, 1.0, 2.0, 2.0]]
    od, oi = oracle.merge_topk(d, i, 6)
    assert oi.tolist() == [[40, 7, 1, 3, 9, -1]] and np.isposinf(od[0, 5])
    # the union's k smallest == k smallest of the concatenation (random, with many ties)
    rng = np.random.default_rng(0)
    for _ in range(20):
        G, kk, k = int(rng.integers(1, 5)), int(rng.integers(1, 9)), int(rng.integers(1, 9))
        dd = rng.integers(0, 4, size=(3, G, kk)).astype(np.float32)
        ii = rng.permutation(3 * G * kk).reshape(3, G, kk).astype(np.int64)
        od, oi = oracle.merge_topk(dd, ii, k)
        for q in range(3):
            pairs = sorted(zip(dd[q].ravel().tolist(), ii[q].ravel().tolist()))[:k]
            assert [p[1] for p in pairs] == oi[q, :len(pairs)].tolist()
