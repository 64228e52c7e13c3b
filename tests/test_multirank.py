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
