"""GPU parity of the all-vs-all k-NN graph (f4; section 6.5): fs_ivfpq_knn_graph's rows are
fs_ivfpq_search's answers for the stored vectors as queries, batch by batch, so every row must meet the
same predicates against the oracle (tests/test_gpu_ivfpq.verify_search); the batch size must not change
the result beyond what the scan's dispatch allows (near-ties)."""
import numpy as np
import pytest
import torch

import datagen

pytestmark = pytest.mark.gpu


def _index(n, d, M, nlist):
    import paper_1702_08734_b200 as fs
    from datagen import gen_torch as gt
    x = gt.deep_like(0, n, d=d)
    ix = fs.IvfPq(d, nlist, M)
    ix.train(x, niter=6, seed=3)
    ix.add(x[: n // 2])
    ix.add(x[n // 2:])
    return ix, x


@pytest.mark.parametrize("M,k,nprobe,batch", [(16, 10, 4, 1000), (8, 10, 8, 0), (16, 1, 2, 777), (8, 100, 16, 2048)])
def test_graph_rows_meet_the_oracle(M, k, nprobe, batch):
    from test_gpu_ivfpq import verify_search
    n, d, nlist = 6000, 96, 64
    ix, x = _index(n, d, M, nlist)
    gd, gi, gp = ix.knn_graph(x, nprobe, k, batch=batch, want_probed=True)
    torch.cuda.synchronize()
    coarse, pq = (t.cpu().numpy() for t in ix.get_quantizers())
    offs, codes, lids = (t.cpu().numpy() for t in ix.export())
    xs = x.cpu().numpy()
    assert np.array_equal(xs[:3], datagen.deep_like(0, 3, d=d))
    verify_search(coarse, pq, offs, codes, lids, xs, nprobe, k, gd.cpu().numpy(), gi.cpu().numpy(), gp.cpu().numpy())
    # one call per row block == the graph call (same kernels, same batch shapes)
    b = batch if batch else 65536
    sd, si = ix.search(x[:min(b, n)], nprobe, k)
    assert torch.equal(si, gi[:min(b, n)]) and torch.equal(sd, gd[:min(b, n)])
    # the stored vector itself is (nearly always) among its own neighbours: its code is the nearest
    # reproduction value of its own list, which is always probed first
    if k >= 10:
        self_hit = (gi == torch.arange(n, device="cuda")[:, None]).any(1).float().mean().item()
        assert self_hit > 0.95
    ix.close()


def test_graph_batching_and_errors():
    import paper_1702_08734_b200 as fs
    ix, x = _index(5000, 64, 8, 32)
    a = ix.knn_graph(x, 4, 10, batch=512)
    b = ix.knn_graph(x, 4, 10, batch=5000)
    torch.cuda.synchronize()
    assert torch.allclose(a[0], b[0], rtol=1e-5, atol=0)
    assert (a[1] == b[1]).float().mean().item() > 0.995
    e = ix.knn_graph(x[:0], 4, 10)
    assert e[0].shape == (0, 10)
    with pytest.raises(fs.FsError):
        ix.knn_graph(x, 64, 10)          # nprobe > nlist
    with pytest.raises(fs.FsError):
        ix.knn_graph(x, 4, 0)
    ix.close()
