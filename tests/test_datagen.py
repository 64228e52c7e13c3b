"""The torch twin of the seeded generators (datagen/gen_torch.py, used to fill HBM
directly for the big configs) is bit-identical to the numpy version."""
import numpy as np
import pytest
import torch

import datagen
from datagen import gen_torch as gt


def same(a, b):
    return np.array_equal(a.view(np.uint32), b.cpu().numpy().view(np.uint32))


@pytest.mark.parametrize("device", ["cpu", pytest.param("cuda", marks=pytest.mark.gpu)])
def test_twins_bit_identical(device):
    assert same(datagen.gaussian_vectors(5, 300, 64), gt.gaussian_vectors(5, 300, 64, device=device))
    dup, pat = datagen.kselect_dup_rows(700, 100)
    assert set(pat[dup].tolist()) == {0, 1}  # both duplicate patterns are exercised
    assert same(datagen.kselect_rows(700, 100, 1000), gt.kselect_rows(700, 100, 1000, device=device))
    assert same(datagen.sift_like(999_990, 500), gt.sift_like(999_990, 500, device=device))
    assert same(datagen.deep_like(10**8 - 3, 400), gt.deep_like(10**8 - 3, 400, device=device))
    assert same(datagen.deep_like(7, 100, cfg=5), gt.deep_like(7, 100, cfg=5, device=device))


def test_distributions():
    g = datagen.gaussian_vectors(0, 4000, 64)
    assert abs(g.mean()) < 0.01 and abs(g.std() - 1) < 0.01
    u = datagen.kselect_rows(0, 50, 4096, duplicates=False)
    assert 0 <= u.min() and u.max() < 1 and abs(u.mean() - 0.5) < 0.01
    s = datagen.sift_like(0, 500)
    assert s.min() >= 0 and s.max() <= 255 and np.array_equal(s, np.rint(s))
    d = datagen.deep_like(0, 500)
    assert np.allclose((d.astype(np.float64) ** 2).sum(1), 1.0, atol=1e-6)
