"""Pins for the k-selection oracle (oracle.kselect).

Each pin is something other than the oracle's own formula: a hand-worked
example, closed forms, brute force through independent library routines,
invariants, and the Appendix's expectation.
"""
import numpy as np
import pytest

import oracle
from golden_io import load


def test_handworked_example():
    g = load("kselect_handworked.txt")
    row = g["row"].astype(np.float32)[None, :]
    v, i = oracle.kselect(row, 4)
    assert v[0].tolist() == g["k4_val"].tolist() and i[0].tolist() == g["k4_idx"].tolist()
    v, i = oracle.kselect(row, 5)
    assert v[0].tolist() == g["k5_val"].tolist() and i[0].tolist() == g["k5_idx"].tolist()
    v, i = oracle.kselect(row, 8)
    assert i[0].tolist() == g["k8_idx"].tolist()


@pytest.mark.parametrize("n,k", [(1, 1), (7, 3), (64, 64), (100, 32), (1000, 128)])
def test_closed_forms(n, k):
    asc = np.arange(n, dtype=np.float32)[None, :]
    v, i = oracle.kselect(asc, k)
    assert i[0].tolist() == list(range(k)) and v[0].tolist() == list(range(k))
    desc = asc[:, ::-1].copy()
    v, i = oracle.kselect(desc, k)
    assert i[0].tolist() == [n - 1 - t for t in range(k)] and v[0].tolist() == list(range(k))
    const = np.full((1, n), 3.5, np.float32)
    v, i = oracle.kselect(const, k)
    assert i[0].tolist() == list(range(k)) and np.all(v == 3.5)
    rng = np.random.default_rng(n * 131 + k)
    perm = rng.permutation(n)
    v, i = oracle.kselect(perm.astype(np.float32)[None, :], k)
    inv = np.argsort(perm)
    assert v[0].tolist() == list(range(k)) and i[0].tolist() == inv[:k].tolist()


def test_bruteforce_two_independent_routines():
    """Full sort (oracle) vs numpy lexsort and vs argpartition + sort of the head."""
    rng = np.random.default_rng(7)
    for n in (1, 2, 5, 17, 33, 64):
        rows = rng.integers(0, 6, size=(20, n)).astype(np.float32) / 4.0  # many ties
        for k in range(1, n + 1):
            v, i = oracle.kselect(rows, k)
            for r in range(rows.shape[0]):
                order = np.lexsort((np.arange(n), rows[r]))  # value, then index
                assert i[r].tolist() == order[:k].tolist()
                assert v[r].tolist() == rows[r][order[:k]].tolist()
                # second routine: kth value by partition, then count
                kth = np.partition(rows[r], k - 1)[k - 1]
                assert v[r, -1] == kth
                assert np.sum(rows[r] < kth) <= k - 1 < np.sum(rows[r] <= kth)


def check_invariants(rows, n, k, val, idx):
    """Valid for any k-selection output (also used by the GPU parity tests)."""
    for r in range(rows.shape[0]):
        a = rows[r, :n]
        kk = min(k, n)
        ii, vv = idx[r, :kk], val[r, :kk]
        assert np.array_equal(vv.view(np.uint32), a[ii].view(np.uint32))  # original bits
        for t in range(kk - 1):  # strictly increasing (value, index)
            assert vv[t] < vv[t + 1] or (vv[t] == vv[t + 1] and ii[t] < ii[t + 1])
        mask = np.ones(n, bool)
        mask[ii] = False
        if mask.any() and kk:
            rest = a[mask]
            assert rest.min() >= vv[-1]
            tied = np.nonzero(mask & (a == vv[-1]))[0]
            assert tied.size == 0 or tied.min() > ii[vv == vv[-1]].max()
        assert np.all(idx[r, kk:] == -1) and np.all(np.isposinf(val[r, kk:]))


def test_invariants_random_and_padding():
    rng = np.random.default_rng(3)
    rows = rng.random((8, 300), dtype=np.float32)
    rows[3] = np.floor(rows[3] * 8) / 8
    for n, k in [(300, 1), (300, 37), (257, 128), (10, 32)]:
        v, i = oracle.kselect(rows, k, n=n)
        check_invariants(rows, n, k, v, i)


def test_special_values():
    row = np.array([[0.0, -0.0, np.inf, -np.inf, np.nan, 1.0, -0.0, np.inf]], np.float32)
    v, i = oracle.kselect(row, 8)
    # -inf, then the three zeros in index order (-0 == +0), 1, the infs in index order, NaN last
    assert i[0].tolist() == [3, 0, 1, 6, 5, 2, 7, 4]
    assert np.signbit(v[0, 2]) and not np.signbit(v[0, 1])  # original bits kept
    assert np.isnan(v[0, 7])


def test_expected_successive_mink_count():
    """Appendix: on a random permutation the number of elements that are in the
    min-k of their prefix averages k + k (H_l - H_k), H_l for k=1."""
    rng = np.random.default_rng(11)
    n = 4096
    H = np.cumsum(1.0 / np.arange(1, n + 1))
    for k in (1, 32):
        trials = 400
        tot = sum(oracle.successive_mink_count(rng.permutation(n).astype(np.float32), k)
                  for _ in range(trials))
        expect = k + k * (H[n - 1] - H[k - 1])
        assert abs(tot / trials - expect) < 0.05 * expect


def test_survey_derived_counts():
    """k + k(H_l - H_k) at l=16384 is 10.3 / 231 / 749 / 3863."""
    H = np.cumsum(1.0 / np.arange(1, 16385))
    got = [k + k * (H[-1] - H[k - 1]) for k in (1, 32, 128, 1024)]
    assert [round(x) for x in got] == [10, 231, 749, 3863]


def test_largest_handworked_and_bruteforce():
    """The k-largest variant ("other comparators"): hand-worked example, numpy's stable sort of the
    negated row, special values (NaN last, -0 == +0, ties to the lower index), padding (-inf, -1)."""
    g = load("kselect_handworked.txt")
    row = g["row"].astype(np.float32)[None, :]
    v, i = oracle.kselect(row, 3, largest=True)
    assert v[0].tolist() == g["top3_val"].tolist() and i[0].tolist() == g["top3_idx"].tolist()
    v, i = oracle.kselect(row, 8, largest=True)
    assert i[0].tolist() == g["top8_idx"].tolist()
    rng = np.random.default_rng(19)
    for n in (1, 3, 17, 64, 200):
        rows = rng.integers(-5, 6, size=(10, n)).astype(np.float32) / 4.0
        for k in sorted({1, min(2, n), n // 2 + 1, n}):
            v, i = oracle.kselect(rows, k, largest=True)
            for r in range(rows.shape[0]):
                order = np.argsort(-rows[r], kind="stable")  # descending value, ties by lower index
                assert i[r].tolist() == order[:k].tolist()
                assert v[r].tolist() == rows[r][order[:k]].tolist()
    row = np.array([[0.0, -0.0, np.inf, -np.inf, np.nan, 1.0, -0.0, np.inf]], np.float32)
    v, i = oracle.kselect(row, 8, largest=True)
    assert i[0].tolist() == [2, 7, 5, 0, 1, 6, 3, 4]
    assert np.isnan(v[0, 7]) and np.signbit(v[0, 4]) and not np.signbit(v[0, 3])
    v, i = oracle.kselect(np.array([[2.0, 3.0]], np.float32), 4, largest=True)
    assert i[0].tolist() == [1, 0, -1, -1] and np.all(np.isneginf(v[0, 2:]))
    # smallest of the negated row selects the same indices
    rows = rng.standard_normal((4, 500)).astype(np.float32)
    _, a = oracle.kselect(rows, 40, largest=True)
    _, b = oracle.kselect(-rows, 40)
    assert np.array_equal(a, b)
