"""CPU oracle for the hot path of arXiv 1702.08734 -- TEST INFRASTRUCTURE.

Thin numpy/ctypes front for ``oracle.cpp`` (plain C++, double precision, full
sorts).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the
product package ``paper_1702_08734_b200`` never does, and nothing here imports
it.  Each function cites the passage of PAPER.md (``P:L<line>``) it follows;
see the header of ``oracle.cpp`` for the list.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle.cpp with g++ -O3 -fopenmp (OpenMP over rows/queries only).

    No -march=native: the library built on the build box travels to the GPU box with the
    snapshot, whose host CPU may differ; -ffp-contract=off keeps the double arithmetic as
    written (no fused multiply-adds).  These are the flags the reported CPU baseline uses.
    """
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        cmd = ["g++", "-O3", "-std=c++17", "-fopenmp", "-fPIC", "-shared",
               "-ffp-contract=off", "-o", tmp, _SRC]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.orc_num_threads.restype = ctypes.c_int
        _lib.orc_successive_mink_count.restype = ctypes.c_int64
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


_i64 = ctypes.c_int64


def kselect(rows: np.ndarray, k: int, n: int | None = None, largest: bool = False):
    """k lowest values of each row with indices, ties by lower index
    (``largest``: the k highest, descending, ties by lower index -- "other comparators").

    rows: [n_rows, ld] fp32; only the first ``n`` (default ld) columns belong to
    the arrays.  Returns (values fp32 [n_rows,k], indices int32 [n_rows,k]).
    """
    rows = _f32(rows)
    assert rows.ndim == 2
    n_rows, ld = rows.shape
    n = ld if n is None else n
    val = np.empty((n_rows, k), np.float32)
    idx = np.empty((n_rows, k), np.int32)
    fn = lib().orc_kselect_largest if largest else lib().orc_kselect
    fn(_p(rows), _i64(n_rows), _i64(n), _i64(ld), _i64(k), _p(val), _p(idx))
    return val, idx


def flat_l2_knn(xq: np.ndarray, xb: np.ndarray, k: int, want64: bool = False):
    """Eq. (1), squared: exact k-NN, direct-difference double."""
    xq, xb = _f32(xq), _f32(xb)
    nq, d = xq.shape
    nb = xb.shape[0]
    assert xb.shape[1] == d
    dist = np.empty((nq, k), np.float32)
    dist64 = np.empty((nq, k), np.float64)
    ids = np.empty((nq, k), np.int64)
    lib().orc_flat_l2_knn(_p(xq), _i64(nq), _p(xb), _i64(nb), _i64(d), _i64(k),
                          _p(dist), _p(dist64), _p(ids))
    return (dist, ids, dist64) if want64 else (dist, ids)


def pair_l2(xq: np.ndarray, xb: np.ndarray, ids: np.ndarray) -> np.ndarray:
    """||xq_j - xb_{ids[j,t]}||^2 in double for given pairs."""
    xq, xb = _f32(xq), _f32(xb)
    ids = np.ascontiguousarray(ids, dtype=np.int64)
    nq, d = xq.shape
    m = ids.shape[1]
    out = np.empty((nq, m), np.float64)
    lib().orc_pair_l2(_p(xq), _i64(nq), _p(xb), _i64(d), _p(ids), _i64(m), _p(out))
    return out


def ivfpq_encode(coarse: np.ndarray, pq: np.ndarray, y: np.ndarray, margins: bool = False):
    """Eq. (3) P:L61, P:L86-90 -- (list number, M-byte code) of each vector.

    coarse [nlist,d]; pq [M,256,dsub].  With ``margins`` also returns the
    relative best/second-best gaps (coarse [n], codes [n,M]).
    """
    coarse, pq, y = _f32(coarse), _f32(pq), _f32(y)
    nlist, d = coarse.shape
    M = pq.shape[0]
    assert pq.shape == (M, 256, d // M) and d % M == 0
    n = y.shape[0]
    lst = np.empty(n, np.int32)
    codes = np.empty((n, M), np.uint8)
    cm = np.empty(n, np.float64) if margins else None
    km = np.empty((n, M), np.float64) if margins else None
    lib().orc_ivfpq_encode(_p(coarse), _p(pq), _i64(d), _i64(nlist), _i64(M), _p(y), _i64(n),
                           _p(lst), _p(codes), _p(cm), _p(km))
    return (lst, codes, cm, km) if margins else (lst, codes)


def build_lists(list_no: np.ndarray, codes: np.ndarray, ids: np.ndarray, nlist: int):
    """group (code, id) by list, append order = input order.

    Returns CSR (offsets int64 [nlist+1], codes [n,M], ids [n]).
    """
    order = np.argsort(list_no, kind="stable")
    counts = np.bincount(list_no, minlength=nlist)
    offsets = np.zeros(nlist + 1, np.int64)
    np.cumsum(counts, out=offsets[1:])
    return offsets, np.ascontiguousarray(codes[order]), np.ascontiguousarray(ids[order].astype(np.int64))


def ivfpq_search(coarse, pq, offsets, codes, ids, xq, nprobe: int, k: int, probed_in=None):
    """Alg. 4 P:L327-353 with Eq. (5)-(7): distances by explicit reconstruction.

    Returns dict(dist fp32, dist64, ids int64, probed int32, coarse64).
    """
    coarse, pq, xq = _f32(coarse), _f32(pq), _f32(xq)
    nlist, d = coarse.shape
    M = pq.shape[0]
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    ids = np.ascontiguousarray(ids, dtype=np.int64)
    nq = xq.shape[0]
    dist = np.empty((nq, k), np.float32)
    dist64 = np.empty((nq, k), np.float64)
    oid = np.empty((nq, k), np.int64)
    probed = np.empty((nq, nprobe), np.int32)
    coarse64 = np.full((nq, nprobe), np.nan, np.float64)
    pin = None if probed_in is None else np.ascontiguousarray(probed_in, dtype=np.int32)
    lib().orc_ivfpq_search(_p(coarse), _p(pq), _i64(d), _i64(nlist), _i64(M), _p(offsets),
                           _p(codes), _p(ids), _p(xq), _i64(nq), _i64(nprobe), _i64(k), _p(pin),
                           _p(dist), _p(dist64), _p(oid), _p(probed), _p(coarse64))
    return dict(dist=dist, dist64=dist64, ids=oid, probed=probed, coarse64=coarse64)


def adc_reconstruct(coarse, pq, x, list_no, codes) -> np.ndarray:
    """Eq. (7) P:L276 for n (query, list, code) triples; x [n,d]."""
    coarse, pq, x = _f32(coarse), _f32(pq), _f32(x)
    d = coarse.shape[1]
    M = pq.shape[0]
    list_no = np.ascontiguousarray(list_no, dtype=np.int32)
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    n = x.shape[0]
    out = np.empty(n, np.float64)
    lib().orc_adc_reconstruct(_p(coarse), _p(pq), _i64(d), _i64(M), _p(x), _p(list_no), _p(codes),
                              _i64(n), _p(out))
    return out


def adc_lut_sum(coarse, pq, x, list_no: int, codes, want_tables: bool = False):
    """Eq. (10) P:L288-290 -- the ADC distance as a sum of M table look-ups."""
    coarse, pq, x = _f32(coarse), _f32(pq), _f32(x)
    d = coarse.shape[1]
    M = pq.shape[0]
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    n = codes.shape[0]
    out = np.empty(n, np.float64)
    tables = np.empty((M, 256), np.float64)
    lib().orc_adc_lut_sum(_p(coarse), _p(pq), _i64(d), _i64(M), _p(x), _i64(list_no), _p(codes),
                          _i64(n), _p(out), _p(tables))
    return (out, tables) if want_tables else out


def adc_eq11(coarse, pq, x, list_no: int, codes) -> np.ndarray:
    """Eq. (11) P:L302 -- term1 + term2 - 2 term3."""
    coarse, pq, x = _f32(coarse), _f32(pq), _f32(x)
    d = coarse.shape[1]
    M = pq.shape[0]
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    n = codes.shape[0]
    out = np.empty(n, np.float64)
    lib().orc_adc_eq11(_p(coarse), _p(pq), _i64(d), _i64(M), _p(x), _i64(list_no), _p(codes),
                       _i64(n), _p(out))
    return out


def successive_mink_count(a: np.ndarray, k: int) -> int:
    """Appendix Eq. (13), P:L575-577 -- elements in the min-k of their prefix."""
    a = _f32(a)
    return int(lib().orc_successive_mink_count(_p(a), _i64(a.shape[0]), _i64(k)))


def kmeans_step(x: np.ndarray, centroids: np.ndarray, seed: int = 0, it: int = 0, margins: bool = False):
    """one Lloyd iteration: assignment to the nearest centroid (double, ties to the lower
    centroid), means in double; an empty cluster takes the hashed point of fs_kmeans's stated rule.
    Returns (centroids fp32 [K, d], assignment int64 [n]) (+ best/second-best margins [n])."""
    x, centroids = _f32(x), _f32(centroids)
    n, d = x.shape
    K = centroids.shape[0]
    out = np.empty((K, d), np.float32)
    assign = np.empty(n, np.int64)
    mg = np.empty(n, np.float64) if margins else None
    lib().orc_kmeans_step(_p(x), _i64(n), _i64(d), _p(centroids), _i64(K), ctypes.c_uint64(seed), _i64(it),
                          _p(out), _p(assign), _p(mg))
    return (out, assign, mg) if margins else (out, assign)


def merge_topk(dist: np.ndarray, ids: np.ndarray, k: int):
    """join of G partial k-NN lists per query by one more k-selection: the k smallest
    (distance, id) pairs of the union, ascending, ties by lower id; ids < 0 are padding.
    dist [nq, G, kk] (any float), ids [nq, G, kk] -> (dist [nq, k] same dtype, ids int64 [nq, k])."""
    dist = np.asarray(dist)
    ids = np.asarray(ids, dtype=np.int64)
    nq = dist.shape[0]
    d2 = dist.reshape(nq, -1)
    i2 = ids.reshape(nq, -1)
    od = np.full((nq, k), np.inf, dist.dtype)
    oi = np.full((nq, k), -1, np.int64)
    for q in range(nq):
        keep = i2[q] >= 0
        dq, iq = d2[q][keep], i2[q][keep]
        order = np.lexsort((iq, dq))[:k]      # by distance, then id
        od[q, :len(order)] = dq[order]
        oi[q, :len(order)] = iq[order]
    return od, oi
