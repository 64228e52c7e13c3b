"""Seeded synthetic inputs shaped like the paper's workloads (numpy side).

A counter-based, integer-only generator: every element of every tensor is a
pure function of (seed, stream, i, j), so any single vector of a 10^9-vector
set can be regenerated anywhere.  ``gen_cuda.cu`` is its CUDA twin (used to
fill device memory for the big configs); the two are bit-identical by
construction (integer hashing, then a fixed sequence of correctly-rounded
fp32/fp64 operations with no fused multiply-add) and a GPU test compares them.

This module holds NONE of the method's arithmetic (no distances, no selection,
no quantisation); it serves both the oracle and the CUDA path, which is the
only thing they share.  The datasets the paper measures on (SIFT1M/1B, DEEP1B,
YFCC100M) are not available; these inputs stand in
for them.

Streams: 10*cfg + {0: database/rows, 1: (unused: queries are database indices
>= nb), 2: mixture means, 3: component choice, 4: training-sample ids,
5: duplicate-row pattern, 6: oracle query-subset choice, 7: add-check ids}.
"""
from __future__ import annotations

import numpy as np

U64 = np.uint64
_GOLD = U64(0x9E3779B97F4A7C15)
_M1 = U64(0xBF58476D1CE4E5B9)
_M2 = U64(0x94D049BB133111EB)
# float32 nearest to 1 / sqrt(8 * (65536^2 - 1) / 12): unit variance for the sum
# of eight 16-bit fields.
NORMAL_SCALE = np.float32(1.0 / np.sqrt(8.0 * (65536.0 ** 2 - 1.0) / 12.0))
NORMAL_SCALE_HEX = 0x379CC471  # asserted below; the CUDA twin hard-codes it
assert np.float32(NORMAL_SCALE).view(np.uint32) == NORMAL_SCALE_HEX, hex(
    int(np.float32(NORMAL_SCALE).view(np.uint32)))


def mix64(z):
    """splitmix64 finaliser on uint64 arrays (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        z = np.asarray(z, dtype=U64)
        z = (z ^ (z >> U64(30))) * _M1
        z = (z ^ (z >> U64(27))) * _M2
        return z ^ (z >> U64(31))


def h(seed: int, stream: int, i, j):
    """h(seed, stream, i, j) -> uint64; i, j broadcastable uint64 arrays."""
    with np.errstate(over="ignore"):
        a = mix64(U64(seed) * _GOLD + U64(stream))
        b = mix64(a + np.asarray(i, dtype=U64))
        return mix64(b + np.asarray(j, dtype=U64))


def uniform(seed, stream, i, j):
    """U[0,1) with 24 bits: top 24 bits of h times 2^-24 (exact in fp32)."""
    return (h(seed, stream, i, j) >> U64(40)).astype(np.float32) * np.float32(2.0 ** -24)


def normal(seed, stream, i, j):
    """Approximate N(0,1): (sum of eight 16-bit fields - 262140) * NORMAL_SCALE.

    Irwin-Hall with 8 terms, |g| <= 4.9, unit variance; the integer sum is exact
    and the single fp32 multiply is correctly rounded, so CPU == GPU bit for bit.
    """
    j = np.asarray(j, dtype=U64)
    a = h(seed, stream, i, j * U64(2))
    b = h(seed, stream, i, j * U64(2) + U64(1))
    s = np.zeros(np.broadcast(a, b).shape, dtype=np.int64)
    for w in (a, b):
        for sh in (0, 16, 32, 48):
            s += ((w >> U64(sh)) & U64(0xFFFF)).astype(np.int64)
    return (s - 262140).astype(np.float32) * NORMAL_SCALE


def _grid(i0: int, n: int, d: int):
    i = (np.arange(n, dtype=U64) + U64(i0))[:, None]
    j = np.arange(d, dtype=U64)[None, :]
    return i, j


# --------------------------------------------------------------------------
# cfg1: i.i.d. ~N(0,1) vectors (BASELINE.json configs[0])
# --------------------------------------------------------------------------
def gaussian_vectors(i0: int, n: int, d: int, seed: int = 0, cfg: int = 1) -> np.ndarray:
    i, j = _grid(i0, n, d)
    return normal(seed, 10 * cfg + 0, i, j)


# --------------------------------------------------------------------------
# cfg2: rows of U[0,1) with ~1% duplicate-heavy rows (BASELINE.json configs[1])
# --------------------------------------------------------------------------
def kselect_rows(r0: int, n_rows: int, n: int, seed: int = 0, cfg: int = 2,
                 duplicates: bool = True) -> np.ndarray:
    """Rows r0..r0+n_rows-1.  Row r with h(seed,5,r,0) % 100 == 0 is rewritten
    with duplicated runs, two patterns chosen by bit 32 of the same hash:
    quantised (floor(64u)/64) or contiguous runs (a_i = a_{i - i%64})."""
    out = np.empty((n_rows, n), np.float32)
    step = max(1, (1 << 22) // max(n, 1))
    for s in range(0, n_rows, step):
        e = min(n_rows, s + step)
        i, j = _grid(r0 + s, e - s, n)
        out[s:e] = uniform(seed, 10 * cfg + 0, i, j)
    if duplicates:
        r = np.arange(n_rows, dtype=U64) + U64(r0)
        hr = h(seed, 10 * cfg + 5, r, U64(0))
        dup = (hr % U64(100)) == U64(0)
        pat = ((hr >> U64(32)) & U64(1)).astype(np.int64)
        for rr in np.nonzero(dup)[0]:
            if pat[rr] == 0:
                out[rr] = np.floor(out[rr] * np.float32(64.0)) * np.float32(1.0 / 64.0)
            else:
                idx = np.arange(n)
                out[rr] = out[rr][idx - (idx % 64)]
    return out


def kselect_dup_rows(r0: int, n_rows: int, seed: int = 0, cfg: int = 2):
    """(is_duplicate_row bool[n_rows], pattern int[n_rows]) for rows r0.."""
    r = np.arange(n_rows, dtype=U64) + U64(r0)
    hr = h(seed, 10 * cfg + 5, r, U64(0))
    return (hr % U64(100)) == U64(0), ((hr >> U64(32)) & U64(1)).astype(np.int64)


# --------------------------------------------------------------------------
# cfg3: SIFT-like descriptors: 256-component mixture, integers in [0,255]
# --------------------------------------------------------------------------
def sift_like(i0: int, n: int, d: int = 128, seed: int = 0, cfg: int = 3,
              ncomp: int = 256) -> np.ndarray:
    """x = rint(clip(mu_c + 25 g, 0, 255)), mu_c[j] = 10 + 60 max(0, g'), c = h % ncomp.
    Every fp32 operation is a separate correctly-rounded multiply or add."""
    i, j = _grid(i0, n, d)
    comp = (h(seed, 10 * cfg + 3, i, U64(0)) % U64(ncomp)).astype(U64)
    gm = normal(seed, 10 * cfg + 2, comp, j)
    mu = np.float32(10.0) + np.float32(60.0) * np.maximum(np.float32(0.0), gm)
    x = mu + np.float32(25.0) * normal(seed, 10 * cfg + 0, i, j)
    return np.rint(np.clip(x, np.float32(0.0), np.float32(255.0))).astype(np.float32)


# --------------------------------------------------------------------------
# cfg4/5: deep-feature-like: 4096-component mixture, skewed weights, unit norm
# --------------------------------------------------------------------------
def deep_like(i0: int, n: int, d: int = 96, seed: int = 0, cfg: int = 4,
              ncomp: int = 4096, ids=None) -> np.ndarray:
    """c = floor(ncomp * u^1.5) (u*sqrt(u) in double), x = mu_c + 0.35 g, then
    L2-normalised: squared norm accumulated in double in dimension order, one
    double sqrt, one double divide per element, rounded to fp32.
    With ``ids`` (int array) the vectors with exactly those indices are generated
    (i0 and n are ignored): any vector of a 10^9-vector set can be regenerated."""
    if ids is not None:
        ids = np.asarray(ids, dtype=np.int64)
        n = len(ids)
    out = np.empty((n, d), np.float32)
    step = max(1, (1 << 20) // d)
    for s in range(0, n, step):
        e = min(n, s + step)
        i, j = _grid(i0 + s, e - s, d)
        if ids is not None:
            i = ids[s:e].astype(U64)[:, None]
        u = uniform(seed, 10 * cfg + 3, i, U64(0)).astype(np.float64)
        comp = np.minimum(np.floor(np.float64(ncomp) * (u * np.sqrt(u))), ncomp - 1).astype(U64)
        mu = normal(seed, 10 * cfg + 2, comp, j)
        x = mu + np.float32(0.35) * normal(seed, 10 * cfg + 0, i, j)
        xd = x.astype(np.float64)
        acc = np.zeros(e - s, np.float64)
        for c in range(d):  # sequential, as the CUDA twin does
            acc = acc + xd[:, c] * xd[:, c]
        nrm = np.sqrt(acc)
        out[s:e] = (xd / nrm[:, None]).astype(np.float32)
    return out


def sample_ids(count: int, modulo: int, seed: int = 0, stream: int = 44) -> np.ndarray:
    """ids h(seed, stream, s, 0) % modulo, s = 0..count-1 (training / check samples)."""
    s = np.arange(count, dtype=U64)
    return (h(seed, stream, s, U64(0)) % U64(modulo)).astype(np.int64)


def gather(fn, ids: np.ndarray, **kw) -> np.ndarray:
    """Regenerate the vectors with the given ids using generator ``fn``."""
    ids = np.asarray(ids, dtype=np.int64)
    out = None
    for t, i in enumerate(ids):
        v = fn(int(i), 1, **kw)
        if out is None:
            out = np.empty((len(ids), v.shape[1]), np.float32)
        out[t] = v[0]
    return out


# --------------------------------------------------------------------------
# Shapes of BASELINE.json configs[3] / configs[4] (cfg4 / cfg5): sizes only, shared by
# tests/ and bench.py so that both build the same index.  ntrain for cfg5 is not fixed by
# BASELINE.json (SURVEY 8d proposes 16 per centroid).  check_queries = the size of the
# seeded oracle query subset, add_check = how many seeded ids the add path is re-encoded for.
# --------------------------------------------------------------------------
IVFPQ_CONFIGS = {
    4: dict(nb=100_000_000, d=96, nlist=65_536, M=16, ntrain=1_000_000, nq=10_000,
            searches=((16, 100), (64, 100), (256, 100)), check_queries=500, add_check=10_000),
    5: dict(nb=1_000_000_000, d=96, nlist=262_144, M=8, ntrain=4_194_304, nq=10_000,
            searches=((32, 1), (32, 100), (128, 1), (128, 100)), check_queries=200, add_check=10_000),
}


def unique_sample_ids(count: int, modulo: int, seed: int = 0, stream: int = 46) -> np.ndarray:
    """`count` distinct ids in [0, modulo), ascending: the first distinct values of the
    seeded sequence h(seed, stream, s, 0) % modulo (streams 10*cfg + 6 / + 7 of the header)."""
    assert count <= modulo
    got = np.empty(0, np.int64)
    s0 = 0
    while len(got) < count:
        s = np.arange(s0, s0 + 2 * count, dtype=U64)
        got = np.unique(np.concatenate([got, (h(seed, stream, s, U64(0)) % U64(modulo)).astype(np.int64)]))
        s0 += 2 * count
    rng_order = np.argsort(h(seed, stream + 1000, got.astype(U64), U64(0)), kind="stable")
    return np.sort(got[rng_order[:count]])
