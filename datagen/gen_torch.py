"""Device twin of gen.py: the same counter-based generator written with torch
integer/float ops, so the big configs can be filled directly in HBM.

Bit-identical to the numpy version by construction: the hash is wrapping 64-bit
integer arithmetic (int64 two's complement == uint64 modulo 2^64; logical right
shifts are emulated by masking), and every floating-point step is a separate
correctly-rounded IEEE operation in the same order (no fused multiply-add: each
torch op is its own kernel).  tests/test_gpu_datagen.py compares the two.

Holds none of the method's arithmetic (see gen.py).
"""
from __future__ import annotations

import numpy as np
import torch

from . import gen as _np

_MASK64 = (1 << 64) - 1
_GOLD = 0x9E3779B97F4A7C15
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB


def _s64(v: int) -> int:
    """Python int (mod 2^64) -> the int64 with the same bits."""
    v &= _MASK64
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical right shift of int64 bit patterns."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def _mix64_t(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _s64(_M1)
    z = (z ^ _lsr(z, 27)) * _s64(_M2)
    return z ^ _lsr(z, 31)


def _mix64_i(z: int) -> int:
    z &= _MASK64
    z = ((z ^ (z >> 30)) * _M1) & _MASK64
    z = ((z ^ (z >> 27)) * _M2) & _MASK64
    return z ^ (z >> 31)


def h(seed: int, stream: int, i: torch.Tensor, j) -> torch.Tensor:
    """h(seed, stream, i, j) as int64 bit patterns; i int64 tensor, j tensor or int."""
    a = _mix64_i(seed * _GOLD + stream)
    b = _mix64_t(i + _s64(a))
    return _mix64_t(b + j)


def uniform(seed, stream, i, j) -> torch.Tensor:
    return _lsr(h(seed, stream, i, j), 40).to(torch.float32) * float(2.0 ** -24)


def normal(seed, stream, i, j) -> torch.Tensor:
    a = h(seed, stream, i, j * 2)
    b = h(seed, stream, i, j * 2 + 1)
    s = torch.zeros(torch.broadcast_shapes(a.shape, b.shape), dtype=torch.int64, device=a.device)
    for w in (a, b):
        for sh in (0, 16, 32, 48):
            s += (w >> sh) & 0xFFFF
    scale = torch.tensor(float(_np.NORMAL_SCALE), dtype=torch.float32, device=a.device)
    return (s - 262140).to(torch.float32) * scale


def _umod(hh: torch.Tensor, m: int) -> torch.Tensor:
    """Unsigned 64-bit hh % m for 0 < m < 2^31."""
    return ((_lsr(hh, 1) % m) * 2 + (hh & 1)) % m


def _grid(i0, n, d, device):
    i = (torch.arange(n, dtype=torch.int64, device=device) + i0)[:, None]
    j = torch.arange(d, dtype=torch.int64, device=device)[None, :]
    return i, j


def gaussian_vectors(i0, n, d, seed=0, cfg=1, device="cuda") -> torch.Tensor:
    i, j = _grid(i0, n, d, device)
    return normal(seed, 10 * cfg + 0, i, j)


def kselect_rows(r0, n_rows, n, seed=0, cfg=2, duplicates=True, device="cuda") -> torch.Tensor:
    out = torch.empty((n_rows, n), dtype=torch.float32, device=device)
    step = max(1, (1 << 24) // max(n, 1))
    for s in range(0, n_rows, step):
        e = min(n_rows, s + step)
        i, j = _grid(r0 + s, e - s, n, device)
        out[s:e] = uniform(seed, 10 * cfg + 0, i, j)
    if duplicates:
        dup, pat = _np.kselect_dup_rows(r0, n_rows, seed=seed, cfg=cfg)
        idx = torch.arange(n, device=device)
        src = idx - (idx % 64)
        for rr in np.nonzero(dup)[0]:
            if pat[rr] == 0:
                out[rr] = torch.floor(out[rr] * 64.0) * (1.0 / 64.0)
            else:
                out[rr] = out[rr][src]
    return out


def sift_like(i0, n, d=128, seed=0, cfg=3, ncomp=256, device="cuda") -> torch.Tensor:
    out = torch.empty((n, d), dtype=torch.float32, device=device)
    step = max(1, (1 << 24) // d)
    for s in range(0, n, step):
        e = min(n, s + step)
        i, j = _grid(i0 + s, e - s, d, device)
        comp = _umod(h(seed, 10 * cfg + 3, i, 0), ncomp)
        gm = normal(seed, 10 * cfg + 2, comp, j)
        mu = torch.clamp_min(gm, 0.0) * 60.0 + 10.0
        x = normal(seed, 10 * cfg + 0, i, j) * 25.0 + mu
        out[s:e] = torch.round(torch.clamp(x, 0.0, 255.0))
    return out


def deep_like(i0, n, d=96, seed=0, cfg=4, ncomp=4096, device="cuda") -> torch.Tensor:
    out = torch.empty((n, d), dtype=torch.float32, device=device)
    step = max(1, (1 << 24) // d)
    for s in range(0, n, step):
        e = min(n, s + step)
        i, j = _grid(i0 + s, e - s, d, device)
        u = uniform(seed, 10 * cfg + 3, i, 0).to(torch.float64)
        comp = torch.clamp_max(torch.floor((u * torch.sqrt(u)) * float(ncomp)), ncomp - 1).to(torch.int64)
        mu = normal(seed, 10 * cfg + 2, comp, j)
        x = normal(seed, 10 * cfg + 0, i, j) * 0.35
        x = mu + x
        xd = x.to(torch.float64)
        acc = torch.zeros(e - s, dtype=torch.float64, device=device)
        for c in range(d):
            acc = acc + xd[:, c] * xd[:, c]
        nrm = torch.sqrt(acc)
        out[s:e] = (xd / nrm[:, None]).to(torch.float32)
    return out
