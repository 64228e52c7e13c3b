"""Python binding of libfs.so (include/fs.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; torch is
used for device memory and streams.  There is no CPU fallback: importing works
without the library (so that ``build`` can be imported), but the first call
raises if ``libfs.so`` has not been built.  Nothing here imports ``oracle``.

Names follow the C ABI: ``kselect`` -> ``fs_kselect``, ``flat_l2_knn`` ->
``fs_flat_l2_knn`` (Eq. 1-2), ``IvfPq`` -> ``fs_ivfpq_*`` (Eq. 3-7,
Alg. 4).
"""
from __future__ import annotations

import ctypes
import os
import re

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("FS_LIB_PATH") or os.path.join(_HERE, "libfs.so")  # override: A/B builds
HEADER_PATH = os.path.join(os.path.dirname(_HERE), "include", "fs.h")
_lib = None

FS_OK = 0
FS_MAX_K = 1024

_vp, _i64, _int, _sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_size_t


class FsError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("fs error %d: %s" % (code, msg))
        self.code = code


def declared_symbols() -> list[str]:
    """Function names include/fs.h declares (used by the ABI test)."""
    with open(HEADER_PATH) as f:
        return re.findall(r"^FS_API [^(]*?\b(fs_[a-z0-9_]+)\(", f.read(), flags=re.M)


def lib():
    """Load libfs.so; raise (never fall back) if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FsError(-1, "libfs.so not built: run `python -m paper_1702_08734_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        L.fs_last_error.restype = ctypes.c_char_p
        L.fs_version.restype = ctypes.c_char_p
        L.fs_flat_engine.restype = ctypes.c_char_p
        L.fs_launch_count.restype = _i64
        L.fs_reset_launch_count.restype = None
        for name in ("fs_kselect_ws_bytes", "fs_flat_l2_knn_ws_bytes", "fs_ivfpq_search_ws_bytes",
                     "fs_merge_topk_ws_bytes", "fs_kselect_noalloc_max_scratch", "fs_flat_prepare_bytes"):
            if hasattr(L, name):
                getattr(L, name).restype = _sz
        for name in ("fs_ivfpq_ntotal", "fs_ivfpq_last_scanned_codes"):
            if hasattr(L, name):
                getattr(L, name).restype = _i64
        _lib = L
    return _lib


def _check(rc: int):
    if rc != FS_OK:
        raise FsError(rc, lib().fs_last_error().decode())


def _stream() -> _vp:
    return _vp(torch.cuda.current_stream().cuda_stream)


def _dev(t: torch.Tensor, dtype, name: str) -> torch.Tensor:
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise ValueError("%s must be a contiguous CUDA tensor of %s" % (name, dtype))
    return t


def _ptr(t):
    return _vp(0 if t is None else t.data_ptr())


def flat_engine() -> str:
    return lib().fs_flat_engine().decode()


def launch_count() -> int:
    return int(lib().fs_launch_count())


def reset_launch_count() -> None:
    lib().fs_reset_launch_count()


# ---------------------------------------------------------------------------
def kselect_ws_bytes(n_rows: int, n: int, k: int) -> int:
    return int(lib().fs_kselect_ws_bytes(_i64(n_rows), _i64(n), _int(k)))


def kselect(rows: torch.Tensor, k: int, n: int | None = None, out_val=None, out_idx=None, ws=None,
            largest: bool = False):
    """fs_kselect: k smallest of each row (ascending, ties by lower index); ``largest=True`` calls
    fs_kselect_largest (k largest, descending, ties by lower index).

    rows: CUDA fp32 [n_rows, ld] (row stride ld = rows.stride(0)); n defaults to
    rows.shape[1].  Returns (values fp32 [n_rows,k], indices int32 [n_rows,k]).
    """
    if not (rows.is_cuda and rows.dtype == torch.float32 and rows.dim() == 2
            and (rows.shape[1] == 0 or rows.stride(1) == 1)):
        raise ValueError("rows must be a 2-D CUDA fp32 tensor with unit column stride")
    n_rows = rows.shape[0]
    n = rows.shape[1] if n is None else n
    ld = rows.stride(0) if n_rows > 1 else max(rows.shape[1], n)
    if out_val is None:
        out_val = torch.empty((n_rows, k), dtype=torch.float32, device=rows.device)
    if out_idx is None:
        out_idx = torch.empty((n_rows, k), dtype=torch.int32, device=rows.device)
    _dev(out_val, torch.float32, "out_val")
    _dev(out_idx, torch.int32, "out_idx")
    fn = lib().fs_kselect_largest if largest else lib().fs_kselect
    _check(fn(_ptr(rows), _i64(n_rows), _i64(n), _i64(ld), _int(k), _ptr(out_val),
              _ptr(out_idx), _ptr(ws), _sz(0 if ws is None else ws.numel() * ws.element_size()),
              _stream()))
    return out_val, out_idx


def kselect_noalloc(rows: torch.Tensor, k: int, out_val: torch.Tensor, out_idx: torch.Tensor, n: int | None = None):
    """fs_kselect_noalloc: fs_kselect on the library's built-in scratch array; allocates nothing, so the
    outputs must be given.  Raises FsError (FS_EUNSUPPORTED) when the call needs more scratch than
    kselect_noalloc_max_scratch().  Calls that overlap on the GPU race on the shared array."""
    if not (rows.is_cuda and rows.dtype == torch.float32 and rows.dim() == 2
            and (rows.shape[1] == 0 or rows.stride(1) == 1)):
        raise ValueError("rows must be a 2-D CUDA fp32 tensor with unit column stride")
    n_rows = rows.shape[0]
    n = rows.shape[1] if n is None else n
    ld = rows.stride(0) if n_rows > 1 else max(rows.shape[1], n)
    _dev(out_val, torch.float32, "out_val")
    _dev(out_idx, torch.int32, "out_idx")
    _check(lib().fs_kselect_noalloc(_ptr(rows), _i64(n_rows), _i64(n), _i64(ld), _int(k), _ptr(out_val),
                                    _ptr(out_idx), _stream()))
    return out_val, out_idx


def kselect_noalloc_max_scratch() -> int:
    return int(lib().fs_kselect_noalloc_max_scratch())


def _host_ptr(a, dtype_np, dtype_t, name):
    """Address of a contiguous HOST buffer: numpy array or CPU torch tensor (pinned or not)."""
    import numpy as np
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != dtype_t or not a.is_contiguous():
            raise ValueError("%s must be a contiguous CPU tensor of %s" % (name, dtype_t))
        return a, a.data_ptr()
    a = np.ascontiguousarray(a, dtype=dtype_np)
    return a, a.ctypes.data


def kselect_host(rows, k: int, out_val=None, out_idx=None):
    """fs_kselect_host: same through HOST buffers (numpy or CPU torch fp32 [n_rows, n]);
    the library copies in, runs and copies out.  Outputs are numpy unless given."""
    import numpy as np
    rows, rp = _host_ptr(rows, np.float32, torch.float32, "rows")
    n_rows, n = rows.shape
    val = np.empty((n_rows, k), np.float32) if out_val is None else out_val
    idx = np.empty((n_rows, k), np.int32) if out_idx is None else out_idx
    val, vp = _host_ptr(val, np.float32, torch.float32, "out_val")
    idx, ip = _host_ptr(idx, np.int32, torch.int32, "out_idx")
    _check(lib().fs_kselect_host(_vp(rp), _i64(n_rows), _i64(n), _i64(n), _int(k), _vp(vp), _vp(ip)))
    return val, idx


# ---------------------------------------------------------------------------
def flat_l2_knn_ws_bytes(nq: int, nb: int, d: int, k: int) -> int:
    return int(lib().fs_flat_l2_knn_ws_bytes(_i64(nq), _i64(nb), _int(d), _int(k)))


def flat_l2_knn(xq: torch.Tensor, xb: torch.Tensor, k: int, out_dist=None, out_ids=None, ws=None, prep=None):
    """fs_flat_l2_knn (prep given: fs_flat_l2_knn_prepared, prep from flat_prepare(xb)): exact squared-L2
    k-NN; returns (dist fp32 [nq,k], ids int64 [nq,k])."""
    _dev(xq, torch.float32, "xq")
    _dev(xb, torch.float32, "xb")
    nq, d = xq.shape
    nb = xb.shape[0]
    if xb.dim() != 2 or (nb and xb.shape[1] != d):
        raise ValueError("xb must be [nb, d]")
    if out_dist is None:
        out_dist = torch.empty((nq, k), dtype=torch.float32, device=xq.device)
    if out_ids is None:
        out_ids = torch.empty((nq, k), dtype=torch.int64, device=xq.device)
    wsz = _sz(0 if ws is None else ws.numel() * ws.element_size())
    if prep is not None:
        _check(lib().fs_flat_l2_knn_prepared(_ptr(xq), _i64(nq), _ptr(xb), _ptr(prep),
                                             _sz(prep.numel() * prep.element_size()), _i64(nb), _int(d), _int(k),
                                             _ptr(out_dist), _ptr(out_ids), _ptr(ws), wsz, _stream()))
        return out_dist, out_ids
    _check(lib().fs_flat_l2_knn(_ptr(xq), _i64(nq), _ptr(xb), _i64(nb), _int(d), _int(k),
                                _ptr(out_dist), _ptr(out_ids), _ptr(ws), wsz, _stream()))
    return out_dist, out_ids


def flat_prepare(xb: torch.Tensor, prep: torch.Tensor | None = None) -> torch.Tensor:
    """fs_flat_prepare: the database's share of the pre-pass (norms, operand split), once.  Returns the
    prepared block (a uint8 CUDA tensor of fs_flat_prepare_bytes) for flat_l2_knn(..., prep=...)."""
    _dev(xb, torch.float32, "xb")
    nb, d = xb.shape
    need = int(lib().fs_flat_prepare_bytes(_i64(nb), _int(d)))
    if prep is None:
        prep = torch.empty(need, dtype=torch.uint8, device=xb.device)
    _check(lib().fs_flat_prepare(_ptr(xb), _i64(nb), _int(d), _ptr(prep), _sz(prep.numel() * prep.element_size()),
                                 _stream()))
    return prep


def flat_l2_knn_host(xq, xb, k: int, out_dist=None, out_ids=None):
    """fs_flat_l2_knn_host: HOST buffers in and out (numpy or CPU torch tensors)."""
    import numpy as np
    xq, qp = _host_ptr(xq, np.float32, torch.float32, "xq")
    xb, bp = _host_ptr(xb, np.float32, torch.float32, "xb")
    nq, d = xq.shape
    dist = np.empty((nq, k), np.float32) if out_dist is None else out_dist
    ids = np.empty((nq, k), np.int64) if out_ids is None else out_ids
    dist, dp = _host_ptr(dist, np.float32, torch.float32, "out_dist")
    ids, ip = _host_ptr(ids, np.int64, torch.int64, "out_ids")
    _check(lib().fs_flat_l2_knn_host(_vp(qp), _i64(nq), _vp(bp), _i64(xb.shape[0]), _int(d), _int(k),
                                     _vp(dp), _vp(ip)))
    return dist, ids


def kmeans(x: torch.Tensor, K: int, niter: int, seed: int = 0, centroids: torch.Tensor | None = None,
           want_assign: bool = False):
    """fs_kmeans: Lloyd's k-means on CUDA fp32 x [n, d].  centroids given: start from them (they are not
    modified; a copy is returned), else from evenly strided input points.  Returns centroids [K, d]
    (and the int64 assignment of the last iteration with want_assign)."""
    _dev(x, torch.float32, "x")
    n, d = x.shape
    init = centroids is None
    cent = torch.empty((K, d), dtype=torch.float32, device=x.device) if init else _dev(centroids, torch.float32, "centroids").clone()
    assign = torch.empty(n, dtype=torch.int64, device=x.device) if want_assign else None
    _check(lib().fs_kmeans(_ptr(x), _i64(n), _int(d), _int(K), _int(niter), ctypes.c_uint64(seed), _int(1 if init else 0),
                           _ptr(cent), _ptr(assign), _stream()))
    return (cent, assign) if want_assign else cent


def merge_topk(dist: torch.Tensor, ids: torch.Tensor, out_dist=None, out_ids=None):
    """fs_merge_topk: dist fp32 [nq, G, k] and ids int64 [nq, G, k] (G partial lists per query, ids < 0 =
    padding) -> the k smallest (distance, id) pairs per query, ascending, ties by lower id."""
    _dev(dist, torch.float32, "dist")
    _dev(ids, torch.int64, "ids")
    nq, G, k = dist.shape
    if tuple(ids.shape) != (nq, G, k):
        raise ValueError("ids must have the shape of dist")
    if out_dist is None:
        out_dist = torch.empty((nq, k), dtype=torch.float32, device=dist.device)
    if out_ids is None:
        out_ids = torch.empty((nq, k), dtype=torch.int64, device=dist.device)
    _check(lib().fs_merge_topk(_ptr(dist), _ptr(ids), _i64(nq), _int(G), _int(k), _ptr(out_dist), _ptr(out_ids),
                               _vp(0), _sz(0), _stream()))
    return out_dist, out_ids


# ---------------------------------------------------------------------------
class IvfPq:
    """fs_ivfpq_*: IVFADC index with 8-bit residual PQ (Eq. 3-7, Alg. 4)."""

    def __init__(self, d: int, nlist: int, M: int):
        self.d, self.nlist, self.M = d, nlist, M
        self._h = _vp()
        _check(lib().fs_ivfpq_create(ctypes.byref(self._h), _int(d), _int(nlist), _int(M)))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().fs_ivfpq_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_quantizers(self, coarse: torch.Tensor, pq: torch.Tensor):
        _dev(coarse, torch.float32, "coarse")
        _dev(pq, torch.float32, "pq")
        assert tuple(coarse.shape) == (self.nlist, self.d)
        assert tuple(pq.shape) == (self.M, 256, self.d // self.M)
        _check(lib().fs_ivfpq_set_quantizers(self._h, _ptr(coarse), _ptr(pq), _stream()))

    def get_quantizers(self):
        dev = torch.device("cuda", torch.cuda.current_device())
        coarse = torch.empty((self.nlist, self.d), dtype=torch.float32, device=dev)
        pq = torch.empty((self.M, 256, self.d // self.M), dtype=torch.float32, device=dev)
        _check(lib().fs_ivfpq_get_quantizers(self._h, _ptr(coarse), _ptr(pq), _stream()))
        return coarse, pq

    def train(self, x: torch.Tensor, niter: int = 10, seed: int = 0):
        _dev(x, torch.float32, "x")
        _check(lib().fs_ivfpq_train(self._h, _ptr(x), _i64(x.shape[0]), _int(niter),
                                    ctypes.c_uint64(seed), _stream()))

    def add(self, xb: torch.Tensor, ids: torch.Tensor | None = None):
        _dev(xb, torch.float32, "xb")
        if ids is not None:
            _dev(ids, torch.int64, "ids")
        _check(lib().fs_ivfpq_add(self._h, _ptr(xb), _i64(xb.shape[0]), _ptr(ids), _stream()))

    @property
    def ntotal(self) -> int:
        return int(lib().fs_ivfpq_ntotal(self._h))

    @property
    def last_scanned_codes(self) -> int:
        return int(lib().fs_ivfpq_last_scanned_codes(self._h))

    @property
    def last_stage_ms(self):
        """fs_ivfpq_last_stage_ms: (C1, C2-C4, C5) device milliseconds of the last search."""
        ms = (ctypes.c_float * 3)()
        _check(lib().fs_ivfpq_last_stage_ms(self._h, ms))
        return tuple(float(v) for v in ms)

    def search_ws_bytes(self, nq: int, nprobe: int, k: int) -> int:
        return int(lib().fs_ivfpq_search_ws_bytes(self._h, _i64(nq), _int(nprobe), _int(k)))

    def search(self, xq: torch.Tensor, nprobe: int, k: int, want_probed: bool = False,
               out_dist=None, out_ids=None, ws=None):
        _dev(xq, torch.float32, "xq")
        nq = xq.shape[0]
        if out_dist is None:
            out_dist = torch.empty((nq, k), dtype=torch.float32, device=xq.device)
        if out_ids is None:
            out_ids = torch.empty((nq, k), dtype=torch.int64, device=xq.device)
        probed = torch.empty((nq, nprobe), dtype=torch.int32, device=xq.device) if want_probed else None
        _check(lib().fs_ivfpq_search(self._h, _ptr(xq), _i64(nq), _int(nprobe), _int(k),
                                     _ptr(out_dist), _ptr(out_ids), _ptr(probed), _ptr(ws),
                                     _sz(0 if ws is None else ws.numel() * ws.element_size()),
                                     _stream()))
        return (out_dist, out_ids, probed) if want_probed else (out_dist, out_ids)

    def knn_graph(self, x: torch.Tensor, nprobe: int, k: int, batch: int = 0, want_probed: bool = False,
                  out_dist=None, out_ids=None):
        """fs_ivfpq_knn_graph: all-vs-all search, row i = the k nearest stored vectors of x[i]."""
        _dev(x, torch.float32, "x")
        n = x.shape[0]
        if out_dist is None:
            out_dist = torch.empty((n, k), dtype=torch.float32, device=x.device)
        if out_ids is None:
            out_ids = torch.empty((n, k), dtype=torch.int64, device=x.device)
        _dev(out_dist, torch.float32, "out_dist")
        _dev(out_ids, torch.int64, "out_ids")
        probed = torch.empty((n, nprobe), dtype=torch.int32, device=x.device) if want_probed else None
        _check(lib().fs_ivfpq_knn_graph(self._h, _ptr(x), _i64(n), _int(nprobe), _int(k), _i64(batch),
                                        _ptr(out_dist), _ptr(out_ids), _ptr(probed), _stream()))
        return (out_dist, out_ids, probed) if want_probed else (out_dist, out_ids)

    def search_host(self, xq, nprobe: int, k: int, out_dist=None, out_ids=None):
        import numpy as np
        xq, qp = _host_ptr(xq, np.float32, torch.float32, "xq")
        nq = xq.shape[0]
        dist = np.empty((nq, k), np.float32) if out_dist is None else out_dist
        ids = np.empty((nq, k), np.int64) if out_ids is None else out_ids
        dist, dp = _host_ptr(dist, np.float32, torch.float32, "out_dist")
        ids, ip = _host_ptr(ids, np.int64, torch.int64, "out_ids")
        _check(lib().fs_ivfpq_search_host(self._h, _vp(qp), _i64(nq), _int(nprobe), _int(k), _vp(dp), _vp(ip)))
        return dist, ids

    def export(self):
        """CSR copy of the inverted file: (offsets int64 [nlist+1], codes uint8 [ntotal,M], ids int64)."""
        dev = torch.device("cuda", torch.cuda.current_device())
        nt = self.ntotal
        offsets = torch.empty(self.nlist + 1, dtype=torch.int64, device=dev)
        codes = torch.empty((nt, self.M), dtype=torch.uint8, device=dev)
        ids = torch.empty(nt, dtype=torch.int64, device=dev)
        _check(lib().fs_ivfpq_export(self._h, _ptr(offsets), _ptr(codes), _ptr(ids), _stream()))
        return offsets, codes, ids

    def export_lists(self, list_nos):
        """fs_ivfpq_export_lists: the given lists back to back.  list_nos: int sequence / numpy array.
        Returns (offsets numpy int64 [n+1] (host), codes uint8 [total,M] (device), ids int64 [total] (device))."""
        import numpy as np
        ln = np.ascontiguousarray(list_nos, dtype=np.int32)
        offs = np.empty(len(ln) + 1, np.int64)
        lp, op = _vp(ln.ctypes.data), _vp(offs.ctypes.data)
        _check(lib().fs_ivfpq_export_lists(self._h, lp, _i64(len(ln)), op, _vp(0), _vp(0), _stream()))
        dev = torch.device("cuda", torch.cuda.current_device())
        total = int(offs[-1])
        codes = torch.empty((total, self.M), dtype=torch.uint8, device=dev)
        ids = torch.empty(total, dtype=torch.int64, device=dev)
        _check(lib().fs_ivfpq_export_lists(self._h, lp, _i64(len(ln)), op, _ptr(codes), _ptr(ids), _stream()))
        return offs, codes, ids
