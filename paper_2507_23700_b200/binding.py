"""Thin Python binding of the C ABI in include/arbx.h (argument marshalling only).

Every step of the hot path runs inside libarbx.so (hand-written sm_100a kernels); PyTorch is
used for device memory and streams.  There is NO CPU fallback: if the shared library is
missing or no CUDA device is present, calls raise.

The functions carry the ABI's names (arbx_build, arbx_query_count, arbx_query_spatial,
arbx_query_knn, ...).  `Index` is a small convenience wrapper owning one handle.
"""
from __future__ import annotations

import ctypes
import os

import torch

POINT, BOX, SPHERE = 0, 1, 2
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_CAPACITY, ERR_OVERFLOW, ERR_CUDA, ERR_OOM = range(7)
K_MAX = 256

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libarbx.so")

EXPORTS = (
    "arbx_build", "arbx_destroy", "arbx_size", "arbx_bounds", "arbx_query_count",
    "arbx_query_count_upto", "arbx_query_spatial", "arbx_query_spatial_upto", "arbx_query_pairs", "arbx_dbscan", "arbx_query_knn", "arbx_sort_pairs", "arbx_debug_validate",
    "arbx_query_knn_var", "arbx_trim", "arbx_debug_set",
    "arbx_build_f64", "arbx_query_count_f64", "arbx_query_spatial_f64", "arbx_query_knn_f64",
    "arbx_query_count_noalloc",
    "arbx_launch_count", "arbx_profile_enable", "arbx_profile_num_kernels",
    "arbx_profile_kernel_name", "arbx_profile_read", "arbx_status_string", "arbx_last_error",
)


class ArbxError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        L = lib()
        super().__init__(f"{where}: {L.arbx_status_string(status).decode()} -- {L.arbx_last_error().decode()}")


_lib = None


def lib() -> ctypes.CDLL:
    """Load libarbx.so (built by `make -C paper_2507_23700_b200/csrc` or __graft_entry__.build())."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
                "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
        L.arbx_build.argtypes = [vp, i64, i32, i32, vp, ctypes.POINTER(vp)]
        L.arbx_destroy.argtypes = [vp, vp]
        L.arbx_size.argtypes = [vp, ctypes.POINTER(i64)]
        L.arbx_bounds.argtypes = [vp, vp, vp, vp]
        L.arbx_query_count.argtypes = [vp, vp, i64, i32, vp, vp]
        L.arbx_query_count_upto.argtypes = [vp, vp, i64, i32, i32, vp, vp]
        L.arbx_query_spatial.argtypes = [vp, vp, i64, i32, vp, vp, i64, ctypes.POINTER(i64), vp]
        L.arbx_query_spatial_upto.argtypes = [vp, vp, i64, i32, i32, vp, vp, i64, ctypes.POINTER(i64), vp]
        L.arbx_query_pairs.argtypes = [vp, ctypes.c_float, vp, vp, i64, ctypes.POINTER(i64), vp]
        L.arbx_dbscan.argtypes = [vp, ctypes.c_float, i32, vp, vp]
        L.arbx_query_knn.argtypes = [vp, vp, i64, i32, vp, vp, vp]
        L.arbx_query_knn_var.argtypes = [vp, vp, i64, vp, i32, vp, vp, vp]
        L.arbx_build_f64.argtypes = [vp, i64, i32, i32, vp, ctypes.POINTER(vp)]
        L.arbx_query_count_f64.argtypes = [vp, vp, i64, i32, vp, vp]
        L.arbx_query_spatial_f64.argtypes = [vp, vp, i64, i32, vp, vp, i64, ctypes.POINTER(i64), vp]
        L.arbx_query_knn_f64.argtypes = [vp, vp, i64, i32, vp, vp, vp]
        L.arbx_query_count_noalloc.argtypes = [vp, vp, i64, i32, vp, vp]
        L.arbx_trim.argtypes = [i64]
        L.arbx_debug_set.argtypes = [ctypes.c_char_p, ctypes.c_double]
        L.arbx_sort_pairs.argtypes = [vp, vp, i64, i32, i32, vp]
        L.arbx_debug_validate.argtypes = [vp, ctypes.POINTER(i64), vp]
        L.arbx_launch_count.restype = i64
        L.arbx_profile_enable.argtypes = [i32]
        L.arbx_profile_enable.restype = i32
        L.arbx_profile_num_kernels.restype = i32
        L.arbx_profile_kernel_name.argtypes = [i32]
        L.arbx_profile_kernel_name.restype = ctypes.c_char_p
        L.arbx_profile_read.argtypes = [vp, vp, i32]
        L.arbx_profile_read.restype = i32
        L.arbx_status_string.restype = ctypes.c_char_p
        L.arbx_status_string.argtypes = [i32]
        L.arbx_last_error.restype = ctypes.c_char_p
        for name in EXPORTS[:21]:
            getattr(L, name).restype = i32
        _lib = L
    return _lib


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _dev_f32(t: torch.Tensor, what: str, dtype=torch.float32) -> torch.Tensor:
    if not (isinstance(t, torch.Tensor) and t.is_cuda):
        raise TypeError(f"{what} must be a CUDA tensor (no CPU path exists)")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{what} must be contiguous {dtype}")
    return t


def _ptr(t) -> int:
    return 0 if t is None or t.numel() == 0 else t.data_ptr()


def row_width(kind: int, dim: int) -> int:
    return dim if kind == POINT else 2 * dim if kind == BOX else dim + 1


def _check(st: int, where: str):
    if st != OK:
        raise ArbxError(st, where)


# ---- functions named after the ABI ----------------------------------------------------------
def arbx_build(prims: torch.Tensor, dim: int, kind: int, stream=None) -> int:
    prims = _dev_f32(prims, "prims")
    n = prims.numel() // row_width(kind, dim) if prims.numel() else 0
    h = ctypes.c_void_p()
    _check(lib().arbx_build(_ptr(prims), n, dim, kind, _stream(stream), ctypes.byref(h)), "arbx_build")
    return h.value


def arbx_build_f64(prims: torch.Tensor, dim: int, kind: int, stream=None) -> int:
    prims = _dev_f32(prims, "prims", torch.float64)
    n = prims.numel() // row_width(kind, dim) if prims.numel() else 0
    h = ctypes.c_void_p()
    _check(lib().arbx_build_f64(_ptr(prims), n, dim, kind, _stream(stream), ctypes.byref(h)), "arbx_build_f64")
    return h.value


def arbx_query_count_f64(handle: int, queries: torch.Tensor, nq: int, qkind: int, counts: torch.Tensor, stream=None) -> None:
    _check(lib().arbx_query_count_f64(handle, _ptr(queries), nq, qkind, _ptr(counts), _stream(stream)), "arbx_query_count_f64")


def arbx_query_spatial_f64(handle: int, queries: torch.Tensor, nq: int, qkind: int, offsets: torch.Tensor,
                           indices, capacity: int, stream=None, raise_on_capacity: bool = True):
    """Returns (status, total)."""
    total = ctypes.c_int64()
    st = lib().arbx_query_spatial_f64(handle, _ptr(queries), nq, qkind, offsets.data_ptr(),
                                      0 if indices is None else indices.data_ptr(), capacity,
                                      ctypes.byref(total), _stream(stream))
    if st != OK and (raise_on_capacity or st != ERR_CAPACITY):
        raise ArbxError(st, "arbx_query_spatial_f64")
    return st, total.value


def arbx_query_knn_f64(handle: int, qpoints: torch.Tensor, nq: int, k: int, indices: torch.Tensor, distances,
                       stream=None) -> None:
    _check(lib().arbx_query_knn_f64(handle, _ptr(qpoints), nq, k, _ptr(indices),
                                    0 if distances is None else _ptr(distances), _stream(stream)), "arbx_query_knn_f64")


def arbx_destroy(handle: int, stream=None) -> None:
    _check(lib().arbx_destroy(handle, _stream(stream)), "arbx_destroy")


def arbx_size(handle: int) -> int:
    n = ctypes.c_int64()
    _check(lib().arbx_size(handle, ctypes.byref(n)), "arbx_size")
    return n.value


def arbx_bounds(handle: int, dim: int, stream=None):
    lo = (ctypes.c_float * dim)()
    hi = (ctypes.c_float * dim)()
    _check(lib().arbx_bounds(handle, ctypes.addressof(lo), ctypes.addressof(hi), _stream(stream)), "arbx_bounds")
    return list(lo), list(hi)


def arbx_query_count(handle: int, queries: torch.Tensor, nq: int, qkind: int, counts: torch.Tensor,
                     stream=None) -> None:
    _check(lib().arbx_query_count(handle, _ptr(queries), nq, qkind, _ptr(counts), _stream(stream)),
           "arbx_query_count")


NOALLOC_MAX_QUERIES = 1 << 20


def arbx_query_count_noalloc(handle: int, queries: torch.Tensor, nq: int, qkind: int, counts: torch.Tensor,
                             stream=None) -> None:
    """arbx_query_count without any allocation (fixed scratch inside the library, nq <= 2^20)."""
    _check(lib().arbx_query_count_noalloc(handle, _ptr(queries), nq, qkind, _ptr(counts), _stream(stream)),
           "arbx_query_count_noalloc")


def arbx_query_count_upto(handle: int, queries: torch.Tensor, nq: int, qkind: int, limit: int,
                          counts: torch.Tensor, stream=None) -> None:
    _check(lib().arbx_query_count_upto(handle, _ptr(queries), nq, qkind, limit, _ptr(counts), _stream(stream)),
           "arbx_query_count_upto")


def arbx_query_spatial(handle: int, queries: torch.Tensor, nq: int, qkind: int, offsets: torch.Tensor,
                       indices, capacity: int, stream=None, raise_on_capacity: bool = True):
    """Returns (status, total)."""
    total = ctypes.c_int64()
    st = lib().arbx_query_spatial(handle, _ptr(queries), nq, qkind, offsets.data_ptr(),
                                  0 if indices is None else indices.data_ptr(), capacity,
                                  ctypes.byref(total), _stream(stream))
    if st != OK and (raise_on_capacity or st != ERR_CAPACITY):
        raise ArbxError(st, "arbx_query_spatial")
    return st, total.value


def arbx_query_spatial_upto(handle: int, queries: torch.Tensor, nq: int, qkind: int, limit: int,
                            offsets: torch.Tensor, indices, capacity: int, stream=None):
    """Returns (status, total); ERR_CAPACITY is returned, not raised."""
    total = ctypes.c_int64()
    st = lib().arbx_query_spatial_upto(handle, _ptr(queries), nq, qkind, limit, offsets.data_ptr(),
                                       0 if indices is None else indices.data_ptr(), capacity,
                                       ctypes.byref(total), _stream(stream))
    if st not in (OK, ERR_CAPACITY):
        raise ArbxError(st, "arbx_query_spatial_upto")
    return st, total.value


def arbx_query_pairs(handle: int, radius: float, offsets: torch.Tensor, indices, capacity: int, stream=None):
    """Returns (status, total); ERR_CAPACITY is returned, not raised."""
    total = ctypes.c_int64()
    st = lib().arbx_query_pairs(handle, radius, offsets.data_ptr(), 0 if indices is None else indices.data_ptr(),
                                capacity, ctypes.byref(total), _stream(stream))
    if st not in (OK, ERR_CAPACITY):
        raise ArbxError(st, "arbx_query_pairs")
    return st, total.value


def arbx_dbscan(handle: int, eps: float, min_pts: int, labels: torch.Tensor, stream=None) -> None:
    _check(lib().arbx_dbscan(handle, eps, min_pts, _ptr(labels), _stream(stream)), "arbx_dbscan")


def arbx_query_knn(handle: int, qpoints: torch.Tensor, nq: int, k: int, indices: torch.Tensor,
                   distances, stream=None) -> None:
    _check(lib().arbx_query_knn(handle, _ptr(qpoints), nq, k, _ptr(indices),
                                0 if distances is None else _ptr(distances), _stream(stream)),
           "arbx_query_knn")


def arbx_query_knn_var(handle: int, qpoints: torch.Tensor, nq: int, k_per_query: torch.Tensor, kmax: int,
                       indices: torch.Tensor, distances, stream=None) -> None:
    if not (k_per_query.is_cuda and k_per_query.dtype == torch.int32 and k_per_query.is_contiguous()):
        raise TypeError("k_per_query must be a contiguous CUDA int32 tensor")
    _check(lib().arbx_query_knn_var(handle, _ptr(qpoints), nq, _ptr(k_per_query), kmax, _ptr(indices),
                                    0 if distances is None else _ptr(distances), _stream(stream)),
           "arbx_query_knn_var")


def arbx_trim(keep_bytes: int = 0) -> None:
    _check(lib().arbx_trim(keep_bytes), "arbx_trim")


def arbx_debug_set(key: str, value: float) -> None:
    _check(lib().arbx_debug_set(key.encode(), float(value)), "arbx_debug_set")


def arbx_sort_pairs(keys: torch.Tensor, values, key_bits: int, stream=None) -> None:
    assert keys.is_cuda and keys.is_contiguous() and keys.element_size() in (4, 8)
    _check(lib().arbx_sort_pairs(_ptr(keys), 0 if values is None else _ptr(values), keys.numel(),
                                 keys.element_size(), key_bits, _stream(stream)), "arbx_sort_pairs")


def arbx_debug_validate(handle: int, stream=None) -> int:
    v = ctypes.c_int64()
    _check(lib().arbx_debug_validate(handle, ctypes.byref(v), _stream(stream)), "arbx_debug_validate")
    return v.value


def arbx_launch_count() -> int:
    return int(lib().arbx_launch_count())


def arbx_profile_enable(on: bool) -> None:
    _check(lib().arbx_profile_enable(1 if on else 0), "arbx_profile_enable")


def arbx_profile_read() -> dict:
    """{kernel name: (milliseconds, bracketed steps)} accumulated since the last read."""
    L = lib()
    nk = L.arbx_profile_num_kernels()
    ms = (ctypes.c_double * nk)()
    calls = (ctypes.c_int64 * nk)()
    _check(L.arbx_profile_read(ctypes.addressof(ms), ctypes.addressof(calls), nk), "arbx_profile_read")
    return {L.arbx_profile_kernel_name(i).decode(): (ms[i], calls[i]) for i in range(nk) if calls[i]}


# ---- convenience wrapper -----------------------------------------------------------------------
class Index:
    """One BVH over `prims` (CUDA float32 [n, row_width]).  PAPER.md:L89-123 (BVH class)."""

    def __init__(self, prims: torch.Tensor, kind: int = POINT, dim: int | None = None, stream=None):
        self.f64 = isinstance(prims, torch.Tensor) and prims.dtype == torch.float64
        self.dtype = torch.float64 if self.f64 else torch.float32
        prims = _dev_f32(prims, "prims", self.dtype)
        if dim is None:
            if prims.dim() != 2:
                raise ValueError("give dim= for a flat prims array")
            w = prims.shape[1]
            dim = w if kind == POINT else w // 2 if kind == BOX else w - 1
        self.dim, self.kind, self.device = dim, kind, prims.device
        self.handle = (arbx_build_f64 if self.f64 else arbx_build)(prims, dim, kind, stream)
        self._per_query = 16.0      # matches per query seen so far: sizes the next CSR buffer

    def close(self, stream=None):
        if getattr(self, "handle", None):
            arbx_destroy(self.handle, stream)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def size(self) -> int:
        return arbx_size(self.handle)

    def empty(self) -> bool:
        return self.size() == 0

    def bounds(self, stream=None):
        return arbx_bounds(self.handle, self.dim, stream)

    def _nq(self, queries: torch.Tensor, qkind: int) -> int:
        _dev_f32(queries, "queries", self.dtype)
        return queries.numel() // row_width(qkind, self.dim)

    def query_count(self, queries: torch.Tensor, qkind: int = SPHERE, stream=None,
                    limit: int | None = None) -> torch.Tensor:
        """counts[q] = matches of query q; with `limit`, min(matches, limit) with early exit."""
        nq = self._nq(queries, qkind)
        counts = torch.empty(nq, dtype=torch.int32, device=self.device)
        if self.f64:
            if limit is not None:
                raise ArbxError(ERR_UNSUPPORTED, "capped count on an fp64 index")
            arbx_query_count_f64(self.handle, queries, nq, qkind, counts, stream)
        elif limit is None:
            arbx_query_count(self.handle, queries, nq, qkind, counts, stream)
        else:
            arbx_query_count_upto(self.handle, queries, nq, qkind, limit, counts, stream)
        return counts

    def query_spatial(self, queries: torch.Tensor, qkind: int = SPHERE, capacity: int | None = None,
                      stream=None):
        """CSR result (offsets int32[nq+1], indices int32[total]).  One ABI call (one traversal)
        when `capacity` -- given by the caller, else guessed from the matches per query this
        index has seen so far -- holds the result; on ARBX_ERR_CAPACITY the call has left the
        exact total, and a second call with a buffer of that size fills."""
        nq = self._nq(queries, qkind)
        offsets = torch.empty(nq + 1, dtype=torch.int32, device=self.device)
        if capacity is None:
            capacity = int(nq * self._per_query * 1.25) + 1024
        call = arbx_query_spatial_f64 if self.f64 else arbx_query_spatial
        indices = torch.empty(capacity, dtype=torch.int32, device=self.device)
        st, total = call(self.handle, queries, nq, qkind, offsets, indices, capacity, stream, raise_on_capacity=False)
        if nq:
            self._per_query = max(1.0, total / nq)
        if st == OK:
            return offsets, indices[:total]
        indices = torch.empty(total, dtype=torch.int32, device=self.device)
        call(self.handle, queries, nq, qkind, offsets, indices, total, stream)
        return offsets, indices

    def query_spatial_upto(self, queries: torch.Tensor, limit: int, qkind: int = SPHERE, stream=None):
        """CSR result with at most `limit` matches per query (early exit)."""
        nq = self._nq(queries, qkind)
        offsets = torch.empty(nq + 1, dtype=torch.int32, device=self.device)
        indices = torch.empty(max(nq * limit, 1), dtype=torch.int32, device=self.device)
        _, total = arbx_query_spatial_upto(self.handle, queries, nq, qkind, limit, offsets, indices,
                                           indices.numel(), stream)
        return offsets, indices[:total]

    def query_pairs(self, radius: float, stream=None):
        """Self-join: CSR (offsets int32[n+1], indices) holding every unordered pair within radius once."""
        n = self.size()
        offsets = torch.empty(n + 1, dtype=torch.int32, device=self.device)
        _, total = arbx_query_pairs(self.handle, radius, offsets, None, 0, stream)
        indices = torch.empty(max(total, 1), dtype=torch.int32, device=self.device)
        arbx_query_pairs(self.handle, radius, offsets, indices, indices.numel(), stream)
        return offsets, indices[:total]

    def dbscan(self, eps: float, min_pts: int, stream=None) -> torch.Tensor:
        """labels int32[n]: smallest core index of the point's cluster, -1 = noise."""
        labels = torch.empty(self.size(), dtype=torch.int32, device=self.device)
        arbx_dbscan(self.handle, eps, min_pts, labels, stream)
        return labels

    def query_knn(self, qpoints: torch.Tensor, k, want_distances: bool = True, stream=None, kmax: int | None = None):
        """k: one int for all queries, or a CUDA int32 tensor with one k per query (rows of kmax
        entries, padded with -1 / +inf; kmax defaults to max(k))."""
        nq = self._nq(qpoints, POINT)
        per_query = isinstance(k, torch.Tensor)
        width = int(k) if not per_query else max(1, int(kmax if kmax is not None else (int(k.max()) if nq else 1)))
        idx = torch.empty((nq, max(width, 0)), dtype=torch.int32, device=self.device)
        dist = torch.empty((nq, max(width, 0)), dtype=self.dtype, device=self.device) if want_distances else None
        if self.f64:
            if per_query:
                raise ArbxError(ERR_UNSUPPORTED, "per-query k on an fp64 index")
            arbx_query_knn_f64(self.handle, qpoints, nq, width, idx, dist, stream)
        elif per_query:
            arbx_query_knn_var(self.handle, qpoints, nq, k, width, idx, dist, stream)
        else:
            arbx_query_knn(self.handle, qpoints, nq, width, idx, dist, stream)
        return idx, dist

    def validate(self, stream=None) -> int:
        return arbx_debug_validate(self.handle, stream)
