"""ORACLE — TEST INFRASTRUCTURE ONLY (ctypes binding of oracle/arbx_oracle.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares nothing with paper_2507_23700_b200 (the CUDA path) and never
imports it.  See the header of arbx_oracle.cpp for what is computed and how it is pinned.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "arbx_oracle.cpp")
_LIB = os.path.join(_HERE, "libarbx_oracle.so")

POINT, BOX, SPHERE = 0, 1, 2
EPS = 1e-6  # tolerance band of BASELINE.json north_star / SURVEY.md §8(c-3)


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (C++17, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp, i64, i32, f64 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
        L.orc_num_threads.restype = i32
        L.orc_grid_build.restype = vp
        L.orc_grid_build.argtypes = [vp, i64, i32, i32, f64]
        L.orc_grid_free.argtypes = [vp]
        L.orc_grid_cell.restype = f64
        L.orc_grid_cell.argtypes = [vp]
        L.orc_spatial.restype = vp
        L.orc_spatial.argtypes = [vp, vp, i64, i32, i32, vp, i64, i32, f64]
        L.orc_spatial_total.restype = i64
        L.orc_spatial_total.argtypes = [vp]
        L.orc_spatial_copy.argtypes = [vp, vp, vp, vp]
        L.orc_spatial_free.argtypes = [vp]
        L.orc_knn.argtypes = [vp, vp, i64, i32, i32, vp, i64, i32, vp, vp]
        L.orc_knn_distance_pairs.argtypes = [vp, i32, i32, vp, vp, vp, i64, vp]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _f32(a) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _dim(prims: np.ndarray, pkind: int) -> int:
    w = prims.shape[1]
    return w if pkind == POINT else w // 2 if pkind == BOX else w - 1


class Grid:
    """Hashed uniform grid over the primitives (Mode B)."""

    def __init__(self, prims, pkind: int, cell: float):
        self.prims = _f32(prims)
        self.pkind = pkind
        self.dim = _dim(self.prims, pkind)
        self.h = lib().orc_grid_build(_ptr(self.prims), self.prims.shape[0], self.dim, pkind, float(cell))

    @property
    def cell(self) -> float:
        return float(lib().orc_grid_cell(self.h))

    def __del__(self):
        try:
            if self.h:
                lib().orc_grid_free(self.h)
                self.h = None
        except Exception:
            pass


def spatial(prims, pkind: int, queries, qkind: int, grid: Grid | None = None, eps: float = EPS):
    """Rows {i : predicate(query, prim_i)} as CSR.  Returns (offsets int64[nq+1],
    indices int32[total] ascending per row, band uint8[total]); band==1 marks pairs with
    |t-T| <= eps*T which a correct fp32 implementation may report either way."""
    prims = grid.prims if grid is not None else _f32(prims)
    queries = _f32(queries)
    dim = _dim(prims, pkind)
    nq = queries.shape[0]
    L = lib()
    r = L.orc_spatial(grid.h if grid is not None else None, _ptr(prims), prims.shape[0], dim, pkind,
                      _ptr(queries), nq, qkind, float(eps))
    try:
        total = L.orc_spatial_total(r)
        offsets = np.zeros(nq + 1, dtype=np.int64)
        indices = np.zeros(total, dtype=np.int32)
        band = np.zeros(total, dtype=np.uint8)
        L.orc_spatial_copy(r, _ptr(offsets), _ptr(indices), _ptr(band))
    finally:
        L.orc_spatial_free(r)
    return offsets, indices, band


def knn(prims, pkind: int, qpoints, k: int, grid: Grid | None = None):
    """k nearest primitives per query point: (indices int32[nq,k], distances float64[nq,k]),
    ascending distance, ties by lower index, padded with -1/+inf when n < k."""
    prims = grid.prims if grid is not None else _f32(prims)
    qpoints = _f32(qpoints)
    dim = _dim(prims, pkind)
    nq = qpoints.shape[0]
    idx = np.full((nq, k), -1, dtype=np.int32)
    dist = np.full((nq, k), np.inf, dtype=np.float64)
    lib().orc_knn(grid.h if grid is not None else None, _ptr(prims), prims.shape[0], dim, pkind,
                  _ptr(qpoints), nq, int(k), _ptr(idx), _ptr(dist))
    return idx, dist


def knn_var(prims, pkind: int, qpoints, kq, kmax: int, grid: Grid | None = None):
    """Per-query k (a nearest query is "a pair of a query point and a number of
    neighbors"): row q holds the k_q = clip(kq[q], 0, kmax) nearest primitives, i.e. the first
    k_q entries of the kmax-nearest row (rows ascend, ties by lower index), then padding
    (-1 / +inf).  Returns (indices int32[nq,kmax], distances float64[nq,kmax])."""
    idx, dist = knn(prims, pkind, qpoints, kmax, grid)
    kq = np.clip(np.asarray(kq, dtype=np.int64), 0, kmax)
    cut = np.arange(kmax)[None, :] >= kq[:, None]
    idx[cut] = -1
    dist[cut] = np.inf
    return idx, dist


def knn_distance_pairs(prims, pkind: int, qpoints, qids, pids) -> np.ndarray:
    """fp64 kNN distance of named (query, primitive) pairs (comparator rule 4)."""
    prims = _f32(prims)
    qpoints = _f32(qpoints)
    qids = np.ascontiguousarray(qids, dtype=np.int64)
    pids = np.ascontiguousarray(pids, dtype=np.int32)
    out = np.empty(qids.shape[0], dtype=np.float64)
    lib().orc_knn_distance_pairs(_ptr(prims), _dim(prims, pkind), pkind, _ptr(qpoints), _ptr(qids),
                                 _ptr(pids), qids.shape[0], _ptr(out))
    return out


def default_cell(prims, pkind: int, mode: str, r: float | None = None, per_cell: float = 3.0) -> float:
    """Cell-size heuristic of SURVEY.md §8(c-2) step 2 (any positive value is correct)."""
    prims = _f32(prims)
    dim = _dim(prims, pkind)
    n = max(1, prims.shape[0])
    c = prims[:, :dim] if pkind != BOX else 0.5 * (prims[:, :dim] + prims[:, dim:])
    ext = np.maximum(c.max(axis=0).astype(np.float64) - c.min(axis=0).astype(np.float64), 1e-30)
    vol = float(np.prod(ext))
    occ = (per_cell * vol / n) ** (1.0 / dim)
    if mode == "spatial" and r is not None and r > 0:
        return max(float(r), 0.5 * occ)
    return occ


def dbscan(points, eps: float, min_pts: int):
    """Textbook DBSCAN on the brute-force /
    grid neighbour lists of this oracle.  A point is core iff >= min_pts points (itself
    included) lie within eps (closed); clusters are the connected components of the core
    points under "within eps"; a non-core point within eps of a core point is a border point
    and may belong to ANY adjacent core's cluster; the rest is noise.
    Returns (core bool[n], comp int[n] (component id of core points, -1 otherwise),
             allowed: list of sets of component ids a border point may take (empty = noise),
             band_any: True if some pair sits in the 1e-6 tolerance band (then compare loosely))."""
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import connected_components
    points = _f32(points)
    n = points.shape[0]
    q = np.concatenate([points, np.full((n, 1), eps, dtype=np.float32)], axis=1)
    grid = Grid(points, POINT, max(float(eps), 1e-6)) if n > 20000 else None
    off, idx, band = spatial(points, POINT, q, SPHERE, grid)
    counts = np.diff(off)
    core = counts >= min_pts
    rows = np.repeat(np.arange(n), counts)
    keep = core[rows] & core[idx]
    g = csr_matrix((np.ones(int(keep.sum()), dtype=np.int8), (rows[keep], idx[keep])), shape=(n, n))
    _, lab = connected_components(g, directed=False)
    comp = np.where(core, lab, -1)
    allowed = [set() for _ in range(n)]
    nb = (~core[rows]) & core[idx]
    for r, c in zip(rows[nb], idx[nb]):
        allowed[r].add(int(comp[c]))
    return core, comp, allowed, bool(band.any())
