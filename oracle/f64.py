"""ORACLE — TEST INFRASTRUCTURE ONLY: fp64-coordinate searches (
PAPER.md:L32-34 "different ... floating point precisions").

Plain numpy brute force in float64 on float64 inputs: the definition of SURVEY.md §8(c-1)
verbatim (the same predicate table and kNN distance as oracle/arbx_oracle.cpp, which does its
fp64 arithmetic on fp32 inputs).  Pins (tests/test_oracle_pins.py): the integer-lattice closed
forms, and exact agreement with the (separately pinned) C++ oracle on inputs that are exactly
representable in fp32 -- both then do the same fp64 arithmetic on the same numbers.
Shares nothing with the CUDA path.
"""
from __future__ import annotations

import numpy as np

POINT, BOX, SPHERE = 0, 1, 2
EPS = 1e-6


def _dim(a: np.ndarray, kind: int) -> int:
    w = a.shape[1]
    return w if kind == POINT else w // 2 if kind == BOX else w - 1


def _dist2_pp(x, y):            # [nq,1,D] - [1,n,D]
    d = x[:, None, :] - y[None, :, :]
    return np.einsum("qnd,qnd->qn", d, d)


def _dist2_pb(x, lo, hi):       # points x [a,D] against boxes lo/hi [b,D] -> [a,b]
    d = np.maximum(0.0, np.maximum(lo[None, :, :] - x[:, None, :], x[:, None, :] - hi[None, :, :]))
    return np.einsum("abd,abd->ab", d, d)


def _classify(t, T, eps):
    """0 no match, 1 sure, 2 inside the band |t - T| <= eps*T (exact comparison when T == 0)."""
    T = np.broadcast_to(T, t.shape)
    out = np.where(t < T, 1, 0).astype(np.int8)
    out = np.where(np.abs(t - T) <= eps * T, 2, out)
    out = np.where(T == 0.0, np.where(t <= 0.0, 1, 0), out)
    return out


def _predicate(q, qkind, p, pkind, D, eps):
    """Matrix [nq, n] of classify codes; closed sets everywhere (reading A1)."""
    if qkind == SPHERE:
        c, r = q[:, :D], q[:, D]
        if pkind == POINT:
            m = _classify(_dist2_pp(c, p[:, :D]), (r * r)[:, None], eps)
        elif pkind == BOX:
            m = _classify(_dist2_pb(c, p[:, :D], p[:, D:2 * D]), (r * r)[:, None], eps)
        else:
            rr = r[:, None] + p[None, :, D]
            m = _classify(_dist2_pp(c, p[:, :D]), rr * rr, eps)
        return np.where((r < 0.0)[:, None], 0, m)          # reading A21
    if qkind == BOX:
        qlo, qhi = q[:, :D], q[:, D:2 * D]
        if pkind == POINT:
            return np.all((qlo[:, None, :] <= p[None, :, :D]) & (p[None, :, :D] <= qhi[:, None, :]), axis=2).astype(np.int8)
        if pkind == BOX:
            return np.all((p[None, :, :D] <= qhi[:, None, :]) & (qlo[:, None, :] <= p[None, :, D:2 * D]), axis=2).astype(np.int8)
        R = p[:, D]
        return _classify(_dist2_pb(p[:, :D], qlo, qhi).T, (R * R)[None, :], eps)
    if pkind == POINT:
        return np.all(p[None, :, :D] == q[:, None, :D], axis=2).astype(np.int8)
    if pkind == BOX:
        return np.all((p[None, :, :D] <= q[:, None, :D]) & (q[:, None, :D] <= p[None, :, D:2 * D]), axis=2).astype(np.int8)
    R = p[:, D]
    return _classify(_dist2_pp(q[:, :D], p[:, :D]), (R * R)[None, :], eps)


def spatial(prims, pkind: int, queries, qkind: int, eps: float = EPS, chunk: int = 256):
    """CSR rows as oracle.spatial: (offsets int64[nq+1], indices int32 ascending per row, band uint8)."""
    prims = np.ascontiguousarray(prims, dtype=np.float64)
    queries = np.ascontiguousarray(queries, dtype=np.float64)
    D = _dim(prims, pkind)
    counts, idx, band = [], [], []
    for a in range(0, queries.shape[0], chunk):
        m = _predicate(queries[a:a + chunk], qkind, prims, pkind, D, eps)
        rows, cols = np.nonzero(m)
        counts.append(np.bincount(rows, minlength=m.shape[0]))
        idx.append(cols.astype(np.int32))
        band.append((m[rows, cols] == 2).astype(np.uint8))
    counts = np.concatenate(counts) if counts else np.zeros(0, np.int64)
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    return off, (np.concatenate(idx) if idx else np.zeros(0, np.int32)), (np.concatenate(band) if band else np.zeros(0, np.uint8))


def knn_distance_matrix(prims, pkind: int, qpoints):
    prims = np.ascontiguousarray(prims, dtype=np.float64)
    qpoints = np.ascontiguousarray(qpoints, dtype=np.float64)
    D = _dim(prims, pkind)
    if pkind == POINT:
        return np.sqrt(_dist2_pp(qpoints, prims[:, :D]))
    if pkind == BOX:
        return np.sqrt(_dist2_pb(qpoints, prims[:, :D], prims[:, D:2 * D]))
    return np.maximum(0.0, np.sqrt(_dist2_pp(qpoints, prims[:, :D])) - prims[None, :, D])


def knn(prims, pkind: int, qpoints, k: int, chunk: int = 256):
    """(indices int32[nq,k], distances float64[nq,k]) ascending, ties by lower index, padded -1/+inf."""
    prims = np.ascontiguousarray(prims, dtype=np.float64)
    qpoints = np.ascontiguousarray(qpoints, dtype=np.float64)
    nq, n = qpoints.shape[0], prims.shape[0]
    idx = np.full((nq, k), -1, dtype=np.int32)
    dist = np.full((nq, k), np.inf, dtype=np.float64)
    kk = min(k, n)
    for a in range(0, nq, chunk):
        d = knn_distance_matrix(prims, pkind, qpoints[a:a + chunk])
        order = np.lexsort((np.broadcast_to(np.arange(n), d.shape), d), axis=1)[:, :kk]
        idx[a:a + chunk, :kk] = order
        dist[a:a + chunk, :kk] = np.take_along_axis(d, order, axis=1)
    return idx, dist
