"""ORACLE-side comparators (test infrastructure): the comparison protocol of SURVEY.md §8(c-3)
/ BASELINE.json north_star, applied to result arrays produced by ANY implementation.

  spatial : sure(q) ⊆ G(q) ⊆ sure(q) ∪ band(q); rows duplicate-free; counts consistent.
  kNN     : rules (1)..(5) of §8(c-3).
Nothing here touches the CUDA path; inputs are plain numpy arrays.
"""
from __future__ import annotations

import numpy as np

from . import EPS, knn_distance_pairs


def _keys(offsets: np.ndarray, indices: np.ndarray, n: int) -> np.ndarray:
    offsets = np.asarray(offsets, dtype=np.int64)
    rows = np.repeat(np.arange(offsets.shape[0] - 1, dtype=np.int64), np.diff(offsets))
    return rows * np.int64(max(n, 1)) + np.asarray(indices, dtype=np.int64)


def check_csr_format(offsets, indices, n: int, nq: int) -> None:
    """Pin P4: offsets[0]=0, non-decreasing, offsets[nq]=total, indices in [0,n)."""
    offsets = np.asarray(offsets)
    assert offsets.shape[0] == nq + 1, "offsets must have nq+1 entries"
    assert int(offsets[0]) == 0, "offsets[0] != 0"
    assert np.all(np.diff(offsets.astype(np.int64)) >= 0), "offsets decrease"
    total = int(offsets[-1])
    assert total == len(indices), f"offsets[nq]={total} != len(indices)={len(indices)}"
    if total:
        ind = np.asarray(indices)
        assert ind.min() >= 0 and ind.max() < n, "index out of range"


def compare_spatial(n: int, orc, got, what: str = "") -> dict:
    """orc = (offsets, indices, band) from oracle.spatial; got = (offsets, indices)."""
    o_off, o_idx, o_band = orc
    g_off, g_idx = got
    nq = len(o_off) - 1
    check_csr_format(g_off, g_idx, n, nq)
    ko = _keys(o_off, o_idx, n)
    kg = np.sort(_keys(g_off, g_idx, n))
    assert np.all(np.diff(kg) > 0), f"{what}: duplicate index inside a row"
    sure = ko[np.asarray(o_band) == 0]
    missing = ~np.isin(sure, kg, assume_unique=True)
    assert not missing.any(), (
        f"{what}: {int(missing.sum())} sure pairs missing, first (q,i)="
        f"{divmod(int(sure[missing][0]), max(n, 1))}")
    extra = ~np.isin(kg, ko, assume_unique=True)
    assert not extra.any(), (
        f"{what}: {int(extra.sum())} pairs reported that are neither sure nor band, first (q,i)="
        f"{divmod(int(kg[extra][0]), max(n, 1))}")
    return dict(pairs=int(len(kg)), sure=int(len(sure)), band=int(len(ko) - len(sure)))


def compare_counts(orc, counts, what: str = "") -> None:
    """|sure| <= counts[q] <= |sure|+|band| per query (bit-exact where the band is empty)."""
    o_off, _, o_band = orc
    o_off = np.asarray(o_off, dtype=np.int64)
    allc = np.diff(o_off)
    bandc = np.add.reduceat(np.concatenate([np.asarray(o_band, dtype=np.int64), [0]]),
                            np.minimum(o_off[:-1], len(o_band)))
    bandc = np.where(allc == 0, 0, bandc)
    counts = np.asarray(counts, dtype=np.int64)
    bad = (counts < allc - bandc) | (counts > allc)
    assert not bad.any(), f"{what}: {int(bad.sum())} counts outside [sure, sure+band], first q={int(np.argmax(bad))}"


def _sphere_slack(prims, dim: int, idx, d) -> np.ndarray:
    """Per-pair absolute slack for SPHERE primitives, where the fp32 distance ||y-c|| - R
    cancels: |error| <= 4 * 2^-23 * (||y-c|| + R) <= 2^-21 * (d + 2R), because
    ||y-c|| <= d + R.  idx < 0 (padding) gets 0."""
    idx = np.asarray(idx)
    R = np.where(idx >= 0, prims[np.maximum(idx, 0), dim].astype(np.float64), 0.0)
    dd = np.where(np.isfinite(d), d, 0.0)
    return 2.0 ** -21 * (dd + 2.0 * R)


def compare_knn(prims, pkind: int, qpoints, k: int, orc, got, eps: float = EPS, what: str = "") -> None:
    """orc = (idx[nq,k], dist64[nq,k]); got = (idx[nq,k] int32, dist[nq,k] fp32 or None).
    For SPHERE primitives every distance tolerance is widened by the per-pair cancellation
    bound of _sphere_slack (position-wise rules use the largest slack of the row, since fp32
    keys that differ by less than the slack may swap places)."""
    SPHERE = 2
    o_idx, o_d = orc
    g_idx, g_d = got
    g_idx = np.asarray(g_idx)
    nq = o_idx.shape[0]
    n = prims.shape[0]
    kk = min(k, n)
    assert g_idx.shape == (nq, k)
    # (1) min(k,n) valid entries, padding only when n < k, no duplicates
    assert np.all(g_idx[:, :kk] >= 0) and np.all(g_idx[:, :kk] < n), f"{what}: invalid index"
    assert np.all(g_idx[:, kk:] == -1), f"{what}: padding must be -1"
    if kk > 1:
        s = np.sort(g_idx[:, :kk], axis=1)
        assert np.all(np.diff(s, axis=1) > 0), f"{what}: duplicate neighbour in a row"
    if kk == 0:
        return
    qids = np.repeat(np.arange(nq, dtype=np.int64), kk)
    d_true = knn_distance_pairs(prims, pkind, qpoints, qids, g_idx[:, :kk].reshape(-1)).reshape(nq, kk)
    Dk = o_d[:, kk - 1][:, None]
    if pkind == SPHERE:
        dim = qpoints.shape[1]
        pair_tol = _sphere_slack(prims, dim, g_idx[:, :kk], d_true)
        abs_tol = np.maximum(pair_tol, _sphere_slack(prims, dim, o_idx[:, :kk], o_d[:, :kk])).max(axis=1)[:, None]
    else:
        pair_tol = abs_tol = 0.0
    # (5b) every reported neighbour lies within D_k(1+eps)
    assert np.all(d_true <= Dk * (1 + eps) + abs_tol), f"{what}: reported neighbour farther than D_k(1+eps)"
    # (5a) every oracle neighbour strictly closer than D_k(1-eps) is reported
    must = o_d[:, :kk] < Dk * (1 - eps) - abs_tol
    key_g = np.sort((np.arange(nq, dtype=np.int64)[:, None] * n + g_idx[:, :kk]).reshape(-1))
    key_o = (np.arange(nq, dtype=np.int64)[:, None] * n + o_idx[:, :kk])[must]
    assert np.isin(key_o, key_g).all(), f"{what}: a neighbour strictly inside D_k is missing"
    if g_d is not None:
        g_d = np.asarray(g_d, dtype=np.float64)
        assert np.all(np.isinf(g_d[:, kk:])), f"{what}: padding distance must be +inf"
        gd = g_d[:, :kk]
        # (2) ascending in fp32
        assert np.all(np.diff(gd, axis=1) >= 0), f"{what}: distances not ascending"
        # (3) position-wise agreement with the oracle distances
        od = o_d[:, :kk]
        assert np.all(np.abs(gd - od) <= eps * od + abs_tol), (
            f"{what}: distance mismatch, max rel {np.max(np.abs(gd - od) / np.maximum(od, 1e-300)):.3e}")
        # (4) the reported distance belongs to the reported index
        assert np.all(np.abs(gd - d_true) <= eps * d_true + pair_tol), f"{what}: distance does not match its index"


def compare_counts_upto(orc, counts, limit: int, what: str = "") -> None:
    """Capped count (PAPER.md:L180-209 CountUpToN, reading A20): the definition is
    min(|row(q)|, limit); with the tolerance band, min(|sure|, limit) <= counts[q] <=
    min(|sure| + |band|, limit)."""
    o_off, _, o_band = orc
    o_off = np.asarray(o_off, dtype=np.int64)
    allc = np.diff(o_off)
    bandc = np.add.reduceat(np.concatenate([np.asarray(o_band, dtype=np.int64), [0]]),
                            np.minimum(o_off[:-1], len(o_band)))
    bandc = np.where(allc == 0, 0, bandc)
    counts = np.asarray(counts, dtype=np.int64)
    lo, hi = np.minimum(allc - bandc, limit), np.minimum(allc, limit)
    bad = (counts < lo) | (counts > hi)
    assert not bad.any(), f"{what}: {int(bad.sum())} capped counts outside [min(sure,L), min(sure+band,L)], first q={int(np.argmax(bad))}"


def compare_spatial_upto(n: int, orc, got, limit: int, what: str = "") -> None:
    """Capped storage query: every reported pair is a (sure or band) pair of the full oracle
    result, rows are duplicate-free, and row sizes obey the capped-count rule."""
    o_off, o_idx, _ = orc
    g_off, g_idx = got
    nq = len(o_off) - 1
    check_csr_format(g_off, g_idx, n, nq)
    ko = _keys(o_off, o_idx, n)
    kg = np.sort(_keys(g_off, g_idx, n))
    assert np.all(np.diff(kg) > 0), f"{what}: duplicate index inside a row"
    extra = ~np.isin(kg, ko, assume_unique=True)
    assert not extra.any(), f"{what}: {int(extra.sum())} reported pairs are not matches"
    compare_counts_upto(orc, np.diff(np.asarray(g_off, dtype=np.int64)), limit, what)


def compare_pairs(n: int, orc, got, what: str = "") -> dict:
    """Self-join: orc = oracle.spatial(points, POINT, (points, r), SPHERE), i.e.
    the full symmetric neighbour lists INCLUDING the self matches; got = (offsets[n+1], indices)
    where every unordered pair {i,j}, i != j, within r must appear exactly once in either row."""
    o_off, o_idx, o_band = orc
    g_off, g_idx = got
    check_csr_format(g_off, g_idx, n, n)
    rows_o = np.repeat(np.arange(n, dtype=np.int64), np.diff(np.asarray(o_off, dtype=np.int64)))
    oi = np.asarray(o_idx, dtype=np.int64)
    up = rows_o < oi                                        # each unordered pair once, self matches dropped
    ko = rows_o[up] * n + oi[up]
    sure = ko[np.asarray(o_band)[up] == 0]
    rows_g = np.repeat(np.arange(n, dtype=np.int64), np.diff(np.asarray(g_off, dtype=np.int64)))
    gi = np.asarray(g_idx, dtype=np.int64)
    assert not np.any(rows_g == gi), f"{what}: a primitive is paired with itself"
    kg = np.sort(np.minimum(rows_g, gi) * n + np.maximum(rows_g, gi))
    assert np.all(np.diff(kg) > 0), f"{what}: an unordered pair is reported more than once"
    assert np.isin(sure, kg, assume_unique=True).all(), f"{what}: a sure pair is missing"
    assert np.isin(kg, ko, assume_unique=True).all(), f"{what}: a reported pair is not within the radius"
    return dict(pairs=int(len(kg)), sure=int(len(sure)))


def compare_dbscan(orc, labels, what: str = "") -> dict:
    """orc = oracle.dbscan(...); labels = int32[n] with -1 = noise.  The core partition must
    be the same up to renaming; a border point must carry the label of one of its adjacent
    cores' clusters; noise must be -1.  (Use inputs without band pairs: orc[3] False.)"""
    core, comp, allowed, band_any = orc
    assert not band_any, f"{what}: choose eps so that no pair sits in the tolerance band"
    labels = np.asarray(labels, dtype=np.int64)
    n = len(core)
    assert labels.shape == (n,)
    lc, cc = labels[core], comp[core]
    assert np.all(lc >= 0), f"{what}: a core point is labelled noise"
    # bijection between oracle components and reported labels on the core points
    pairs = np.unique(np.stack([cc, lc], axis=1), axis=0)
    assert len(np.unique(pairs[:, 0])) == len(pairs) == len(np.unique(pairs[:, 1])), f"{what}: core partition differs"
    to_label = {int(c): int(l) for c, l in pairs}
    nborder = 0
    for i in np.nonzero(~core)[0]:
        if allowed[i]:
            nborder += 1
            assert int(labels[i]) in {to_label[c] for c in allowed[i]}, f"{what}: border point {i} has a foreign label"
        else:
            assert labels[i] == -1, f"{what}: noise point {i} has label {labels[i]}"
    return dict(clusters=len(pairs), core=int(core.sum()), border=nborder, noise=int(n - core.sum() - nborder))


def compare_knn_var(prims, pkind: int, qpoints, kq, kmax: int, orc, got, eps: float = EPS, what: str = "") -> None:
    """Per-query k: orc / got are rows of kmax entries.  Queries are grouped by their k_q; the
    first k_q columns of each group go through compare_knn with k = k_q, and every later column
    must be padding (-1 / +inf)."""
    o_idx, o_d = orc
    g_idx, g_d = got
    g_idx = np.asarray(g_idx)
    nq = o_idx.shape[0]
    assert g_idx.shape == (nq, kmax), f"{what}: shape {g_idx.shape} != {(nq, kmax)}"
    kq = np.clip(np.asarray(kq, dtype=np.int64), 0, kmax)
    cols = np.arange(kmax)[None, :]
    pad = cols >= kq[:, None]
    assert np.all(g_idx[pad] == -1), f"{what}: entries past k_q must be -1"
    if g_d is not None:
        assert np.all(np.isposinf(np.asarray(g_d)[pad])), f"{what}: distances past k_q must be +inf"
    for kv in np.unique(kq):
        if kv == 0:
            continue
        sel = np.nonzero(kq == kv)[0]
        compare_knn(prims, pkind, np.ascontiguousarray(qpoints[sel]), int(kv),
                    (np.ascontiguousarray(o_idx[sel, :kv]), np.ascontiguousarray(o_d[sel, :kv])),
                    (np.ascontiguousarray(g_idx[sel, :kv]), None if g_d is None else np.ascontiguousarray(np.asarray(g_d)[sel, :kv])),
                    eps=eps, what=f"{what} k_q={kv}")
