"""Pins for the oracle (CPU only): the oracle is checked against what the mathematics fixes,
never against itself alone.  SURVEY.md §8(c-5) P1..P12; BASELINE.json north_star."""
import itertools
import os

import numpy as np
import pytest

from paper_2507_23700_b200 import datagen as dg

GOLD = os.path.join(os.path.dirname(__file__), "golden", "lattice_closed_forms.txt")


def _golden():
    interior, totals = {}, {}
    for line in open(GOLD):
        t = line.split()
        if not t or t[0].startswith("#"):
            continue
        if t[0] == "total":
            totals[(int(t[1]), int(t[2]))] = int(t[3])
        else:
            interior[(int(t[0]), int(t[1]))] = int(t[2])
    return interior, totals


def _modes(orc, prims, pkind, kind, r=None):
    """None = brute force, plus two grids with different cell sizes."""
    cell = orc.default_cell(prims, pkind, kind, r)
    return [None, orc.Grid(prims, pkind, cell), orc.Grid(prims, pkind, 0.37 * cell)]


@pytest.mark.parametrize("D,g", [(1, 10), (2, 6), (3, 5), (4, 4)])
def test_lattice_radius_one_counts_and_total(orc, D, g):
    # P2: count(x) = 1 + sum_a [(x_a>0) + (x_a<g-1)];  total = g^D + 2D g^(D-1) (g-1)
    _, totals = _golden()
    p = dg.lattice_points(g, D)
    q = dg.sphere_queries(p, 1.0)
    expect = 1 + (p > 0).sum(1) + (p < g - 1).sum(1)
    for grid in _modes(orc, p, dg.POINT, "spatial", 1.0):
        off, idx, band = orc.spatial(p, dg.POINT, q, dg.SPHERE, grid)
        assert np.array_equal(np.diff(off), expect)
        assert int(off[-1]) == totals[(D, g)]
        # neighbours are exactly self and the axis neighbours (L2, closed, self included)
        rows = np.repeat(np.arange(len(p)), np.diff(off))
        d1 = np.abs(p[rows] - p[idx]).sum(1)
        assert set(np.unique(d1)) <= {0.0, 1.0}
        # pairs at exactly d = r are flagged as band, the self pair is not
        assert np.array_equal(band == 1, d1 == 1.0)


@pytest.mark.parametrize("D,r", [(1, 1), (1, 2), (2, 1), (2, 2), (3, 1), (3, 2), (3, 3), (4, 1), (4, 2)])
def test_lattice_interior_counts(orc, D, r):
    interior, _ = _golden()
    g = 2 * r + 3
    p = dg.lattice_points(g, D)
    centre = np.full((1, D), r + 1, dtype=np.float32)
    q = dg.sphere_queries(centre, float(r))
    for grid in _modes(orc, p, dg.POINT, "spatial", float(r)):
        off, idx, _ = orc.spatial(p, dg.POINT, q, dg.SPHERE, grid)
        assert int(off[-1]) == interior[(D, r)]
    # L-infinity or L1 norms would give (2r+1)^D or the cross-polytope count instead
    if D == 3 and r == 2:
        assert interior[(D, r)] not in (125, 25)


@pytest.mark.parametrize("D", [1, 2, 3])
def test_lattice_knn(orc, D):
    # P2': k = 2D+1 at interior points -> self + 2D axis neighbours, distances (0,1,...,1)
    g = 5
    p = dg.lattice_points(g, D)
    interior = np.all((p > 0) & (p < g - 1), axis=1)
    qp = p[interior]
    k = 2 * D + 1
    for grid in _modes(orc, p, dg.POINT, "knn"):
        idx, d = orc.knn(p, dg.POINT, qp, k, grid)
        assert np.array_equal(idx[:, 0], np.nonzero(interior)[0])
        assert np.all(d[:, 0] == 0.0) and np.all(d[:, 1:] == 1.0)
        l1 = np.abs(p[idx] - qp[:, None, :]).sum(2)
        assert np.all(l1[:, 1:] == 1.0)
        # k = 1 with queries = points -> self at distance exactly 0
        i1, d1 = orc.knn(p, dg.POINT, p, 1, grid)
        assert np.array_equal(i1[:, 0], np.arange(len(p))) and np.all(d1 == 0.0)


@pytest.mark.parametrize("D", [1, 2, 3])
def test_box_lattice(orc, D):
    # P3: unit cells as boxes; touching counts (closed sets)
    g = 5
    cells = dg.lattice_cells(g, D)
    z = np.full(D, 2, dtype=np.float32)
    q_cell = np.concatenate([z, z + 1])[None, :]
    q_shrunk = np.concatenate([z + 0.25, z + 0.75])[None, :]
    for grid in _modes(orc, cells, dg.BOX, "spatial"):
        off, _, band = orc.spatial(cells, dg.BOX, q_cell, dg.BOX, grid)
        assert int(off[-1]) == 3 ** D and not band.any()
        off, idx, _ = orc.spatial(cells, dg.BOX, q_shrunk, dg.BOX, grid)
        assert int(off[-1]) == 1
        off, _, _ = orc.spatial(cells, dg.BOX, (z + 0.5)[None, :], dg.POINT, grid)
        assert int(off[-1]) == 1
        off, _, _ = orc.spatial(cells, dg.BOX, z[None, :], dg.POINT, grid)
        assert int(off[-1]) == 2 ** D
        # kNN to boxes: the containing cell is at distance 0, face neighbours at 0.5
        qi, qd = orc.knn(cells, dg.BOX, (z + 0.5)[None, :], 1 + 2 * D, grid)
        assert qd[0, 0] == 0.0 and np.all(qd[0, 1:] == 0.5)


def test_one_dimensional_searchsorted(orc):
    # P12: in 1-D a radius search is two binary searches on the sorted coordinates
    rs = dg.rng(7)
    x = np.sort(rs.random(5000).astype(np.float32))
    s = rs.random(700).astype(np.float32)
    r = np.float32(0.003)
    q = dg.sphere_queries(s[:, None], r)
    # closed ball in exact arithmetic on the fp32 inputs
    lo = np.searchsorted(x.astype(np.float64), s.astype(np.float64) - np.float64(r), "left")
    hi = np.searchsorted(x.astype(np.float64), s.astype(np.float64) + np.float64(r), "right")
    for grid in _modes(orc, x[:, None], dg.POINT, "spatial", float(r)):
        off, idx, band = orc.spatial(x[:, None], dg.POINT, q, dg.SPHERE, grid)
        sure = np.diff(off) - np.add.reduceat(np.append(band, 0).astype(np.int64), np.minimum(off[:-1], len(band))) * (np.diff(off) > 0)
        assert np.all(sure <= hi - lo) and np.all(hi - lo <= np.diff(off))
        nb = band == 0
        rows = np.repeat(np.arange(len(s)), np.diff(off))
        assert np.all(idx[nb] >= lo[rows[nb]]) and np.all(idx[nb] < hi[rows[nb]])
    # kNN in 1-D: the k nearest of a sorted array form a contiguous window
    k = 5
    i_b, d_b = orc.knn(x[:, None], dg.POINT, s[:, None], k)
    ref = np.sort(np.abs(x[None, :].astype(np.float64) - s[:, None].astype(np.float64)), axis=1)[:, :k]
    assert np.array_equal(d_b, ref)
    srt = np.sort(i_b, axis=1)
    assert np.all(srt[:, -1] - srt[:, 0] == k - 1)


KINDS = [dg.POINT, dg.BOX, dg.SPHERE]


def _rand_prims(kind, n, D, seed):
    if kind == dg.POINT:
        return dg.uniform_points(n, D, seed)
    if kind == dg.BOX:
        return dg.uniform_boxes(n, D, seed, 0.5 * n ** (-1.0 / D))
    return dg.uniform_spheres(n, D, seed, 0.7 * n ** (-1.0 / D))


def _naive_predicate(q, qkind, p, pkind, D):
    """Independent, per-pair python restatement of SURVEY §8(c-1) used on tiny inputs only."""
    q = q.astype(np.float64); p = p.astype(np.float64)

    def pb(x, lo, hi):
        return float((np.maximum(0, np.maximum(lo - x, x - hi)) ** 2).sum())
    if qkind == dg.SPHERE:
        s, r = q[:D], q[D]
        if pkind == dg.POINT: return ((p - s) ** 2).sum(), r * r
        if pkind == dg.BOX: return pb(s, p[:D], p[D:]), r * r
        return ((p[:D] - s) ** 2).sum(), (r + p[D]) ** 2
    if qkind == dg.BOX:
        if pkind == dg.POINT: return float(not np.all((q[:D] <= p) & (p <= q[D:]))), 0.5
        if pkind == dg.BOX: return float(not np.all((p[:D] <= q[D:]) & (q[:D] <= p[D:]))), 0.5
        return pb(p[:D], q[:D], q[D:]), p[D] ** 2
    if pkind == dg.POINT: return float(not np.all(p == q)), 0.5
    if pkind == dg.BOX: return float(not np.all((p[:D] <= q) & (q <= p[D:]))), 0.5
    return ((q - p[:D]) ** 2).sum(), p[D] ** 2


@pytest.mark.parametrize("pkind,qkind", list(itertools.product(KINDS, KINDS)))
def test_bruteforce_matches_naive_python(orc, pkind, qkind):
    # P1 on tiny inputs: C++ brute force == per-pair python loop of the definition table
    D, n, nq = 2, 60, 40
    p = _rand_prims(pkind, n, D, 3)
    q = _rand_prims(qkind, nq, D, 4)
    if qkind == dg.SPHERE:
        q[:, D] *= 2.0
    if qkind == dg.POINT and pkind == dg.POINT:
        q[:10] = p[:10]
    off, idx, band = orc.spatial(p, pkind, q, qkind)
    for j in range(nq):
        got = set(idx[off[j]:off[j + 1]][band[off[j]:off[j + 1]] == 0].tolist())
        exp = set()
        for i in range(n):
            t, T = _naive_predicate(q[j], qkind, p[i], pkind, D)
            if t < T * (1 - 1e-6):
                exp.add(i)
        assert got == exp, (pkind, qkind, j)


@pytest.mark.parametrize("D", [1, 2, 3, 5])
@pytest.mark.parametrize("pkind", KINDS)
def test_grid_equals_bruteforce(orc, D, pkind):
    # P1/P11: Mode B must reproduce Mode A exactly (both fp64, same predicate)
    n, nq = 1500, 300
    p = _rand_prims(pkind, n, D, 10 + D)
    for qkind in KINDS:
        q = _rand_prims(qkind, nq, D, 20 + D)
        if qkind == dg.SPHERE:
            q[:, D] = np.float32(1.2 * n ** (-1.0 / D))
        rr = float(q[0, D]) if qkind == dg.SPHERE else None
        a = orc.spatial(p, pkind, q, qkind)
        for grid in _modes(orc, p, pkind, "spatial", rr)[1:]:
            b = orc.spatial(p, pkind, q, qkind, grid)
            for x, y in zip(a, b):
                assert np.array_equal(x, y), (D, pkind, qkind)
    qp = dg.uniform_points(nq, D, 30 + D)
    qp[::7] = qp[::7] * 3.0 - 1.0          # some queries far outside the scene
    for k in (1, 4, 9):
        ia, da = orc.knn(p, pkind, qp, k)
        for grid in _modes(orc, p, pkind, "knn")[1:]:
            ib, db = orc.knn(p, pkind, qp, k, grid)
            assert np.array_equal(da, db) and np.array_equal(ia, ib), (D, pkind, k)


def test_symmetry_and_monotonicity(orc):
    # P5: i in row(j) <=> j in row(i) for a point self-search;  P7: r1<r2 => rows nested
    p = dg.uniform_points(2000, 3, 5)
    n = len(p)
    r1, r2 = 0.05, 0.08
    o1 = orc.spatial(p, dg.POINT, dg.sphere_queries(p, r1), dg.SPHERE)
    o2 = orc.spatial(p, dg.POINT, dg.sphere_queries(p, r2), dg.SPHERE)
    k1 = np.repeat(np.arange(n), np.diff(o1[0])) * n + o1[1]
    kt = o1[1].astype(np.int64) * n + np.repeat(np.arange(n), np.diff(o1[0]))
    assert np.array_equal(np.sort(k1), np.sort(kt))
    k2 = np.repeat(np.arange(n), np.diff(o2[0])) * n + o2[1]
    assert np.isin(k1, k2).all() and len(k2) > len(k1)
    # huge r: every row is [0, n)
    o3 = orc.spatial(p[:200], dg.POINT, dg.sphere_queries(p[:50], 10.0), dg.SPHERE)
    assert np.array_equal(np.diff(o3[0]), np.full(50, 200))
    # P8 (sanity): mean count ~ rho * V(r) * (1 - 1.125 r) in the unit cube
    m = len(k1) / n
    expect = 1 + n * 4 / 3 * np.pi * r1 ** 3 * (1 - 1.125 * r1)   # +1: the self pair
    assert abs(m - expect) / expect < 0.1


def test_knn_radius_consistency_and_edges(orc):
    # P6: radius search at D_k(1+2eps) holds >= k hits incl. the kNN set; at D_k(1-2eps) < k
    p = dg.uniform_points(3000, 3, 8)
    qp = dg.uniform_points(100, 3, 9)
    k = 7
    idx, d = orc.knn(p, dg.POINT, qp, k)
    assert np.all(np.diff(d, axis=1) >= 0)
    for j in range(0, 100, 9):
        q_hi = dg.sphere_queries(qp[j:j + 1], 1.0)
        q_hi = q_hi.astype(np.float64)
        off, ind, band = orc.spatial(p, dg.POINT, dg.sphere_queries(qp[j:j + 1], d[j, -1] * (1 + 1e-5)), dg.SPHERE)
        assert set(idx[j].tolist()) <= set(ind.tolist())
        off, ind, band = orc.spatial(p, dg.POINT, dg.sphere_queries(qp[j:j + 1], d[j, -1] * (1 - 1e-5)), dg.SPHERE)
        assert len(ind) < k
    # A8: n < k pads with -1 / +inf;  n = 0 gives empty rows
    i2, d2 = orc.knn(p[:3], dg.POINT, qp[:5], 5)
    assert np.all(i2[:, 3:] == -1) and np.all(np.isinf(d2[:, 3:])) and np.all(i2[:, :3] >= 0)
    off, ind, _ = orc.spatial(p[:0], dg.POINT, dg.sphere_queries(qp[:5], 0.1), dg.SPHERE)
    assert np.array_equal(off, np.zeros(6, dtype=np.int64)) and len(ind) == 0
    # A21: negative radius matches nothing; r = 0 matches only coincident points (exact)
    off, _, _ = orc.spatial(p, dg.POINT, dg.sphere_queries(p[:10], -1.0), dg.SPHERE)
    assert int(off[-1]) == 0
    off, ind, band = orc.spatial(p, dg.POINT, dg.sphere_queries(p[:10], 0.0), dg.SPHERE)
    assert np.array_equal(ind, np.arange(10)) and not band.any()


def test_sphere_primitive_knn_distance(orc):
    # A4: distance to a sphere primitive is max(0, |y-c| - R); worked by hand
    s = np.array([[0, 0, 0, 1.0], [10, 0, 0, 2.0]], dtype=np.float32)
    y = np.array([[3, 4, 0], [0.5, 0, 0], [9, 0, 0]], dtype=np.float32)
    idx, d = orc.knn(s, dg.SPHERE, y, 2)
    assert np.allclose(d[0], [4.0, np.sqrt(49 + 16) - 2.0])
    assert idx[1, 0] == 0 and d[1, 0] == 0.0
    assert idx[2, 0] == 1 and d[2, 0] == 0.0 and np.isclose(d[2, 1], 8.0)
    # box primitive: 0 inside, Euclidean to the nearest face/corner outside
    b = np.array([[0, 0, 0, 1, 1, 1]], dtype=np.float32)
    _, d = orc.knn(b, dg.BOX, np.array([[0.5, 0.5, 0.5], [2, 2, 1]], dtype=np.float32), 1)
    assert d[0, 0] == 0.0 and np.isclose(d[1, 0], np.sqrt(2.0))


def test_capped_count_comparator_is_min_of_definition(orc):
    """compare_counts_upto accepts exactly min(|row|, limit) on an exact-predicate case and
    rejects an off-by-one (the CountUpToN example's min(total, n+1), reading A20)."""
    from oracle import compare as cmp
    from paper_2507_23700_b200 import datagen as dg
    cells = dg.lattice_cells(5, 2)
    o = orc.spatial(cells, dg.BOX, cells, dg.BOX)
    rows = np.diff(o[0])
    assert rows.max() == 9 and rows.min() == 4                # 3^2 interior, 2^2 corners (touching counts)
    for limit in (1, 4, 6, 20):
        cmp.compare_counts_upto(o, np.minimum(rows, limit), limit)
    with pytest.raises(AssertionError):
        cmp.compare_counts_upto(o, np.minimum(rows, 6 + 1), 6)


def test_pair_comparator_closed_form(orc):
    """compare_pairs on a lattice: r = 1.2 gives exactly the 3 g^2 (g-1) axis-neighbour pairs (all
    clear of the tolerance band); it rejects a duplicated pair, a self pair and a missing pair."""
    from oracle import compare as cmp
    from paper_2507_23700_b200 import datagen as dg
    g = 4
    p = dg.lattice_points(g, 3)
    n = len(p)
    o = orc.spatial(p, dg.POINT, dg.sphere_queries(p, 1.2), dg.SPHERE)
    assert not o[2].any()
    rows = np.repeat(np.arange(n), np.diff(o[0]))
    up = rows < o[1]
    a, b = rows[up], o[1][up]
    assert len(a) == 3 * g * g * (g - 1)
    order = np.argsort(a, kind="stable")
    off = np.concatenate([[0], np.cumsum(np.bincount(a, minlength=n))])
    good = (off, b[order].astype(np.int32))
    assert cmp.compare_pairs(n, o, good)["pairs"] == len(a)
    flipped = (np.concatenate([[0], np.cumsum(np.bincount(b, minlength=n))]), a[np.argsort(b, kind="stable")].astype(np.int32))
    cmp.compare_pairs(n, o, flipped)                          # the other endpoint may own the pair
    both = (o[0], o[1])                                       # full symmetric lists: pairs twice + self
    with pytest.raises(AssertionError):
        cmp.compare_pairs(n, o, both)
    with pytest.raises(AssertionError):
        cmp.compare_pairs(n, o, (np.maximum(off - (off > 0), 0), good[1][1:]))   # one pair dropped


def test_dbscan_oracle_closed_forms(orc):
    """DBSCAN oracle on cases with a known answer: a 1-D chain (ends are border points), two far
    apart blobs, and isolated points (noise)."""
    from oracle import compare as cmp
    chain = np.zeros((7, 2), np.float32)
    chain[:, 0] = np.arange(7)                                 # 0..6 on a line, spacing 1
    iso = np.float32([[100, 100], [200, 200]])
    pts = np.concatenate([chain, chain + np.float32([0, 50]), iso])
    core, comp, allowed, band = orc.dbscan(pts, 1.25, 3)       # each inner point sees itself + 2 neighbours
    assert not band
    assert core.tolist() == [False, True, True, True, True, True, False] * 2 + [False, False]
    assert len(set(comp[core].tolist())) == 2                   # two clusters
    assert allowed[0] == {int(comp[1])} and allowed[6] == {int(comp[5])}   # chain ends are border points
    assert allowed[14] == set() and allowed[15] == set()        # isolated points are noise
    labels = np.array([1, 1, 1, 1, 1, 1, 1, 8, 8, 8, 8, 8, 8, 8, -1, -1])
    st = cmp.compare_dbscan((core, comp, allowed, band), labels)
    assert st == dict(clusters=2, core=10, border=4, noise=2)
    bad = labels.copy(); bad[7:14] = 1                          # merging the two clusters must be rejected
    with pytest.raises(AssertionError):
        cmp.compare_dbscan((core, comp, allowed, band), bad)
    bad = labels.copy(); bad[0] = -1                            # a border point may not be noise
    with pytest.raises(AssertionError):
        cmp.compare_dbscan((core, comp, allowed, band), bad)


# ---- hand-worked cases for every cell of the predicate table ---------------------------------------
CELLS = os.path.join(os.path.dirname(__file__), "golden", "predicate_cells.txt")
_KIND = {"P": dg.POINT, "B": dg.BOX, "S": dg.SPHERE}
_ARITH = {("S", "P"), ("S", "B"), ("S", "S"), ("B", "S"), ("P", "S")}   # predicates with arithmetic (a band exists)


def _cell_cases():
    out = []
    for ln, line in enumerate(open(CELLS), 1):
        line = line.split("#")[0].strip()
        if not line:
            continue
        head, q, p, expect = [t.strip() for t in line.split("|")]
        qk, pk, D = head.split()
        out.append(pytest.param(qk, pk, int(D), np.float32(q.split()), np.float32(p.split()), expect,
                                id=f"L{ln}-{qk}x{pk}-D{D}-{expect}"))
    return out


@pytest.mark.parametrize("qk,pk,D,q,p,expect", _cell_cases())
def test_predicate_cells_hand_worked(orc, qk, pk, D, q, p, expect):
    """tests/golden/predicate_cells.txt: one hit, one miss and one exactly-touching pair (and the
    mirrored / single-axis variants) for every (query kind x primitive kind) cell, D in {1,3}.
    Checked in brute force and through the grid (alone and among far-away decoys)."""
    width = {"P": D, "B": 2 * D, "S": D + 1}
    assert len(q) == width[qk] and len(p) == width[pk]
    decoys = np.tile(p, (5, 1))
    decoys[:, :D] += np.float32(1000.0) * np.arange(1, 6, dtype=np.float32)[:, None]   # far away on every axis
    if pk == "B":
        decoys[:, D:] += np.float32(1000.0) * np.arange(1, 6, dtype=np.float32)[:, None]
    many = np.concatenate([decoys[:2], p[None, :], decoys[2:]])
    for prims, at in ((p[None, :], 0), (many, 2)):
        for grid in [None, orc.Grid(prims, _KIND[pk], 1.0), orc.Grid(prims, _KIND[pk], 0.3)]:
            off, idx, band = orc.spatial(prims, _KIND[pk], q[None, :], _KIND[qk], grid)
            if expect == "miss":
                assert int(off[-1]) == 0, "a miss was reported"
                continue
            assert idx.tolist() == [at], "the match is missing"
            T_is_zero = (qk == "S" and pk != "S" and q[D] == 0) or (pk == "S" and qk != "S" and p[D] == 0)
            want_band = expect == "touch" and (qk, pk) in _ARITH and not T_is_zero
            assert bool(band[0]) == want_band, "boundary pair must be flagged iff the predicate has arithmetic"


@pytest.mark.parametrize("D", [1, 2, 3])
def test_unit_cells_queried_by_half_radius_sphere(orc, D):
    """SPHERE query x BOX primitives on the unit-cell lattice: a ball of radius 1/2 at a cell
    centre holds the cell itself (distance 0) and touches its 2D face neighbours at exactly
    1/2; edge neighbours are at sqrt(2)/2 > 1/2."""
    g = 5
    cells = dg.lattice_cells(g, D)
    q = np.float32([[2.5] * D + [0.5]])
    for grid in _modes(orc, cells, dg.BOX, "spatial", 0.5):
        off, idx, band = orc.spatial(cells, dg.BOX, q, dg.SPHERE, grid)
        assert int(off[-1]) == 1 + 2 * D and int(band.sum()) == 2 * D
        own = idx[band == 0]
        assert len(own) == 1 and np.array_equal(cells[own[0], :D], np.full(D, 2.0, np.float32))
        l1 = np.abs(cells[idx[band == 1], :D] - 2.0).sum(1)
        assert np.all(l1 == 1.0)
    # radius 3/4: a neighbour cell offset on j axes is at distance sqrt(j)/2 -> the 2D face cells
    # (0.5) and the 2D(D-1) edge cells (0.707) are inside, the corner cells (0.866) are not
    q2 = np.float32([[2.5] * D + [0.75]])
    off, idx, band = orc.spatial(cells, dg.BOX, q2, dg.SPHERE)
    expect = 1 + 2 * D + (2 * D * (D - 1) if D >= 2 else 0)
    assert int(off[-1]) == expect and not band.any()


# ---- the comparators reject wrong answers --------------------------------------------------------------
def _small_spatial(orc):
    p = dg.uniform_points(400, 3, 1)
    q = dg.sphere_queries(dg.uniform_points(60, 3, 2), 0.2)
    o = orc.spatial(p, dg.POINT, q, dg.SPHERE)
    assert not o[2].any() and int(o[0][-1]) > 200
    return p, q, o


def test_compare_spatial_and_counts_reject_corruption(orc):
    from oracle import compare as cmp
    p, q, o = _small_spatial(orc)
    n = len(p)
    off, idx = o[0].copy(), o[1].copy()
    cmp.compare_spatial(n, o, (off, idx))                          # the oracle's own answer passes
    cmp.compare_counts(o, np.diff(off))
    g = dg.rng(5)
    shuffled = idx.copy()
    for j in range(len(off) - 1):                                  # order inside a row is free
        shuffled[off[j]:off[j + 1]] = g.permutation(shuffled[off[j]:off[j + 1]])
    cmp.compare_spatial(n, o, (off, shuffled))
    row = int(np.argmax(np.diff(off) >= 2))
    # a dropped pair
    o2 = off.copy(); o2[row + 1:] -= 1
    with pytest.raises(AssertionError, match="missing"):
        cmp.compare_spatial(n, o, (o2, np.delete(idx, off[row])))
    # a foreign index (a primitive that does not match) in place of a real one
    foreign = np.setdiff1d(np.arange(n), idx[off[row]:off[row + 1]])[0]
    bad = idx.copy(); bad[off[row]] = foreign
    with pytest.raises(AssertionError):
        cmp.compare_spatial(n, o, (off, bad))
    # an extra pair
    o3 = off.copy(); o3[row + 1:] += 1
    with pytest.raises(AssertionError, match="neither sure nor band"):
        cmp.compare_spatial(n, o, (o3, np.insert(idx, off[row], foreign)))
    # a duplicated index inside a row
    dup = idx.copy(); dup[off[row]] = dup[off[row] + 1]
    with pytest.raises(AssertionError):
        cmp.compare_spatial(n, o, (off, dup))
    # an index out of range, offsets that do not start at 0 / decrease / disagree with len(indices)
    oob = idx.copy(); oob[0] = n
    with pytest.raises(AssertionError):
        cmp.compare_spatial(n, o, (off, oob))
    with pytest.raises(AssertionError):
        cmp.compare_spatial(n, o, (off + 1, idx))
    with pytest.raises(AssertionError):
        cmp.compare_spatial(n, o, (off, idx[:-1]))
    # counts off by one in either direction
    for delta in (+1, -1):
        c = np.diff(off).copy(); c[row] += delta
        with pytest.raises(AssertionError, match="counts outside"):
            cmp.compare_counts(o, c)


def test_compare_spatial_band_pairs_are_optional_but_nothing_else(orc):
    from oracle import compare as cmp
    p = dg.lattice_points(4, 3)
    q = dg.sphere_queries(p, 1.0)                                  # axis neighbours sit exactly at d = r: band
    o = orc.spatial(p, dg.POINT, q, dg.SPHERE)
    n = len(p)
    assert o[2].sum() == 2 * 3 * 16 * 3 and (o[2] == 0).sum() == n
    cmp.compare_spatial(n, o, (o[0], o[1]))                        # with every band pair
    only_self = (np.arange(n + 1, dtype=np.int64), np.arange(n, dtype=np.int32))
    cmp.compare_spatial(n, o, only_self)                           # with none of them
    cmp.compare_counts(o, np.ones(n, dtype=np.int64))
    with pytest.raises(AssertionError):
        cmp.compare_counts(o, np.zeros(n, dtype=np.int64))         # the sure (self) pair is not optional
    with pytest.raises(AssertionError):
        cmp.compare_counts(o, np.diff(o[0]) + 1)


def test_compare_knn_rejects_corruption(orc):
    from oracle import compare as cmp
    p = dg.uniform_points(500, 3, 3)
    qp = dg.uniform_points(40, 3, 4)
    k = 6
    o = orc.knn(p, dg.POINT, qp, k)
    gi, gd = o[0].copy(), o[1].astype(np.float32)
    cmp.compare_knn(p, dg.POINT, qp, k, o, (gi, gd))               # fp32-rounded oracle answer passes
    cmp.compare_knn(p, dg.POINT, qp, k, o, (gi, None))             # distances are optional
    # a distance off by 5e-6 relative
    bad = gd.copy(); bad[3, 2] = np.float32(bad[3, 2] * (1 + 5e-6))
    with pytest.raises(AssertionError):
        cmp.compare_knn(p, dg.POINT, qp, k, o, (gi, bad))
    # a wrong neighbour (a far primitive) with the right distance column
    far = int(np.argmax(((p - qp[5]) ** 2).sum(1)))
    wi = gi.copy(); wi[5, k - 1] = far
    with pytest.raises(AssertionError):
        cmp.compare_knn(p, dg.POINT, qp, k, o, (wi, gd))
    with pytest.raises(AssertionError):
        cmp.compare_knn(p, dg.POINT, qp, k, o, (wi, None))
    # a duplicate neighbour
    di = gi.copy(); di[7, 1] = di[7, 0]
    with pytest.raises(AssertionError, match="duplicate"):
        cmp.compare_knn(p, dg.POINT, qp, k, o, (di, gd))
    # the (k+1)-th neighbour in place of the k-th (clearly farther than D_k)
    o7 = orc.knn(p, dg.POINT, qp, k + 1)
    assert np.all(o7[1][:, k] > o7[1][:, k - 1] * (1 + 1e-5))
    si = gi.copy(); si[:, k - 1] = o7[0][:, k]
    sd = gd.copy(); sd[:, k - 1] = o7[1][:, k]
    with pytest.raises(AssertionError):
        cmp.compare_knn(p, dg.POINT, qp, k, o, (si, sd))
    # descending rows, an invalid index, padding where none is due
    with pytest.raises(AssertionError):
        cmp.compare_knn(p, dg.POINT, qp, k, o, (gi[:, ::-1].copy(), gd[:, ::-1].copy()))
    ii = gi.copy(); ii[0, 0] = -1
    with pytest.raises(AssertionError):
        cmp.compare_knn(p, dg.POINT, qp, k, o, (ii, gd))
    # n < k: padding is required
    o3 = orc.knn(p[:4], dg.POINT, qp, k)
    cmp.compare_knn(p[:4], dg.POINT, qp, k, o3, (o3[0], o3[1].astype(np.float32)))
    np_ = o3[0].copy(); np_[:, 4:] = 0
    with pytest.raises(AssertionError, match="padding"):
        cmp.compare_knn(p[:4], dg.POINT, qp, k, o3, (np_, o3[1].astype(np.float32)))


def test_compare_knn_sphere_tolerance_is_per_pair(orc):
    """Sphere primitives: fp32 ||y-c|| - R cancels, so compare_knn widens the tolerance by the
    per-pair bound 2^-21 (d + 2R) and by nothing more."""
    from oracle import compare as cmp
    s = np.float32([[0, 0, 0, 1000.0], [3000, 0, 0, 1.0], [0, 5000, 0, 2.0]])
    y = np.float32([[1000.5, 0, 0]])                               # 0.5 outside a sphere of radius 1000
    o = orc.knn(s, dg.SPHERE, y, 3)
    assert o[0][0].tolist() == [0, 1, 2] and o[1][0, 0] == 0.5
    gd = o[1].astype(np.float32)
    ok = gd.copy(); ok[0, 0] = np.float32(0.5 + 2.0 ** -21 * 2000.0)       # inside the cancellation bound
    cmp.compare_knn(s, dg.SPHERE, y, 3, o, (o[0], ok))
    bad = gd.copy(); bad[0, 0] = np.float32(0.5 + 2.0 ** -21 * 2100.0 + 1e-6)
    with pytest.raises(AssertionError):
        cmp.compare_knn(s, dg.SPHERE, y, 3, o, (o[0], bad))
    bad2 = gd.copy(); bad2[0, 1] = np.float32(bad2[0, 1] * (1 + 4e-6))      # 4e-6 relative is far outside eps + slack
    with pytest.raises(AssertionError):
        cmp.compare_knn(s, dg.SPHERE, y, 3, o, (o[0], bad2))


# ---- NEXT-4: one k per query -----------------------------------------------------------
def test_knn_var_lattice_closed_form(orc):
    """Integer lattice, queries on interior lattice points: k_q = 0 -> an empty (padded) row;
    k_q = 1 -> the point itself at distance 0; k_q = 2D+1 -> itself + its 2D axis neighbours at
    distance exactly 1; k_q > kmax is clamped to kmax.  (Worked by hand: the 2D neighbours
    p +- e_a are the only lattice points at distance 1, the next shell is at sqrt(2).)"""
    from paper_2507_23700_b200 import datagen as dg
    for D, g in ((1, 30), (2, 9), (3, 7)):
        p = dg.lattice_points(g, D)
        interior = np.nonzero(np.all((p > 0) & (p < g - 1), axis=1))[0]
        qp = p[interior]
        kmax = 2 * D + 1
        kq = np.array([[0, 1, kmax, kmax + 5][i % 4] for i in range(len(interior))], dtype=np.int32)
        idx, dist = orc.knn_var(p, orc.POINT, qp, kq, kmax)
        for r, (qi, kk) in enumerate(zip(interior, kq)):
            kk = min(int(kk), kmax)
            assert np.all(idx[r, kk:] == -1) and np.all(np.isposinf(dist[r, kk:]))
            if kk >= 1:
                assert idx[r, 0] == qi and dist[r, 0] == 0.0
            if kk == kmax:
                assert np.all(dist[r, 1:] == 1.0)
                assert np.all(np.abs(p[idx[r, 1:]] - qp[r]).sum(axis=1) == 1)


def test_compare_knn_var_rejects_corruption(orc):
    from oracle import compare as cmp
    from paper_2507_23700_b200 import datagen as dg
    p = dg.uniform_points(400, 3, 5)
    qp = dg.uniform_points(50, 3, 6)
    kmax = 6
    kq = (np.arange(50) % (kmax + 1)).astype(np.int32)
    o = orc.knn_var(p, orc.POINT, qp, kq, kmax)
    good = (o[0].copy(), o[1].astype(np.float32))
    cmp.compare_knn_var(p, orc.POINT, qp, kq, kmax, o, good, what="ok")
    bad_pad = (good[0].copy(), good[1].copy())
    r = int(np.nonzero(kq == 2)[0][0])
    bad_pad[0][r, 3] = 7                                     # an entry past k_q
    with pytest.raises(AssertionError):
        cmp.compare_knn_var(p, orc.POINT, qp, kq, kmax, o, bad_pad, what="pad")
    bad_row = (good[0].copy(), good[1].copy())
    r = int(np.nonzero(kq == 4)[0][0])
    far = int(np.argmax(np.linalg.norm(p - qp[r], axis=1)))
    bad_row[0][r, 3] = far                                   # a wrong neighbour inside the first k_q
    with pytest.raises(AssertionError):
        cmp.compare_knn_var(p, orc.POINT, qp, kq, kmax, o, bad_row, what="row")


# ---- NEXT-4: fp64 coordinates (oracle/f64.py) ---------------------------------------------------------
def test_f64_oracle_lattice_closed_forms():
    """The fp64 oracle against the lattice closed forms (worked by hand): radius 1 around an
    interior lattice point = itself + its 2D axis neighbours; radius 2 in 3-D = 33 points;
    k = 2D+1 nearest = the same 2D+1 points at distances 0 and 1."""
    from oracle import f64
    from paper_2507_23700_b200 import datagen as dg
    for D, g in ((1, 20), (2, 9), (3, 7)):
        p = dg.lattice_points(g, D).astype(np.float64)
        interior = np.nonzero(np.all((p > 0) & (p < g - 1), axis=1))[0]
        q = np.concatenate([p[interior], np.ones((len(interior), 1))], axis=1)
        off, idx, band = f64.spatial(p, f64.POINT, q, f64.SPHERE)
        assert np.all(np.diff(off) == 2 * D + 1)               # d^2 = 1 <= 1: closed (band or sure)
        ki, kd = f64.knn(p, f64.POINT, p[interior], 2 * D + 1)
        assert np.array_equal(ki[:, 0], interior) and np.all(kd[:, 0] == 0) and np.all(kd[:, 1:] == 1.0)
    p = dg.lattice_points(7, 3).astype(np.float64)
    c = np.array([[3.0, 3.0, 3.0, 2.0]])
    assert np.diff(f64.spatial(p, f64.POINT, c, f64.SPHERE)[0])[0] == 33


@pytest.mark.parametrize("pk", [0, 1, 2])
@pytest.mark.parametrize("qk", [0, 1, 2])
def test_f64_oracle_equals_cpp_oracle_on_fp32_inputs(orc, pk, qk):
    """On inputs that are exactly representable in fp32 the two oracles do the same fp64
    arithmetic on the same numbers: rows, bands and kNN index rows must be identical, distances
    equal up to the order of the fp64 sums."""
    from oracle import f64
    from paper_2507_23700_b200 import datagen as dg
    D, n, nq = 3, 600, 150
    ext = 0.5 * (8.0 / n) ** (1.0 / D)
    p = {0: dg.uniform_points(n, D, 3), 1: dg.uniform_boxes(n, D, 3, ext), 2: dg.uniform_spheres(n, D, 3, ext)}[pk]
    qp = dg.uniform_points(nq, D, 4)
    q = {2: dg.sphere_queries(qp, ext * 1.4), 1: dg.uniform_boxes(nq, D, 5, ext),
         0: np.concatenate([qp[: nq // 2], p[: nq - nq // 2, :D]], axis=0)}[qk]
    a = orc.spatial(p, pk, q, qk)
    b = f64.spatial(p.astype(np.float64), pk, q.astype(np.float64), qk)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    ka = orc.knn(p, pk, qp, 7)
    kb = f64.knn(p.astype(np.float64), pk, qp.astype(np.float64), 7)
    assert np.array_equal(ka[0], kb[0])
    assert np.allclose(ka[1], kb[1], rtol=1e-13, atol=0.0)      # same numbers up to the order of the fp64 sums
