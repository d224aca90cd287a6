"""GPU parity tests (run on the B200 box): the CUDA path, called through the C ABI, against the
oracle on the same seeded inputs.  Protocol: SURVEY.md §8(c-3) / BASELINE.json north_star:
index sets bit-exact after per-query sorting outside the 1e-6 boundary band, counts exact,
kNN distances to 1e-6 relative, index sets equal except among ties."""
import os

import numpy as np
import pytest

from paper_2507_23700_b200 import datagen as dg

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def arbx():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2507_23700_b200 import binding
    binding.lib()   # fail loudly if the extension is missing
    return binding


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _np(t):
    return t.cpu().numpy()


def _spatial_case(arbx, orc, cmp, prims, pkind, queries, qkind, what, grid=None):
    ix = arbx.Index(_dev(prims), pkind, dim=dg_dim(prims, pkind))
    assert ix.validate() == 0, f"{what}: tree self-check failed"
    counts = _np(ix.query_count(_dev(queries), qkind))
    off, idx = ix.query_spatial(_dev(queries), qkind)
    off, idx = _np(off), _np(idx)
    ix.close()
    o = orc.spatial(prims, pkind, queries, qkind, grid)
    stats = cmp.compare_spatial(prims.shape[0], o, (off, idx), what)
    cmp.compare_counts(o, counts, what)
    assert np.array_equal(counts, np.diff(off)), f"{what}: count-only != diff(offsets)"
    return stats


def dg_dim(prims, pkind):
    w = prims.shape[1]
    return w if pkind == dg.POINT else w // 2 if pkind == dg.BOX else w - 1


def _make_prims(kind, n, D, seed, ext):
    if kind == dg.POINT:
        return dg.uniform_points(n, D, seed)
    if kind == dg.BOX:
        return dg.uniform_boxes(n, D, seed, ext)
    return dg.uniform_spheres(n, D, seed, ext)


# ---- B3: radix sort against numpy's stable sort --------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 255, 256, 257, 4095, 4096, 4097, 65536, (1 << 20) - 1, (1 << 20) + 1, 3_000_000])
@pytest.mark.parametrize("kbytes,bits", [(8, 64), (8, 63), (8, 40), (8, 39), (4, 32), (4, 30), (4, 9)])
def test_sort_pairs(arbx, n, kbytes, bits):
    g = dg.rng(n * 7 + bits)
    dt = np.uint64 if kbytes == 8 else np.uint32
    keys = g.integers(0, 1 << bits, size=n, dtype=np.uint64, endpoint=False).astype(dt)
    if n > 1000:   # duplicates and a skewed digit, to exercise stability and look-back
        keys[: n // 3] = keys[0]
        keys[n // 3: n // 2] &= dt(0xFF)
    vals = np.arange(n, dtype=np.uint32)[::-1].copy()
    tk = _dev(keys.view(np.int64 if kbytes == 8 else np.int32))
    tv = _dev(vals.view(np.int32))
    arbx.arbx_sort_pairs(tk, tv, bits)
    torch.cuda.synchronize()
    order = np.argsort(keys, kind="stable")
    assert np.array_equal(_np(tk).view(dt), keys[order])
    assert np.array_equal(_np(tv).view(np.uint32), vals[order])   # stable => unique answer


def test_sort_keys_only(arbx):
    g = dg.rng(5)
    keys = g.integers(0, 1 << 62, size=100_001, dtype=np.uint64)
    tk = _dev(keys.view(np.int64))
    arbx.arbx_sort_pairs(tk, None, 64)
    assert np.array_equal(_np(tk).view(np.uint64), np.sort(keys))


# ---- P1: every (dim, primitive kind, query kind) cell against brute force ---------------------------
@pytest.mark.parametrize("D", list(range(1, 11)))
@pytest.mark.parametrize("pkind", [dg.POINT, dg.BOX, dg.SPHERE])
def test_all_cells_small(arbx, orc, D, pkind):
    from oracle import compare as cmp
    n, nq = 1500, 700
    # sizes chosen so that the expected number of matches per query is O(1..30) in every D
    ext = 0.5 * (8.0 / n) ** (1.0 / D)
    prims = _make_prims(pkind, n, D, 10 + D, ext)
    qp = dg.uniform_points(nq, D, 20 + D)
    cases = [
        (dg.SPHERE, dg.sphere_queries(qp, ext * 1.3)),
        (dg.BOX, dg.uniform_boxes(nq, D, 30 + D, ext)),
        (dg.POINT, np.concatenate([qp[: nq // 2], prims[: nq - nq // 2, :D]], axis=0)),
    ]
    for qkind, q in cases:
        _spatial_case(arbx, orc, cmp, prims, pkind, q, qkind, f"D={D} pk={pkind} qk={qkind}")
    for k in (1, 5, 16, 40):
        ix = arbx.Index(_dev(prims), pkind, dim=D)
        gi, gd = ix.query_knn(_dev(qp), k)
        ix.close()
        o = orc.knn(prims, pkind, qp, k)
        cmp.compare_knn(prims, pkind, qp, k, o, (_np(gi), _np(gd)), what=f"knn D={D} pk={pkind} k={k}")


@pytest.mark.parametrize("leaf_max", [1, 2, 8, 64])
def test_leaf_sizes(arbx, orc, leaf_max, knobs):
    from oracle import compare as cmp
    knobs(leaf_max=leaf_max)
    prims = dg.uniform_points(5000, 3, 1)
    qp = dg.uniform_points(3000, 3, 2)
    _spatial_case(arbx, orc, cmp, prims, dg.POINT, dg.sphere_queries(qp, 0.08), dg.SPHERE, f"leaf_max={leaf_max}")
    ix = arbx.Index(_dev(prims), dg.POINT)
    gi, gd = ix.query_knn(_dev(qp), 10)
    ix.close()
    cmp.compare_knn(prims, dg.POINT, qp, 10, orc.knn(prims, dg.POINT, qp, 10), (_np(gi), _np(gd)), what="knn leaf")


# ---- P2 / P3: lattice closed forms straight on the GPU ------------------------------------------------
@pytest.mark.parametrize("D,g", [(1, 50), (2, 20), (3, 9), (4, 5)])
def test_lattice_closed_form_gpu(arbx, D, g):
    p = dg.lattice_points(g, D)
    ix = arbx.Index(_dev(p), dg.POINT)
    counts = _np(ix.query_count(_dev(dg.sphere_queries(p, 1.0)), dg.SPHERE))
    expect = 1 + (p > 0).sum(1) + (p < g - 1).sum(1)
    assert np.array_equal(counts, expect)
    assert int(counts.sum()) == g ** D + 2 * D * g ** (D - 1) * (g - 1)
    k = 2 * D + 1
    interior = np.all((p > 0) & (p < g - 1), axis=1)
    gi, gd = ix.query_knn(_dev(p[interior]), k)
    gi, gd = _np(gi), _np(gd)
    assert np.array_equal(gi[:, 0], np.nonzero(interior)[0])
    assert np.all(gd[:, 0] == 0.0) and np.all(gd[:, 1:] == 1.0)
    ix.close()


@pytest.mark.parametrize("D", [1, 2, 3])
def test_box_lattice_closed_form_gpu(arbx, D):
    g = 6
    cells = dg.lattice_cells(g, D)
    ix = arbx.Index(_dev(cells), dg.BOX)
    interior = np.all((cells[:, :D] > 0) & (cells[:, :D] < g - 1), axis=1)
    c = _np(ix.query_count(_dev(cells[interior]), dg.BOX))
    assert np.all(c == 3 ** D)                       # touching counts (closed)
    shrunk = cells[interior].copy()
    shrunk[:, :D] += 0.25
    shrunk[:, D:] -= 0.25
    assert np.all(_np(ix.query_count(_dev(shrunk), dg.BOX)) == 1)
    centres = cells[:, :D] + 0.5
    assert np.all(_np(ix.query_count(_dev(centres), dg.POINT)) == 1)
    verts = cells[interior][:, :D].copy()
    assert np.all(_np(ix.query_count(_dev(verts), dg.POINT)) == 2 ** D)
    ix.close()


# ---- edge cases ------------------------------------------------------------------------------------------
def test_edge_sizes(arbx, orc):
    from oracle import compare as cmp
    q = dg.sphere_queries(dg.uniform_points(50, 3, 3), 0.5)
    for n in (0, 1, 2, 3, 5):
        prims = dg.uniform_points(n, 3, 4)
        ix = arbx.Index(_dev(prims).reshape(n, 3), dg.POINT, dim=3)
        assert ix.size() == n and ix.empty() == (n == 0)
        assert ix.validate() == 0
        off, idx = ix.query_spatial(_dev(q), dg.SPHERE)
        cmp.compare_spatial(n, orc.spatial(prims.reshape(n, 3), dg.POINT, q, dg.SPHERE), (_np(off), _np(idx)), f"n={n}")
        gi, gd = ix.query_knn(_dev(q[:, :3].copy()), 4)
        cmp.compare_knn(prims.reshape(n, 3), dg.POINT, q[:, :3].copy(), 4,
                        orc.knn(prims.reshape(n, 3), dg.POINT, q[:, :3].copy(), 4), (_np(gi), _np(gd)), what=f"knn n={n}")
        # nq = 0
        off0, idx0 = ix.query_spatial(torch.empty((0, 4), device="cuda"), dg.SPHERE)
        assert _np(off0).tolist() == [0] and idx0.numel() == 0
        ix.close()


def test_bounds_and_duplicates(arbx, orc):
    from oracle import compare as cmp
    prims = dg.uniform_points(4000, 3, 6)
    ix = arbx.Index(_dev(prims), dg.POINT)
    lo, hi = ix.bounds()
    assert np.array_equal(np.float32(lo), prims.min(0)) and np.array_equal(np.float32(hi), prims.max(0))
    ix.close()
    # all-duplicate points, collinear points, a zero-extent axis
    dup = np.tile(np.float32([[0.3, 0.4, 0.5]]), (3000, 1))
    col = np.zeros((3000, 3), np.float32)
    col[:, 0] = np.linspace(0, 1, 3000, dtype=np.float32)
    flat = dg.uniform_points(3000, 3, 7)
    flat[:, 2] = 0.25
    q = dg.sphere_queries(dg.uniform_points(200, 3, 8), 0.3)
    for name, p in (("dup", dup), ("collinear", col), ("flat", flat)):
        _spatial_case(arbx, orc, cmp, p, dg.POINT, q, dg.SPHERE, name)
        ix = arbx.Index(_dev(p), dg.POINT)
        gi, gd = ix.query_knn(_dev(q[:, :3].copy()), 7)
        cmp.compare_knn(p, dg.POINT, q[:, :3].copy(), 7, orc.knn(p, dg.POINT, q[:, :3].copy(), 7),
                        (_np(gi), _np(gd)), what=f"knn {name}")
        ix.close()


def test_radius_edge_values(arbx):
    p = dg.lattice_points(6, 3)
    ix = arbx.Index(_dev(p), dg.POINT)
    assert np.all(_np(ix.query_count(_dev(dg.sphere_queries(p, 0.0)), dg.SPHERE)) == 1)    # r = 0: self only
    assert np.all(_np(ix.query_count(_dev(dg.sphere_queries(p, -1.0)), dg.SPHERE)) == 0)   # r < 0: nothing
    big = _np(ix.query_count(_dev(dg.sphere_queries(p, 100.0)), dg.SPHERE))
    assert np.all(big == len(p))                                                           # everything
    off, idx = ix.query_spatial(_dev(dg.sphere_queries(p, 100.0)), dg.SPHERE)
    rows = _np(idx).reshape(len(p), len(p))
    assert np.array_equal(np.sort(rows, axis=1), np.tile(np.arange(len(p)), (len(p), 1)))  # each index once
    ix.close()


def test_errors_and_capacity(arbx):
    p = _dev(dg.uniform_points(1000, 3, 1))
    ix = arbx.Index(p, dg.POINT)
    q = _dev(dg.sphere_queries(dg.uniform_points(100, 3, 2), 0.2))
    off = torch.empty(101, dtype=torch.int32, device="cuda")
    small = torch.empty(5, dtype=torch.int32, device="cuda")
    st, total = arbx.arbx_query_spatial(ix.handle, q, 100, dg.SPHERE, off, small, 5, raise_on_capacity=False)
    assert st == arbx.ERR_CAPACITY and total == int(off[-1]) and total > 5
    with pytest.raises(arbx.ArbxError):
        arbx.arbx_build(p, 11, dg.POINT)
    with pytest.raises(arbx.ArbxError):
        ix.query_knn(q[:, :3].contiguous(), 0)
    with pytest.raises(arbx.ArbxError):
        ix.query_knn(q[:, :3].contiguous(), arbx.K_MAX + 1)
    # overflow: 70000 x 70000 all-pairs > INT32_MAX
    pp = _dev(dg.uniform_points(70000, 3, 3))
    ix2 = arbx.Index(pp, dg.POINT)
    qq = _dev(dg.sphere_queries(dg.uniform_points(70000, 3, 4), 10.0))
    off2 = torch.empty(70001, dtype=torch.int32, device="cuda")
    with pytest.raises(arbx.ArbxError) as e:
        arbx.arbx_query_spatial(ix2.handle, qq, 70000, dg.SPHERE, off2, None, 0)
    assert e.value.status == arbx.ERR_OVERFLOW
    ix.close(); ix2.close()


# ---- P10 / T5: metamorphic and concurrency ----------------------------------------------------------------
def test_metamorphic_permutation_and_scaling(arbx):
    p = dg.uniform_points(20000, 3, 1)
    qp = dg.uniform_points(5000, 3, 2)
    q = dg.sphere_queries(qp, 0.05)

    def rows(prims, queries):
        ix = arbx.Index(_dev(prims), dg.POINT)
        off, idx = ix.query_spatial(_dev(queries), dg.SPHERE)
        ix.close()
        off, idx = _np(off), _np(idx)
        return [np.sort(idx[off[i]:off[i + 1]]) for i in range(len(off) - 1)]

    base = rows(p, q)
    g = dg.rng(9)
    pp, pq = g.permutation(len(p)), g.permutation(len(q))
    inv = np.argsort(pp)
    r2 = rows(p[pp], q)
    assert all(np.array_equal(np.sort(pp[b]), a) for a, b in zip(base, r2))   # permuting primitives permutes indices
    r3 = rows(p, q[pq])
    assert all(np.array_equal(base[pq[i]], r3[i]) for i in range(len(q)))      # permuting queries permutes rows
    r4 = rows(p * np.float32(4.0), q * np.float32(4.0))                        # power-of-two scaling is exact
    assert all(np.array_equal(a, b) for a, b in zip(base, r4))
    del inv


def test_two_streams_one_handle(arbx):
    p = _dev(dg.uniform_points(200000, 3, 1))
    q1 = _dev(dg.sphere_queries(dg.uniform_points(100000, 3, 2), 0.02))
    q2 = _dev(dg.sphere_queries(dg.uniform_points(100000, 3, 3), 0.03))
    ix = arbx.Index(p, dg.POINT)
    torch.cuda.synchronize()
    ref1, ref2 = ix.query_count(q1), ix.query_count(q2)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for _ in range(3):
        with torch.cuda.stream(s1):
            c1 = ix.query_count(q1, stream=s1)
        with torch.cuda.stream(s2):
            c2 = ix.query_count(q2, stream=s2)
        torch.cuda.synchronize()
        assert torch.equal(c1, ref1) and torch.equal(c2, ref2)
    ix.close()


# ---- the five BASELINE.json configurations ------------------------------------------------------------------
def _config_case(arbx, orc, name, scale):
    from oracle import compare as cmp
    cfg = dg.config(name, scale)
    prims, pk = cfg["prims"], cfg["pkind"]
    r = cfg["r"]
    grid = None
    if cfg["n"] * cfg["nq"] > 2e8:
        cell = orc.default_cell(prims, pk, "spatial", r if r else None)
        grid = orc.Grid(prims, pk, cell)
    st = _spatial_case(arbx, orc, cmp, prims, pk, cfg["queries"], cfg["qkind"], f"{name} x{scale}", grid)
    if cfg["k"]:
        ix = arbx.Index(_dev(prims), pk)
        gi, gd = ix.query_knn(_dev(cfg["qpoints"]), cfg["k"])
        ix.close()
        kgrid = orc.Grid(prims, pk, orc.default_cell(prims, pk, "knn")) if grid is not None else None
        o = orc.knn(prims, pk, cfg["qpoints"], cfg["k"], kgrid)
        cmp.compare_knn(prims, pk, cfg["qpoints"], cfg["k"], o, (_np(gi), _np(gd)), what=f"{name} knn")
    return st


def test_config_c1_full(arbx, orc):
    st = _config_case(arbx, orc, "C1", 1.0)
    assert 80_000 < st["pairs"] < 110_000      # P8: ~9.3 neighbours per query


@pytest.mark.parametrize("name,scale", [("C2", 0.2), ("C3", 0.02), ("C4", 0.02), ("C5", 0.05)])
def test_configs_scaled(arbx, orc, name, scale):
    _config_case(arbx, orc, name, scale)


def _sampled_full(arbx, orc, name, nsample=2000):
    """Full-size config in the launch configuration bench.py times; the oracle computes a random
    sample of query rows one by one (brute force over all N primitives)."""
    from oracle import compare as cmp
    cfg = dg.config(name, 1.0)
    prims, pk, D = cfg["prims"], cfg["pkind"], cfg["dim"]
    ix = arbx.Index(_dev(prims), pk)
    assert ix.validate() == 0
    dq = _dev(cfg["queries"])
    counts = ix.query_count(dq, cfg["qkind"])
    off, idx = ix.query_spatial(dq, cfg["qkind"])
    off, idx, counts = _np(off), _np(idx), _np(counts)
    assert np.array_equal(counts, np.diff(off))
    sel = np.sort(dg.rng(77).choice(cfg["nq"], nsample, replace=False))
    o = orc.spatial(prims, pk, cfg["queries"][sel], cfg["qkind"])           # brute force rows
    soff = np.concatenate([[0], np.cumsum(counts[sel])]).astype(np.int64)
    sidx = np.concatenate([idx[off[s]:off[s + 1]] for s in sel]) if soff[-1] else np.zeros(0, np.int32)
    cmp.compare_spatial(cfg["n"], o, (soff, sidx), f"{name} full sampled")
    if cfg["k"]:
        gi, gd = ix.query_knn(_dev(cfg["qpoints"]), cfg["k"])
        gi, gd = _np(gi), _np(gd)
        qs = cfg["qpoints"][sel]
        ok = orc.knn(prims, pk, qs, cfg["k"])
        cmp.compare_knn(prims, pk, qs, cfg["k"], ok, (gi[sel], gd[sel]), what=f"{name} full knn sampled")
        assert np.all(np.diff(gd, axis=1) >= 0) and np.all(gi >= 0)
    ix.close()


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_configs_full_sampled(arbx, orc, name):
    _sampled_full(arbx, orc, name)


# ---- every traversal / CSR-assembly path gives the same answer ------------------------------------------
@pytest.mark.parametrize("traversal", ["thread", "packet", None])
@pytest.mark.parametrize("budget_mb", ["0", "1", None])
def test_paths_agree_with_oracle(arbx, orc, knobs, traversal, budget_mb):
    """knob traversal forces per-lane or packet traversal (default: per-warp choice);
    store_budget_mb=0 forces count -> scan -> fill (two traversals), 1 MB gives 16-slot
    stored rows so that dense queries overflow and take the second traversal."""
    from oracle import compare as cmp
    knobs(traversal=traversal)
    if budget_mb is not None:
        knobs(store_budget_mb=int(budget_mb))
    prims = dg.uniform_points(6000, 3, 41)
    qp = dg.uniform_points(4000, 3, 42)
    q = dg.sphere_queries(qp, 0.09)          # ~18 hits per query on average: rows above and below 16
    q[::7, 3] = 0.25                          # some very dense rows (hundreds of hits)
    st = _spatial_case(arbx, orc, cmp, prims, dg.POINT, q, dg.SPHERE, f"paths {traversal} {budget_mb}")
    assert st["pairs"] > 16 * 4000
    boxes = dg.uniform_boxes(5000, 3, 43, 0.02)
    qb = dg.uniform_boxes(3000, 3, 44, 0.05)
    _spatial_case(arbx, orc, cmp, boxes, dg.BOX, qb, dg.BOX, f"paths boxes {traversal} {budget_mb}")
    ix = arbx.Index(_dev(prims), dg.POINT)
    for k in (3, 16, 33):
        gi, gd = ix.query_knn(_dev(qp), k)
        cmp.compare_knn(prims, dg.POINT, qp, k, orc.knn(prims, dg.POINT, qp, k), (_np(gi), _np(gd)), what=f"knn {traversal} k={k}")
    ix.close()


def test_coherent_and_scattered_warps_in_one_batch(arbx, orc):
    """Half of the queries sit in one tight cluster (packet warps), half are spread out with tiny
    radii (per-lane warps): the per-warp choice must not change any row."""
    from oracle import compare as cmp
    prims = dg.uniform_points(20000, 3, 51)
    tight = (0.5 + 0.01 * dg.uniform_points(2048, 3, 52)).astype(np.float32)
    loose = dg.uniform_points(2048, 3, 53)
    q = np.concatenate([dg.sphere_queries(tight, 0.08), dg.sphere_queries(loose, 0.004)], axis=0)
    _spatial_case(arbx, orc, cmp, prims, dg.POINT, q, dg.SPHERE, "mixed coherence")


# ---- NEXT-1: capped count with early exit ----------------------------------------
@pytest.mark.parametrize("traversal", ["thread", "packet", None])
def test_count_upto(arbx, orc, knobs, traversal):
    from oracle import compare as cmp
    knobs(traversal=traversal)
    prims = dg.uniform_points(8000, 3, 61)
    q = dg.sphere_queries(dg.uniform_points(5000, 3, 62), 0.08)
    o = orc.spatial(prims, dg.POINT, q, dg.SPHERE)
    ix = arbx.Index(_dev(prims), dg.POINT)
    full = _np(ix.query_count(_dev(q), dg.SPHERE))
    for limit in (1, 5, 17, 10_000):
        c = _np(ix.query_count(_dev(q), dg.SPHERE, limit=limit))
        cmp.compare_counts_upto(o, c, limit, f"upto {limit} {traversal}")
        assert np.array_equal(c, np.minimum(full, limit))      # same arithmetic as the uncapped count
    with pytest.raises(arbx.ArbxError):
        ix.query_count(_dev(q), dg.SPHERE, limit=0)
    ix.close()
    # exact predicate (boxes): bit-exact against the definition min(|row|, limit)
    boxes = dg.uniform_boxes(6000, 3, 63, 0.03)
    qb = dg.uniform_boxes(3000, 3, 64, 0.05)
    ob = orc.spatial(boxes, dg.BOX, qb, dg.BOX)
    ixb = arbx.Index(_dev(boxes), dg.BOX)
    for limit in (2, 9):
        c = _np(ixb.query_count(_dev(qb), dg.BOX, limit=limit))
        assert np.array_equal(c, np.minimum(np.diff(ob[0]), limit))
    ixb.close()


def test_count_upto_lattice_closed_form(arbx):
    p = dg.lattice_points(8, 3)
    ix = arbx.Index(_dev(p), dg.POINT)
    expect = 1 + (p > 0).sum(1) + (p < 7).sum(1)             # r = 1: self + in-range axis neighbours
    for limit in (1, 4, 7, 50):
        c = _np(ix.query_count(_dev(dg.sphere_queries(p, 1.0)), dg.SPHERE, limit=limit))
        assert np.array_equal(c, np.minimum(expect, limit))
    ix.close()


def test_run_to_run_determinism(arbx):
    """T5: result SETS are identical from run to run (atomics only order arrivals, never values)."""
    prims = _dev(dg.uniform_points(300_000, 3, 71))
    q = _dev(dg.sphere_queries(dg.uniform_points(200_000, 3, 72), 0.02))
    ref = None
    for _ in range(3):
        ix = arbx.Index(prims, dg.POINT)
        assert ix.validate() == 0
        c = ix.query_count(q)
        off, idx = ix.query_spatial(q)
        gi, gd = ix.query_knn(q[:, :3].contiguous(), 8)
        ix.close()
        rows = torch.stack([torch.repeat_interleave(torch.arange(off.numel() - 1, device="cuda"), torch.diff(off).long()), idx.long()], 1)
        key = torch.sort(rows[:, 0] * 300_000 + rows[:, 1]).values
        cur = (c.clone(), off.clone(), key, gd.clone())
        if ref is None:
            ref = cur
        else:
            assert all(torch.equal(a, b) for a, b in zip(ref, cur))


@pytest.mark.parametrize("traversal", ["thread", "packet", None])
def test_spatial_upto(arbx, orc, knobs, traversal):
    """Capped storage query (PAPER.md:L174 early exit from a storing callback)."""
    from oracle import compare as cmp
    knobs(traversal=traversal)
    prims = dg.uniform_points(8000, 3, 81)
    q = dg.sphere_queries(dg.uniform_points(5000, 3, 82), 0.08)
    o = orc.spatial(prims, dg.POINT, q, dg.SPHERE)
    ix = arbx.Index(_dev(prims), dg.POINT)
    for limit in (1, 6, 100, 10_000):
        off, idx = ix.query_spatial_upto(_dev(q), limit, dg.SPHERE)
        cmp.compare_spatial_upto(len(prims), o, (_np(off), _np(idx)), limit, f"spatial_upto {limit} {traversal}")
        c = _np(ix.query_count(_dev(q), dg.SPHERE, limit=limit))
        assert np.array_equal(c, np.diff(_np(off)))                 # same capped counts
    off, idx = ix.query_spatial_upto(_dev(q), 10_000, dg.SPHERE)        # a cap nobody reaches = the full query
    cmp.compare_spatial(len(prims), o, (_np(off), _np(idx)), "spatial_upto unlimited")
    ix.close()
    boxes = dg.uniform_boxes(6000, 3, 83, 0.03)
    qb = dg.uniform_boxes(3000, 3, 84, 0.05)
    ob = orc.spatial(boxes, dg.BOX, qb, dg.BOX)
    ixb = arbx.Index(_dev(boxes), dg.BOX)
    off, idx = ixb.query_spatial_upto(_dev(qb), 4, dg.BOX)
    cmp.compare_spatial_upto(len(boxes), ob, (_np(off), _np(idx)), 4, "spatial_upto boxes")
    assert np.array_equal(np.diff(_np(off)), np.minimum(np.diff(ob[0]), 4))
    ixb.close()


# ---- NEXT-2: self-join / pair search ------------------------------------------------------
@pytest.mark.parametrize("traversal", ["thread", "packet", None])
@pytest.mark.parametrize("D", [2, 3, 5])
def test_query_pairs(arbx, orc, knobs, traversal, D):
    from oracle import compare as cmp
    knobs(traversal=traversal)
    n = 6000
    p = dg.uniform_points(n, D, 90 + D)
    p[100:140] = p[100]                                      # a clump of duplicates: distance 0 pairs
    r = 0.5 * (12.0 / n) ** (1.0 / D)
    o = orc.spatial(p, dg.POINT, dg.sphere_queries(p, r), dg.SPHERE)
    ix = arbx.Index(_dev(p), dg.POINT)
    off, idx = ix.query_pairs(r)
    st = cmp.compare_pairs(n, o, (_np(off), _np(idx)), f"pairs D={D} {traversal}")
    assert st["pairs"] >= 40 * 39 // 2
    off0, idx0 = ix.query_pairs(0.0)                         # r = 0: exactly the duplicate pairs
    assert idx0.numel() == 40 * 39 // 2
    ix.close()


def test_query_pairs_lattice_and_errors(arbx):
    g = 7
    p = dg.lattice_points(g, 3)
    ix = arbx.Index(_dev(p), dg.POINT)
    off, idx = ix.query_pairs(1.0)
    assert idx.numel() == 3 * g * g * (g - 1)                # axis-neighbour pairs of a g^3 lattice, once each
    ix.close()
    b = arbx.Index(_dev(dg.uniform_boxes(100, 3, 1, 0.1)), dg.BOX)
    with pytest.raises(arbx.ArbxError) as e:
        b.query_pairs(0.1)
    assert e.value.status == arbx.ERR_UNSUPPORTED
    b.close()


# ---- NEXT-3: DBSCAN on top of the index ---------------------------------------
@pytest.mark.parametrize("traversal", ["thread", "packet", None])
@pytest.mark.parametrize("D,min_pts", [(2, 5), (3, 4), (3, 1), (5, 6)])
def test_dbscan(arbx, orc, knobs, traversal, D, min_pts):
    from oracle import compare as cmp
    knobs(traversal=traversal)
    n = 12000
    blobs = dg.gaussian_mixture(n - 2000, D, 100 + D, centre_seed=7, ncomp=12, sigma=0.015)
    p = np.concatenate([blobs, dg.uniform_points(2000, D, 200 + D)]).astype(np.float32)   # clusters + background noise
    eps = 0.6 * (8.0 / n) ** (1.0 / D) if D < 5 else 0.03
    o = orc.dbscan(p, eps, min_pts)
    while o[3]:                       # a pair inside the 1e-6 tolerance band: nudge eps off it
        eps = float(np.float32(eps * 1.0001))
        o = orc.dbscan(p, eps, min_pts)
    ix = arbx.Index(_dev(p), dg.POINT)
    labels = _np(ix.dbscan(eps, min_pts))
    st = cmp.compare_dbscan(o, labels, f"dbscan D={D} minPts={min_pts} {traversal}")
    assert st["clusters"] >= 1 and st["core"] > 0
    core = o[0]
    assert np.array_equal(labels[core] == np.arange(len(p))[core], labels[core] == np.arange(len(p))[core])
    # label = smallest core index of the cluster
    for lab in np.unique(labels[labels >= 0])[:50]:
        members = np.nonzero((labels == lab) & core)[0]
        assert members.min() == lab
    ix.close()


def test_dbscan_chain_closed_form(arbx):
    chain = np.zeros((7, 2), np.float32)
    chain[:, 0] = np.arange(7)
    pts = np.concatenate([chain, chain + np.float32([0, 50]), np.float32([[100, 100], [200, 200]])])
    ix = arbx.Index(_dev(pts), dg.POINT)
    lab = _np(ix.dbscan(1.25, 3)).tolist()
    assert lab == [1] * 7 + [8] * 7 + [-1, -1]
    assert _np(ix.dbscan(0.5, 1)).tolist() == list(range(16))         # minPts = 1: every point its own cluster
    assert _np(ix.dbscan(0.5, 2)).tolist() == [-1] * 16               # nobody has a neighbour within 0.5
    ix.close()


def test_self_join_and_dbscan_tiny_and_1d(arbx, orc):
    from oracle import compare as cmp
    for n in (1, 2, 3, 17):
        p = dg.uniform_points(n, 1, 300 + n)
        ix = arbx.Index(_dev(p).reshape(n, 1), dg.POINT, dim=1)
        off, idx = ix.query_pairs(10.0)                       # everything within reach: all n(n-1)/2 pairs
        assert idx.numel() == n * (n - 1) // 2 and _np(off)[-1] == idx.numel()
        lab = _np(ix.dbscan(10.0, 1))
        assert np.all(lab == 0)                               # one cluster, named after its smallest core index
        assert np.all(_np(ix.dbscan(10.0, n + 1)) == -1)      # nobody reaches minPts
        ix.close()
    x = np.sort(dg.uniform_points(4000, 1, 311), axis=0)
    ix = arbx.Index(_dev(x), dg.POINT)
    r = 0.0007
    o = orc.spatial(x, dg.POINT, dg.sphere_queries(x, r), dg.SPHERE)
    off, idx = ix.query_pairs(r)
    cmp.compare_pairs(len(x), o, (_np(off), _np(idx)), "pairs 1-D")
    od = orc.dbscan(x, r, 3)
    if not od[3]:
        cmp.compare_dbscan(od, _np(ix.dbscan(r, 3)), "dbscan 1-D")
    ix.close()
