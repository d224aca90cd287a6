"""GPU parity tests added in round 2: packet kNN against the oracle, per-query k
(arbx_query_knn_var), unaligned kNN outputs, the brute-force index, large k, concurrent streams
on one handle for every query kind, and the five BASELINE.json configurations compared with the
oracle ELEMENT BY ELEMENT AT FULL SIZE (every row of every query, in chunks)."""
import json
import os
import time

import numpy as np
import pytest

from paper_2507_23700_b200 import datagen as dg

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


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


# ---- packet kNN: coherent warps, incoherent warps, both forced modes -----------------------------------
@pytest.mark.parametrize("traversal", ["thread", "packet", None])
@pytest.mark.parametrize("pkind", [dg.POINT, dg.BOX, dg.SPHERE])
def test_knn_packet_coherent_batches(arbx, orc, knobs, traversal, pkind):
    """Queries in tight clumps (every warp coherent: packet path), spread out (per-lane path) and
    mixed in one batch; k below, at and between the register-heap sizes."""
    from oracle import compare as cmp
    knobs(traversal=traversal, brute_max=0)
    D, n = 3, 40_000
    ext = 0.5 * (8.0 / n) ** (1.0 / D)
    prims = {dg.POINT: dg.uniform_points(n, D, 5), dg.BOX: dg.uniform_boxes(n, D, 5, ext),
             dg.SPHERE: dg.uniform_spheres(n, D, 5, ext)}[pkind]
    g = dg.rng(6)
    clumps = g.random((64, D))
    tight = (clumps[g.integers(0, 64, 6000)] + 0.004 * g.standard_normal((6000, D))).astype(np.float32)
    loose = dg.uniform_points(3000, D, 7)
    outside = (1.5 + 0.01 * g.standard_normal((500, D))).astype(np.float32)     # all beyond the scene
    qp = np.concatenate([tight, loose, outside], axis=0)
    ix = arbx.Index(_dev(prims), pkind, dim=D)
    assert ix.validate() == 0
    for k in (1, 3, 8, 16, 20, 32):
        gi, gd = ix.query_knn(_dev(qp), k)
        cmp.compare_knn(prims, pkind, qp, k, orc.knn(prims, pkind, qp, k), (_np(gi), _np(gd)),
                        what=f"packet knn pk={pkind} k={k} {traversal}")
    ix.close()


@pytest.mark.parametrize("traversal", ["packet", None])
@pytest.mark.parametrize("D", [1, 2, 5, 10])
def test_knn_packet_other_dims_and_duplicates(arbx, orc, knobs, traversal, D):
    from oracle import compare as cmp
    knobs(traversal=traversal, brute_max=0)
    n = 20_000
    prims = dg.uniform_points(n, D, 11)
    prims[: n // 4] = prims[0]                                    # a big clump of identical points
    g = dg.rng(12)
    qp = np.concatenate([(prims[g.integers(0, n, 3000)] + 1e-3 * g.standard_normal((3000, D))).astype(np.float32),
                         np.repeat(prims[:1], 100, axis=0)], axis=0)   # 100 queries ON the clump: distances 0
    ix = arbx.Index(_dev(prims), dg.POINT, dim=D)
    for k in (4, 16):
        gi, gd = ix.query_knn(_dev(qp), k)
        cmp.compare_knn(prims, dg.POINT, qp, k, orc.knn(prims, dg.POINT, qp, k), (_np(gi), _np(gd)),
                        what=f"packet knn D={D} k={k} {traversal}")
    ix.close()


# ---- NEXT-4: one k per query ---------------------------------------------------------------
@pytest.mark.parametrize("traversal", ["thread", "packet", None])
@pytest.mark.parametrize("kmax", [1, 8, 16, 40])
def test_knn_var(arbx, orc, knobs, traversal, kmax):
    from oracle import compare as cmp
    knobs(traversal=traversal, brute_max=0)
    prims = dg.uniform_points(30_000, 3, 21)
    g = dg.rng(22)
    qp = np.concatenate([(0.5 + 0.01 * g.standard_normal((2000, 3))).astype(np.float32), dg.uniform_points(2000, 3, 23)])
    kq = g.integers(-1, kmax + 3, size=qp.shape[0]).astype(np.int32)      # includes 0, < 0 and > kmax: clamped
    ix = arbx.Index(_dev(prims), dg.POINT)
    gi, gd = ix.query_knn(_dev(qp), _dev(kq), kmax=kmax)
    cmp.compare_knn_var(prims, dg.POINT, qp, kq, kmax, orc.knn_var(prims, dg.POINT, qp, kq, kmax), (_np(gi), _np(gd)),
                        what=f"knn_var kmax={kmax} {traversal}")
    # a constant k array gives exactly the rows of arbx_query_knn
    gi2, gd2 = ix.query_knn(_dev(qp), _dev(np.full(qp.shape[0], kmax, np.int32)), kmax=kmax)
    gi3, gd3 = ix.query_knn(_dev(qp), kmax)
    assert torch.equal(gd2, gd3)
    ix.close()


def test_knn_var_lattice_closed_form(arbx):
    """Integer lattice, queries on lattice points: k_q = 1 -> the point itself at distance 0;
    k_q = 2D+1 -> itself + its 2D axis neighbours at distance exactly 1 (interior points)."""
    gsz, D = 9, 3
    p = dg.lattice_points(gsz, D)
    ix = arbx.Index(_dev(p), dg.POINT)
    interior = np.nonzero(np.all((p > 0) & (p < gsz - 1), axis=1))[0]
    qp = p[interior]
    kq = np.where(np.arange(len(interior)) % 2 == 0, 1, 2 * D + 1).astype(np.int32)
    gi, gd = ix.query_knn(_dev(qp), _dev(kq), kmax=2 * D + 1)
    gi, gd = _np(gi), _np(gd)
    assert np.array_equal(gi[:, 0], interior) and np.all(gd[:, 0] == 0)
    one = kq == 1
    assert np.all(gi[one, 1:] == -1) and np.all(np.isposinf(gd[one, 1:]))
    assert np.all(gd[~one, 1:] == 1.0)
    assert np.all(np.abs(p[gi[~one, 1:]] - qp[~one][:, None, :]).sum(axis=2) == 1)
    ix.close()


def test_knn_unaligned_outputs(arbx, orc):
    """output pointers need only 4-byte alignment (slices idx[1:], dist[3:])."""
    prims = dg.uniform_points(20_000, 3, 31)
    qp = dg.uniform_points(5_000, 3, 32)
    ix = arbx.Index(_dev(prims), dg.POINT)
    dq = _dev(qp)
    for k in (4, 8, 16, 32):
        ref_i, ref_d = ix.query_knn(dq, k)
        for off_i, off_d in ((1, 3), (2, 0), (0, 1)):
            bi = torch.full((5_000 * k + 4,), -7, dtype=torch.int32, device="cuda")
            bd = torch.full((5_000 * k + 4,), -7.0, dtype=torch.float32, device="cuda")
            oi, od = bi[off_i:off_i + 5_000 * k], bd[off_d:off_d + 5_000 * k]
            arbx.arbx_query_knn(ix.handle, dq, 5_000, k, oi, od)
            torch.cuda.synchronize()
            assert torch.equal(od.view(5_000, k), ref_d)
            assert torch.all(bi[:off_i] == -7) and torch.all(bi[off_i + 5_000 * k:] == -7)
            assert torch.all(bd[:off_d] == -7) and torch.all(bd[off_d + 5_000 * k:] == -7)
    ix.close()


@pytest.mark.parametrize("k", [33, 64, 100, 200, 256])
def test_knn_large_k(arbx, orc, k):
    from oracle import compare as cmp
    prims = dg.uniform_points(3_000, 3, 41)
    qp = dg.uniform_points(500, 3, 42)
    ix = arbx.Index(_dev(prims), dg.POINT)
    gi, gd = ix.query_knn(_dev(qp), k)
    cmp.compare_knn(prims, dg.POINT, qp, k, orc.knn(prims, dg.POINT, qp, k), (_np(gi), _np(gd)), what=f"k={k}")
    ix.close()
    with pytest.raises(arbx.ArbxError):
        arbx.Index(_dev(prims), dg.POINT).query_knn(_dev(qp), 257)


def test_knn_empty_index_padding(arbx):
    """nq > 0 on an empty index: every row is padding, for both kNN calls."""
    ix = arbx.Index(torch.empty((0, 3), device="cuda"), dg.POINT, dim=3)
    qp = _dev(dg.uniform_points(100, 3, 1))
    gi, gd = ix.query_knn(qp, 5)
    assert torch.all(gi == -1) and torch.all(torch.isinf(gd))
    gi, gd = ix.query_knn(qp, _dev(np.full(100, 3, np.int32)), kmax=5)
    assert torch.all(gi == -1) and torch.all(torch.isinf(gd))
    ix.close()


# ---- NEXT-4: brute-force index --------------------------------------------------------------
@pytest.mark.parametrize("D", [1, 3, 7])
@pytest.mark.parametrize("pkind", [dg.POINT, dg.BOX, dg.SPHERE])
def test_brute_force_index(arbx, orc, knobs, D, pkind):
    from oracle import compare as cmp
    from test_gpu_parity import _spatial_case
    knobs(brute_max=1 << 20)
    n, nq = 3000, 1500
    ext = 0.5 * (8.0 / n) ** (1.0 / D)
    prims = {dg.POINT: dg.uniform_points(n, D, 51), dg.BOX: dg.uniform_boxes(n, D, 51, ext),
             dg.SPHERE: dg.uniform_spheres(n, D, 51, ext)}[pkind]
    qp = dg.uniform_points(nq, D, 52)
    for qkind, q in ((dg.SPHERE, dg.sphere_queries(qp, ext * 1.3)), (dg.BOX, dg.uniform_boxes(nq, D, 53, ext)), (dg.POINT, qp)):
        _spatial_case(arbx, orc, cmp, prims, pkind, q, qkind, f"brute D={D} pk={pkind} qk={qkind}")
    ix = arbx.Index(_dev(prims), pkind, dim=D)
    assert ix.validate() == 0
    lo, hi = ix.bounds()
    for k in (1, 10, 40):
        gi, gd = ix.query_knn(_dev(qp), k)
        cmp.compare_knn(prims, pkind, qp, k, orc.knn(prims, pkind, qp, k), (_np(gi), _np(gd)), what=f"brute knn k={k}")
    if pkind == dg.POINT:
        r = float(np.float32(ext))
        po, pi = ix.query_pairs(r)
        cmp.compare_pairs(n, orc.spatial(prims, dg.POINT, dg.sphere_queries(prims, r), dg.SPHERE), (_np(po), _np(pi)), "brute pairs")
        od = orc.dbscan(prims, r, 4)
        if not od[3]:
            cmp.compare_dbscan(od, _np(ix.dbscan(r, 4)), "brute dbscan")
    ix.close()


def test_brute_default_threshold_matches_tree(arbx, knobs):
    """Below the default threshold arbx_build makes a brute-force index; its results equal the
    tree's bit for bit (same per-pair arithmetic)."""
    prims = _dev(dg.uniform_points(400, 3, 61))
    q = _dev(dg.sphere_queries(dg.uniform_points(1000, 3, 62), 0.15))
    res = []
    for bm in (-1, 0):
        knobs(brute_max=bm)
        ix = arbx.Index(prims, dg.POINT)
        assert ix.validate() == 0
        off, idx = ix.query_spatial(q, dg.SPHERE)
        gi, gd = ix.query_knn(q[:, :3].contiguous(), 7)
        rows = [np.sort(_np(idx)[a:b]) for a, b in zip(_np(off)[:-1], _np(off)[1:])]
        res.append((_np(off), rows, _np(gd)))
        ix.close()
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][2], res[1][2])
    assert all(np.array_equal(a, b) for a, b in zip(res[0][1], res[1][1]))


# ---- execution spaces: several queries of every kind at once on one handle -------------
def test_two_streams_every_query_kind(arbx):
    p = _dev(dg.uniform_points(300_000, 3, 1))
    q1 = _dev(dg.sphere_queries(dg.uniform_points(150_000, 3, 2), 0.02))
    q2 = _dev(dg.sphere_queries(dg.uniform_points(150_000, 3, 3), 0.025))
    y1, y2 = q1[:, :3].contiguous(), q2[:, :3].contiguous()
    ix = arbx.Index(p, dg.POINT)
    torch.cuda.synchronize()
    r1, r2 = ix.query_spatial(q1), ix.query_spatial(q2)
    k1, k2 = ix.query_knn(y1, 16), ix.query_knn(y2, 5)
    torch.cuda.synchronize()

    def rows(off, idx):
        off, idx = _np(off), _np(idx)
        seg = np.repeat(np.arange(len(off) - 1), np.diff(off))
        return off, idx[np.lexsort((idx, seg))]
    ref1, ref2 = rows(*r1), rows(*r2)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for _ in range(3):
        with torch.cuda.stream(s1):
            a = ix.query_spatial(q1, stream=s1)
            ka = ix.query_knn(y1, 16, stream=s1)
        with torch.cuda.stream(s2):
            kb = ix.query_knn(y2, 5, stream=s2)
            b = ix.query_spatial(q2, stream=s2)
        torch.cuda.synchronize()
        for got, ref in ((rows(*a), ref1), (rows(*b), ref2)):
            assert np.array_equal(got[0], ref[0]) and np.array_equal(got[1], ref[1])
        assert torch.equal(ka[1], k1[1]) and torch.equal(kb[1], k2[1])
    ix.close()


def test_trim_and_debug_set(arbx):
    arbx.arbx_trim(0)
    with pytest.raises(arbx.ArbxError):
        arbx.arbx_debug_set("no_such_knob", 1)
    p = _dev(dg.uniform_points(10_000, 3, 1))
    ix = arbx.Index(p, dg.POINT)
    c = ix.query_count(_dev(dg.sphere_queries(dg.uniform_points(100, 3, 2), 0.1)))
    assert int(c.sum()) > 0
    ix.close()
    arbx.arbx_trim(0)


def test_l2_window_knob_does_not_change_results(arbx, knobs):
    p = _dev(dg.uniform_points(200_000, 3, 1))
    q = _dev(dg.sphere_queries(dg.uniform_points(50_000, 3, 2), 0.02))
    ix = arbx.Index(p, dg.POINT)
    a = ix.query_count(q)
    knobs(l2_persist=1)
    b = ix.query_count(q)
    kb = ix.query_knn(q[:, :3].contiguous(), 8)
    knobs(l2_persist=0)
    ka = ix.query_knn(q[:, :3].contiguous(), 8)
    assert torch.equal(a, b) and torch.equal(ka[1], kb[1])
    ix.close()


# ---- the BASELINE.json configurations at FULL size, every row against the oracle -----------------------------
def _full_elementwise(arbx, orc, name, chunk=1_000_000):
    """GPU results of the whole batch (the launch configuration bench.py times) against the oracle's
    Mode B (hashed grid) over ALL queries, chunk by chunk; Mode B itself is checked against brute
    force on a sample (pin P11).  Pair totals are checked against tests/golden/config_totals.json
    (written by tests/golden/make_config_totals.py from the oracle alone)."""
    from oracle import compare as cmp
    t0 = time.time()
    cfg = dg.config(name, 1.0)
    prims, pk, nq, qk = cfg["prims"], cfg["pkind"], cfg["nq"], cfg["qkind"]
    ix = arbx.Index(_dev(prims), pk)
    assert ix.validate() == 0
    dq = _dev(cfg["queries"])
    counts = _np(ix.query_count(dq, qk))
    off, idx = ix.query_spatial(dq, qk)
    off, idx = _np(off).astype(np.int64), _np(idx)
    assert np.array_equal(counts, np.diff(off))
    knn_out = None
    if cfg["k"]:
        gi, gd = ix.query_knn(_dev(cfg["qpoints"]), cfg["k"])
        knn_out = (_np(gi), _np(gd))
    ix.close()
    del dq
    torch.cuda.empty_cache()
    grid = orc.Grid(prims, pk, orc.default_cell(prims, pk, "spatial", cfg["r"] if cfg["r"] else None))
    sure = band = 0
    for a in range(0, nq, chunk):
        b = min(a + chunk, nq)
        o = orc.spatial(prims, pk, cfg["queries"][a:b], qk, grid)
        got = (off[a:b + 1] - off[a], idx[off[a]:off[b]])
        st = cmp.compare_spatial(cfg["n"], o, got, f"{name} full rows [{a},{b})")
        cmp.compare_counts(o, counts[a:b], f"{name} full counts [{a},{b})")
        band += int(np.asarray(o[2], dtype=np.int64).sum())
        sure += int(o[0][-1]) - int(np.asarray(o[2], dtype=np.int64).sum())
    total = int(off[-1])
    assert sure <= total <= sure + band
    with open(os.path.join(GOLDEN, "config_totals.json")) as f:
        gold = json.load(f)[name]
    assert (sure, band) == (gold["sure"], gold["band"]), f"{name}: oracle totals {sure}+{band} differ from the golden file {gold}"
    # Mode B against brute force on a sample of the same queries
    sel = np.sort(dg.rng(78).choice(nq, 500, replace=False))
    ob, og = orc.spatial(prims, pk, cfg["queries"][sel], qk), orc.spatial(prims, pk, cfg["queries"][sel], qk, grid)
    assert np.array_equal(ob[0], og[0]) and np.array_equal(ob[1], og[1])
    del grid
    if knn_out is not None:
        k = cfg["k"]
        kgrid = orc.Grid(prims, pk, orc.default_cell(prims, pk, "knn"))
        for a in range(0, nq, chunk):
            b = min(a + chunk, nq)
            qs = np.ascontiguousarray(cfg["qpoints"][a:b])
            o = orc.knn(prims, pk, qs, k, kgrid)
            cmp.compare_knn(prims, pk, qs, k, o, (knn_out[0][a:b], knn_out[1][a:b]), what=f"{name} full knn [{a},{b})")
        qs = np.ascontiguousarray(cfg["qpoints"][sel])
        okb, okg = orc.knn(prims, pk, qs, k), orc.knn(prims, pk, qs, k, kgrid)
        assert np.array_equal(okb[1], okg[1])
    print(f"{name} full element-wise: total={total} (oracle sure={sure} band={band}) in {time.time() - t0:.0f} s")
    return total


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_configs_full_elementwise(arbx, orc, name):
    _full_elementwise(arbx, orc, name)


# ---- NEXT-4: fp64 coordinates ---------------------------------------------------------------
def _f64_prims(kind, n, D, seed, ext):
    """fp64 inputs that are NOT representable in fp32: fp32-scale coordinates plus offsets far below
    the fp32 resolution, on top of a large common shift (1000) where fp32 resolves only ~6e-5."""
    g = np.random.default_rng(seed)
    c = 1000.0 + g.random((n, D))
    if kind == dg.POINT:
        return c
    if kind == dg.BOX:
        w = ext * (0.5 + g.random((n, D)))
        return np.concatenate([c - w, c + w], axis=1)
    return np.concatenate([c, ext * (0.5 + g.random((n, 1)))], axis=1)


@pytest.mark.parametrize("D", [1, 3, 6])
@pytest.mark.parametrize("pkind", [dg.POINT, dg.BOX, dg.SPHERE])
def test_f64_coordinates_against_fp64_oracle(arbx, knobs, D, pkind):
    """Every (query kind x primitive kind) cell and kNN on fp64 inputs whose structure lies BELOW
    fp32 resolution (coordinates ~1000 with features of size ~1e-2 .. 1e-6): an fp32 path could
    not answer these; the fp64 path must match the fp64 oracle (oracle/f64.py)."""
    from oracle import compare as cmp, f64
    from test_gpu_parity import _np
    knobs(brute_max=0)
    n, nq = 6000, 1200
    ext = 0.5 * (8.0 / n) ** (1.0 / D)
    prims = _f64_prims(pkind, n, D, 70 + D, ext)
    g = np.random.default_rng(90 + D)
    qp = 1000.0 + g.random((nq, D))
    qp[: nq // 4] = prims[: nq // 4, :D] + 1e-7 * g.standard_normal((nq // 4, D))     # far below fp32 resolution
    cases = [(dg.SPHERE, np.concatenate([qp, np.full((nq, 1), ext * 1.3)], axis=1)),
             (dg.BOX, np.concatenate([qp - ext, qp + ext], axis=1)),
             (dg.POINT, np.concatenate([qp[: nq // 2], prims[: nq - nq // 2, :D]], axis=0))]
    ix = arbx.Index(torch.from_numpy(prims).cuda(), pkind, dim=D)
    assert ix.f64 and ix.validate() == 0 and ix.size() == n
    for qkind, q in cases:
        dq = torch.from_numpy(np.ascontiguousarray(q)).cuda()
        counts = _np(ix.query_count(dq, qkind))
        off, idx = ix.query_spatial(dq, qkind)
        o = f64.spatial(prims, pkind, q, qkind)
        cmp.compare_spatial(n, o, (_np(off), _np(idx)), f"f64 D={D} pk={pkind} qk={qkind}")
        cmp.compare_counts(o, counts, f"f64 counts D={D} pk={pkind} qk={qkind}")
        assert np.array_equal(counts, np.diff(_np(off)))
    for k in (1, 8, 40):
        gi, gd = ix.query_knn(torch.from_numpy(qp).cuda(), k)
        gi, gd = _np(gi), _np(gd)
        oi, od = f64.knn(prims, pkind, qp, k)
        assert gd.dtype == np.float64 and np.all(np.diff(gd, axis=1) >= 0)
        assert np.allclose(gd, od, rtol=1e-12, atol=1e-12)            # fp64 agreement, far inside 1e-6
        dm = f64.knn_distance_matrix(prims, pkind, qp)
        assert np.allclose(np.take_along_axis(dm, gi.astype(np.int64), axis=1), gd, rtol=1e-12, atol=1e-12)
        assert np.all(np.sort(gi, axis=1)[:, 1:] != np.sort(gi, axis=1)[:, :-1]) if k > 1 else True
    ix.close()


def test_f64_resolves_what_fp32_cannot(arbx):
    """Points 1e-6 apart at coordinate 1000 collapse in fp32 (resolution 6e-5); the fp64 index keeps
    them apart: radius 1.5e-6 around point i of a line of points spaced 1e-6 finds exactly i-1, i, i+1."""
    n = 2000
    x = 1000.0 + 1e-6 * np.arange(n)
    prims = np.stack([x, np.zeros(n), np.zeros(n)], axis=1)
    ix = arbx.Index(torch.from_numpy(prims).cuda(), dg.POINT)
    q = np.concatenate([prims, np.full((n, 1), 1.5e-6)], axis=1)
    off, idx = ix.query_spatial(torch.from_numpy(q).cuda(), dg.SPHERE)
    off, idx = off.cpu().numpy(), idx.cpu().numpy()
    assert np.array_equal(np.diff(off)[1:-1], np.full(n - 2, 3)) and np.diff(off)[0] == 2 and np.diff(off)[-1] == 2
    for i in (1, 500, n - 2):
        assert sorted(idx[off[i]:off[i + 1]].tolist()) == [i - 1, i, i + 1]
    gi, gd = ix.query_knn(torch.from_numpy(prims[10:20]).cuda(), 3)
    assert np.allclose(gd.cpu().numpy()[:, 1:], 1e-6, rtol=1e-6) and np.all(gd.cpu().numpy()[:, 0] == 0)
    ix.close()


def test_f64_edges_and_type_checks(arbx):
    p64 = torch.from_numpy(1000.0 + np.random.default_rng(1).random((300, 3))).cuda()
    p32 = p64.float()
    q64 = torch.cat([p64[:50], torch.full((50, 1), 0.1, dtype=torch.float64, device="cuda")], dim=1).contiguous()
    ix64, ix32 = arbx.Index(p64, dg.POINT), arbx.Index(p32, dg.POINT)
    cnt = torch.empty(50, dtype=torch.int32, device="cuda")
    with pytest.raises(arbx.ArbxError):
        arbx.arbx_query_count_f64(ix32.handle, q64, 50, dg.SPHERE, cnt)           # fp32 handle, fp64 call
    with pytest.raises(arbx.ArbxError):
        arbx.arbx_query_count(ix64.handle, q64.float().contiguous(), 50, dg.SPHERE, cnt)   # fp64 handle, fp32 call
    with pytest.raises(arbx.ArbxError):
        arbx.arbx_query_pairs(ix64.handle, 0.1, torch.empty(301, dtype=torch.int32, device="cuda"), None, 0)
    # brute-force fp64 index (n <= 512 by default) equals the tree-based one
    c1 = ix64.query_count(q64, dg.SPHERE)
    arbx.arbx_debug_set("brute_max", 0)
    ix64t = arbx.Index(p64, dg.POINT)
    arbx.arbx_debug_set("reset", 0)
    assert torch.equal(c1, ix64t.query_count(q64, dg.SPHERE)) and int(c1.sum()) > 50
    # empty index, nq = 0, n < k padding
    e = arbx.Index(torch.empty((0, 3), dtype=torch.float64, device="cuda"), dg.POINT, dim=3)
    assert e.empty() and int(e.query_count(q64, dg.SPHERE).sum()) == 0
    gi, gd = e.query_knn(p64[:5].contiguous(), 4)
    assert torch.all(gi == -1) and torch.all(torch.isinf(gd))
    small = arbx.Index(p64[:2].contiguous(), dg.POINT)
    gi, gd = small.query_knn(p64[:5].contiguous(), 4)
    assert torch.all(gi[:, 2:] == -1) and torch.all(gi[:, :2] >= 0) and torch.all(torch.isinf(gd[:, 2:]))
    off0, idx0 = ix64.query_spatial(torch.empty((0, 4), dtype=torch.float64, device="cuda"), dg.SPHERE)
    assert off0.cpu().tolist() == [0]
    for ix in (ix64, ix32, ix64t, e, small):
        ix.close()


def test_gather_knob_does_not_change_results(arbx, knobs):
    """The Q3 experiment (sorted copy of the queries + un-permuted counts) is only another route."""
    p = _dev(dg.uniform_points(100_000, 3, 1))
    q = _dev(dg.sphere_queries(dg.uniform_points(30_001, 3, 2), 0.03))
    qb = _dev(dg.uniform_boxes(10_007, 3, 3, 0.02))
    ix = arbx.Index(p, dg.POINT)
    a, ab = ix.query_count(q), ix.query_count(qb, dg.BOX)
    knobs(gather=1)
    b, bb = ix.query_count(q), ix.query_count(qb, dg.BOX)
    assert torch.equal(a, b) and torch.equal(ab, bb) and int(a.sum()) > 0
    ix.close()
