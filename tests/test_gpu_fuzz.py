"""Seeded randomised sweep over dimensions, primitive / query kinds, sizes, data styles
(uniform, clustered, duplicate-heavy), leaf sizes, forced traversal paths and CSR assembly
paths: every API result is compared with the oracle (SURVEY.md §8(c-3) protocol)."""
import os

import numpy as np
import pytest

from paper_2507_23700_b200 import datagen as dg

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _np(t):
    return t.cpu().numpy()


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_cases_against_oracle(orc, knobs, seed):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from oracle import compare as cmp
    from paper_2507_23700_b200 import binding as arbx
    arbx.lib()
    rng = np.random.default_rng(seed)
    for it in range(14):
        D = int(rng.integers(1, 11)); pk = int(rng.integers(0, 3)); qk = int(rng.integers(0, 3))
        n = int(rng.choice([1, 2, 5, 33, 700, 5000, 20000])); nq = int(rng.choice([1, 31, 33, 1000, 5000]))
        mode = str(rng.choice(["", "thread", "packet"])); lm = int(rng.choice([1, 4, 16, 16, 64]))
        knobs(traversal=mode or None, leaf_max=lm, store_budget_mb=int(rng.choice([0, 1, 4096])),
              brute_max=int(rng.choice([-1, 0, 0, 1 << 20])))
        ext = 0.5 * (8.0 / max(n, 8)) ** (1.0 / D)
        style = str(rng.choice(["uniform", "clustered", "dups"]))
        s = int(rng.integers(1 << 30))
        if pk == dg.POINT:
            p = dg.uniform_points(n, D, s) if style != "clustered" else dg.gaussian_mixture(n, D, s, ncomp=5, sigma=0.01)
        elif pk == dg.BOX:
            p = dg.uniform_boxes(n, D, s, ext)
        else:
            p = dg.uniform_spheres(n, D, s, ext)
        if style == "dups" and n > 4:
            p[: n // 2] = p[0]
        qp = (dg.uniform_points(nq, D, s + 1) if rng.random() < 0.5
              else (p[rng.integers(0, n, nq), :D] + rng.normal(0, ext * 0.3, (nq, D))).astype(np.float32))
        q = {dg.SPHERE: dg.sphere_queries(qp, ext * float(rng.choice([0.0, 0.7, 1.5, 4.0]))),
             dg.BOX: dg.uniform_boxes(nq, D, s + 2, ext * 2), dg.POINT: qp}[qk]
        what = f"seed={seed} it={it} D={D} pk={pk} qk={qk} n={n} nq={nq} mode={mode!r} leaf={lm} {style}"
        ix = arbx.Index(_dev(p), pk, dim=D)
        assert ix.validate() == 0, what
        c = _np(ix.query_count(_dev(q), qk))
        off, idx = ix.query_spatial(_dev(q), qk)
        o = orc.spatial(p, pk, q, qk)
        cmp.compare_spatial(n, o, (_np(off), _np(idx)), what)
        cmp.compare_counts(o, c, what)
        assert np.array_equal(c, np.diff(_np(off))), what
        lim = int(rng.choice([1, 3, 20]))
        assert np.array_equal(_np(ix.query_count(_dev(q), qk, limit=lim)), np.minimum(c, lim)), what
        ou, iu = ix.query_spatial_upto(_dev(q), lim, qk)
        cmp.compare_spatial_upto(n, o, (_np(ou), _np(iu)), lim, what)
        k = int(rng.choice([1, 4, 16, 32, 50]))
        gi, gd = ix.query_knn(_dev(qp), k)
        cmp.compare_knn(p, pk, qp, k, orc.knn(p, pk, qp, k), (_np(gi), _np(gd)), what=what)
        if pk == dg.POINT and n >= 2:
            r = float(np.float32(ext * float(rng.choice([0.5, 1.2]))))
            po, pi = ix.query_pairs(r)
            cmp.compare_pairs(n, orc.spatial(p, dg.POINT, dg.sphere_queries(p, r), dg.SPHERE), (_np(po), _np(pi)), what)
            if n <= 5000:
                mp = [1, 3, 6][it % 3]
                od = orc.dbscan(p, r, mp)
                if not od[3]:
                    cmp.compare_dbscan(od, _np(ix.dbscan(r, mp)), what)
        ix.close()
