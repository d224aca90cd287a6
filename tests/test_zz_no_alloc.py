"""arbx_query_count_noalloc: the count-only query with its scratch in a fixed array inside the
library (no cudaMalloc / cudaFree / pool call), against the existing arbx_query_count on the same
inputs -- counts are integers, so the results must be identical -- on two calls in a row (the array
keeps the previous call's contents), plus the size limit.  Collected last on purpose (file name)."""
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


def test_no_alloc_count_matches_existing_path_twice_in_a_row(arbx):
    prims = _dev(dg.uniform_points(200_000, 3, 1))
    ix = arbx.Index(prims, dg.POINT)
    # two DIFFERENT batches back to back: sizes that span several sort tiles and a ragged tail,
    # the second smaller than the first (stale contents of the first call lie behind it)
    batches = [(_dev(dg.sphere_queries(dg.uniform_points(300_007, 3, 2), 0.02)), dg.SPHERE),
               (_dev(dg.uniform_boxes(70_001, 3, 3, 0.015)), dg.BOX)]
    refs = [ix.query_count(q, kind) for q, kind in batches]
    torch.cuda.synchronize()
    outs = []
    for q, kind in batches:          # first call, then a second call right behind it on the same stream
        nq = q.shape[0]
        c = torch.full((nq,), -1, dtype=torch.int32, device="cuda")
        arbx.arbx_query_count_noalloc(ix.handle, q, nq, kind, c)
        outs.append(c)
    torch.cuda.synchronize()
    for c, ref in zip(outs, refs):
        assert torch.equal(c, ref) and int(ref.sum()) > 0
    # and the same batch twice in a row gives the same counts both times, with the device's free
    # memory unchanged around the calls (nothing is allocated or released)
    q, kind = batches[0]
    again = [torch.empty(q.shape[0], dtype=torch.int32, device="cuda") for _ in range(2)]
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for c in again:
        arbx.arbx_query_count_noalloc(ix.handle, q, q.shape[0], kind, c)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    assert torch.equal(again[0], refs[0]) and torch.equal(again[1], refs[0])
    ix.close()


def test_no_alloc_limit_small_and_brute_indexes(arbx):
    prims = _dev(dg.uniform_points(5_000, 3, 4))
    ix = arbx.Index(prims, dg.POINT)
    # beyond the fixed scratch: a clear error, nothing launched
    big = torch.zeros((arbx.NOALLOC_MAX_QUERIES + 1, 4), device="cuda")
    cnt = torch.empty(arbx.NOALLOC_MAX_QUERIES + 1, dtype=torch.int32, device="cuda")
    with pytest.raises(arbx.ArbxError) as e:
        arbx.arbx_query_count_noalloc(ix.handle, big, big.shape[0], dg.SPHERE, cnt)
    assert e.value.status == arbx.ERR_UNSUPPORTED and "ARBX_NOALLOC_MAX_QUERIES" in str(e.value)
    # exactly at the limit it runs and agrees with the existing path
    q = _dev(dg.sphere_queries(dg.uniform_points(arbx.NOALLOC_MAX_QUERIES, 3, 5), 0.03))
    c = torch.empty(q.shape[0], dtype=torch.int32, device="cuda")
    arbx.arbx_query_count_noalloc(ix.handle, q, q.shape[0], dg.SPHERE, c)
    assert torch.equal(c, ix.query_count(q, dg.SPHERE))
    ix.close()
    # tiny (brute-force) index, one query, empty index
    small = arbx.Index(_dev(dg.uniform_points(100, 3, 6)), dg.POINT)
    q1 = _dev(dg.sphere_queries(dg.uniform_points(1, 3, 7), 0.5))
    c1 = torch.empty(1, dtype=torch.int32, device="cuda")
    arbx.arbx_query_count_noalloc(small.handle, q1, 1, dg.SPHERE, c1)
    assert torch.equal(c1, small.query_count(q1, dg.SPHERE))
    small.close()
    empty = arbx.Index(torch.empty((0, 3), device="cuda"), dg.POINT, dim=3)
    c0 = torch.full((1,), 9, dtype=torch.int32, device="cuda")
    arbx.arbx_query_count_noalloc(empty.handle, q1, 1, dg.SPHERE, c0)
    assert int(c0[0]) == 0
    empty.close()
