"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/arbx.h declares; argument validation works without a GPU (no compute calls)."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "arbx.h")


@pytest.fixture(scope="module")
def L():
    from paper_2507_23700_b200 import binding
    if not os.path.exists(binding.LIB_PATH):
        import __graft_entry__ as g
        g.build()
    return binding.lib()


def _declared():
    src = open(HEADER).read()
    return re.findall(r"ARBX_API\s+[\w\s\*]+?\b(arbx_\w+)\s*\(", src)


def test_header_declares_the_north_star_calls():
    names = set(_declared())
    assert {"arbx_build", "arbx_query_spatial", "arbx_query_knn", "arbx_query_count"} <= names
    assert len(names) >= 12


def test_library_exports_every_declared_symbol(L):
    from paper_2507_23700_b200 import binding
    for name in _declared():
        assert hasattr(L, name), f"{name} declared in arbx.h but not exported"
    assert set(_declared()) == set(binding.EXPORTS)
    out = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    exported = {l.split()[-1] for l in out.splitlines() if " T " in l}
    assert {n for n in exported if n.startswith("arbx_")} == set(_declared())


def test_header_compiles_as_plain_c(tmp_path):
    c = tmp_path / "t.c"
    c.write_text('#include "arbx.h"\nint main(void){return (int)ARBX_OK;}\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(c),
                    "-o", str(tmp_path / "t.o")], check=True)


def test_argument_validation_without_gpu(L):
    h = ctypes.c_void_p()
    assert L.arbx_build(None, 5, 3, 0, None, ctypes.byref(h)) == 1          # null prims, n > 0
    assert L.arbx_build(None, 0, 11, 0, None, ctypes.byref(h)) == 1         # dim out of range
    assert L.arbx_build(None, 0, 3, 7, None, ctypes.byref(h)) == 1          # bad kind
    assert L.arbx_build(None, -1, 3, 0, None, ctypes.byref(h)) == 1
    assert L.arbx_query_knn(None, None, 0, 4, None, None, None) == 1        # null handle
    assert L.arbx_sort_pairs(None, None, 0, 3, 8, None) == 1                # key_bytes must be 4 or 8
    assert L.arbx_destroy(None, None) == 0
    assert L.arbx_status_string(4) == b"ARBX_ERR_OVERFLOW"
    assert b"arbx_sort_pairs" in L.arbx_last_error()


def test_binding_refuses_cpu_tensors():
    import torch
    from paper_2507_23700_b200 import binding
    with pytest.raises(TypeError):
        binding.Index(torch.zeros((4, 3)), binding.POINT)
