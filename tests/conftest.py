import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def orc():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture
def knobs():
    """Set internal knobs of libarbx (arbx_debug_set: leaf_max, traversal, store_budget_mb, ...);
    every knob is back at its default after the test.  traversal: "thread" = 1, "packet" = 2."""
    from paper_2507_23700_b200 import binding
    names = {"thread": 1, "packet": 2, None: 0}

    def set_(**kw):
        for k, v in kw.items():
            if k == "traversal":
                v = names.get(v, v)
            if v is not None:
                binding.arbx_debug_set(k, float(v))
    yield set_
    binding.arbx_debug_set("reset", 0)
