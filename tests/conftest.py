import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
# the library reads its launch-geometry knobs (TSA_DENSE_*, TSA_TEAM_*, ... see include/ternary_sa.h) only under this
# switch; the parity tests use them to show that no setting changes a result
os.environ["TSA_TUNING"] = "1"
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def problems_cache():
    """Synthetic configs built once per session; observations come from the ORACLE's simulate."""
    from oracle import oracle as O
    from paper_2506_19866_b200 import problems as PB
    cache = {}

    def get(name):
        if name not in cache:
            cache[name] = PB.make_problem(name, O.simulate_fn)
        return cache[name]
    return get
