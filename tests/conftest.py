import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (run with -m gpu on the GPU box)")
    config.addinivalue_line("markers", "gpu_optional: needs a real B200; tests of options that are off by default and have not "
                                       "yet run on hardware (wide_accum, line_search); not part of -m gpu")


def pytest_collection_modifyitems(config, items):
    """Tests of options that are off by default (marker gpu_optional) run only when asked for by name (-m gpu_optional):
    neither `-m gpu` nor `-m "not gpu"` selects them."""
    if "gpu_optional" in (config.getoption("-m") or ""):
        return
    keep, drop = [], []
    for it in items:
        (drop if it.get_closest_marker("gpu_optional") else keep).append(it)
    if drop:
        config.hook.pytest_deselected(items=drop)
        items[:] = keep


@pytest.fixture(scope="session")
def case_c1():
    import gmco_cases
    return gmco_cases.make_case("C1")


@pytest.fixture(scope="session")
def case_small():
    """C1 geometry with fewer points: fast enough for finite differences and brute force."""
    import gmco_cases
    return gmco_cases.make_case("C1", counts=(120, 40, 50, 50), n_plans=4)
