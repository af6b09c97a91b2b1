import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (run with -m gpu on the GPU box)")


@pytest.fixture(scope="session")
def case_c1():
    import gmco_cases
    return gmco_cases.make_case("C1")


@pytest.fixture(scope="session")
def case_small():
    """C1 geometry with fewer points: fast enough for finite differences and brute force."""
    import gmco_cases
    return gmco_cases.make_case("C1", counts=(120, 40, 50, 50), n_plans=4)
