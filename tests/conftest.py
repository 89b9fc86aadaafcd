import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def plan0():
    """BASELINE.json configs[0] (tiny phantom), generated once per session on the CPU."""
    from paper_2509_20012_b200 import plangen as pg
    return pg.build_plan(pg.config_spec(0))
