import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def small_fit_event():
    """configs[0] at 1/5 size (2000 helices, 10 barrel layers)."""
    from workloads import datagen
    return datagen.config(0, scale=0.2, seed=0)
