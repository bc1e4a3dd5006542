import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def cfg0():
    """BASELINE.json:configs[0]: 100 events, mu=5, seed 1, with generator truth."""
    from paper_2412_05041_b200 import datagen
    return datagen.generate_config(0, truth=True)
