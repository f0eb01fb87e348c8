import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "timeout: pytest-timeout limit for tests that would hang on a dead-locked kernel")


@pytest.fixture(scope="session")
def oracle():
    import oracle as o
    o.lib()
    return o
