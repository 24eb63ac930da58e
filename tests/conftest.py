import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (run with -m gpu on the GPU box)")
    config.addinivalue_line("markers", "slow: full-size oracle runs (minutes of CPU)")


@pytest.fixture(scope="session")
def config0():
    import pdm_inputs
    return pdm_inputs.make_config(0)
