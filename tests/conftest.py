import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cfg0_ops():
    """Oracle operators of BASELINE.json configs[0] (shared by the CPU pin tests)."""
    from pawfe_inputs import get_config, make_system
    from oracle.operators import PawOperators
    sysd = make_system(get_config(0))
    return PawOperators(sysd)
