import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session", autouse=True)
def _build_cpu_helpers():
    # generator + oracle are plain gcc/g++ builds (seconds); the CUDA library is built by the tests that need it
    import oracle
    import pfsm_inputs
    pfsm_inputs.build()
    oracle.build()
