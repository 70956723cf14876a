import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session", autouse=True)
def _build_host_libs():
    """The oracle and the input generator are plain gcc builds; make sure they exist."""
    import oracle
    import ppl_inputs

    ppl_inputs.build()
    oracle.build()
