import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    # The product sends launch-bound shapes (nvirt <= 56, nocc <= 8) through one fused kernel (csrc/ppl_kernels_small.cuh).  Most
    # -m gpu tests use such shapes to exercise the TILED kernels of each symmetry mode (tile edges, ring, split-K, packing):
    # they keep doing so.  The fused path is tested, as the product runs it, by tests/test_gpu_small_fused.py (which passes
    # no_small_fused=0 explicitly), by __graft_entry__.smoke() and by bench.py --config tiny / small.
    import paper_2603_20912_b200.binding as binding

    binding.DEFAULT_DEBUG = {"no_small_fused": 1}


@pytest.fixture(scope="session", autouse=True)
def _build_host_libs():
    """The oracle and the input generator are plain gcc builds; make sure they exist."""
    import oracle
    import ppl_inputs

    ppl_inputs.build()
    oracle.build()
