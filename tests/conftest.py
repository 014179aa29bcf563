import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(params=["large", "small"])
def kernel_set(request, monkeypatch):
    """Both kernel sets on the same small case: the large-batch mappings (one thread per atom in the radial sweeps,
    16 / 8 atoms per warp in the angular ones, the tensor-core network, the multi-CTA reduction) that the bench
    configurations run, and the small-batch ones (8 or 32 lanes per atom, one atom per warp, the plain-FMA network with the
    fused descriptor contraction and radial c-gradient) that a batch of this size would get by itself.
    Read by gnep_load_batch."""
    monkeypatch.setenv("GNEP_SMALL_BATCH", "1" if request.param == "small" else "0")
    return request.param
