import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def cube0():
    """configs[0]: the 64^3 seed-0 cube as a numpy float32 [z, y, x] array."""
    import vr_inputs as vi
    return vi.make_cube(0).numpy()
