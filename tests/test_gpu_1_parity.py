"""GPU parity (`-m gpu`): libvr.so on the B200 through the package's binding, against the CPU oracle.
The cases live in tests/parity_cases.py.  This file sorts before test_gpu_2_fullsize.py so that `pytest -x` goes
from the small cubes to the 32 GiB ones."""
import pytest

pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from tests.parity_cases import *  # noqa: E402,F401,F403  (pytest collects the test_* functions here)


@pytest.fixture(scope="module")
def be():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from tests.backends import GpuBackend
    return GpuBackend()
