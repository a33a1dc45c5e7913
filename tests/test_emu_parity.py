"""The parity cases of tests/parity_cases.py against tests/hostemu/libvr_hostemu.so: the product's own sources
(paper_1001_2049_b200/csrc) compiled by g++ against a host emulation of the CUDA subset they use.  TEST INFRASTRUCTURE:
it holds the library's host logic, its stream / event ordering and the kernels' C++ against the oracle on a box without a
GPU; it is not a product path and proves nothing about the hardware (inline PTX is not executed)."""
import shutil

import pytest

from tests.parity_cases import *  # noqa: F401,F403  (pytest collects the test_* functions here)


@pytest.fixture(scope="module")
def be():
    if shutil.which("g++") is None:
        pytest.skip("g++ not found")
    from tests.backends import EmuBackend
    b = EmuBackend()
    b.set_sched("lazy")         # queued work runs as late as allowed; the streamed cases also run "eager" (be.scheds)
    yield b
    b.restore()
