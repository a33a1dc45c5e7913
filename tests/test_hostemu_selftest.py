"""The host emulation of tests/hostemu held against what it claims to model (see selftest.cpp): a green emulated
parity run is evidence only if the emulation shows the hazards it is meant to show."""
import os
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
EMU = os.path.join(HERE, "hostemu")


def test_hostemu_selftest(tmp_path):
    if shutil.which("g++") is None:
        pytest.skip("g++ not found")
    exe = str(tmp_path / "selftest")
    r = subprocess.run(["g++", "-std=c++17", "-O1", "-g", "-fopenmp", "-mfma", "-ffp-contract=off", "-frounding-math",
                        "-D__CUDA_ARCH__=1000", "-I", EMU, os.path.join(EMU, "selftest.cpp"),
                        os.path.join(EMU, "emu_runtime.cpp"), "-o", exe], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    print(r.stdout)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "hazard shown" in r.stdout and "0 failed" in r.stdout
