"""The parity cases against the host emulation built with AddressSanitizer: every "device" buffer is a red-zoned host
allocation, so a kernel (or the host code of the library) that touches one element outside what it was given aborts
with a report -- the no-GPU stand-in for `compute-sanitizer --tool memcheck` (tests/hostemu/build.py: build(asan=True)).
The instrumented build takes several minutes, so this is opt-in: VR_TEST_ASAN=1.  profiles/r02_hostemu_evidence.md holds
the round's full run."""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.skipif(os.environ.get("VR_TEST_ASAN", "0") != "1", reason="opt-in (VR_TEST_ASAN=1): the ASan build takes minutes")
def test_parity_cases_under_address_sanitizer():
    if shutil.which("g++") is None:
        pytest.skip("g++ not found")
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("libasan.so not found")
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:detect_stack_use_after_return=0", VR_EMU_ASAN="1")
    env.pop("VR_TEST_ASAN")
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_emu_parity.py"), "-x", "-q",
                        "-p", "no:cacheprovider"], capture_output=True, text=True, env=env, cwd=ROOT, timeout=7200)
    assert "AddressSanitizer" not in r.stdout + r.stderr, (r.stdout + r.stderr)[-6000:]
    assert r.returncode == 0, (r.stdout + r.stderr)[-3000:]
