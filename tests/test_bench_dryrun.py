"""bench.py run end to end WITHOUT a GPU: its Python (argument handling, the counting pass, vr_autotune, the timed
loops, the variants / min-max / regime side measurements, the e2e leg, assembling the one JSON line) against the host
emulation of tests/hostemu through tests/fake_cuda.py, on cubes small enough for it.  The numbers mean nothing (the
"device" is this box's CPU); what is checked is that every code path of the default run executes and that the line has
the keys the driver reads."""
import json
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r"""
import sys
sys.path.insert(0, {root!r})
from tests import fake_cuda
fake_cuda.install()
import bench
# the default run's three workloads, shrunk: configs[0]'s cube stands in for the resident cubes, 16^3-cell bricks and a
# 160 x 90 frame for the out-of-core one
bench.WORKLOADS["config1"] = dict(config=0, W=96, H=64, step=0.5, views="config0", lut="A")
bench.WORKLOADS["config2"] = dict(config=0, W=64, H=48, step=1.0, views="config0", lut="A")
bench.STREAM_SHAPE.update(brick=16, W=160, H=90, budget=4.0e5)
bench.CPU_BASELINE.update(n_tiles=4, tile=16, budget_s=0.5)
sys.argv = ["bench.py", "--steps", "2", "--warmup", "1"] + {extra!r}
sys.exit(bench.main())
"""


def run(extra):
    if shutil.which("g++") is None:
        pytest.skip("g++ not found")
    r = subprocess.run([sys.executable, "-c", DRIVER.format(root=ROOT, extra=extra)], capture_output=True, text=True,
                       timeout=1500, cwd=ROOT)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    return json.loads(lines[0]), r.stderr


def test_default_run_produces_the_whole_line():
    line, err = run([])
    assert "failed" not in err, err
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "roofline", "cpu_baseline", "clocks", "per_config"):
        assert k in line, k
    assert line["metric"] == "Gsamples/s" and line["value"] > 0 and line["vs_baseline"] is None and line["dtype"] == "f32"
    assert set(line["per_config"]) == {"config1", "config2", "stream"}
    assert "config2" in line["config"]["headline"]
    for name, sub in line["per_config"].items():
        assert "error" not in sub, (name, sub)
        assert sub["value"] > 0 and sub["ms_per_step"] > 0
        r = sub["roofline"]
        for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
            assert k in r, (name, k)
        e = sub["e2e"]
        assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    r2 = line["per_config"]["config2"]["roofline"]
    assert set(r2["variants_mip_ms"]) == {f"{n}_tiles{t}" for n in ("pipeline1", "pipeline2", "pipeline4", "reuse") for t in (0, 1)}
    assert r2["minmax_kernel"]["ms"] > 0
    assert line["per_config"]["config2"]["config"]["autotuned"]["pipeline"] in (1, 2, 4)
    s = line["per_config"]["stream"]
    assert s["roofline"]["bound"] == "host_link" and 0 < s["roofline"]["frac_of_pcie_nominal"]
    assert set(s["regimes"]) == {"culled", "cached"}, s["regimes"]
    assert s["regimes"]["cached"]["hit_rate"] > 0.0
    assert s["regimes"]["culled"]["bricks_streamed_per_frame"] <= s["bricks_streamed_per_frame"]
    c = line["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and "sample" in c
    assert line["gpu_launches"] > 0


def test_single_workload_and_explicit_variant():
    line, _ = run(["--workload", "config1", "--layout", "linear", "--pipeline", "2", "--tile-order", "1", "--no-cpu-baseline"])
    assert "per_config" not in line and line["config"]["layout"] == "linear"
    assert line["config"]["kernel"] == "raycast_pipe_kernel" and line["config"]["pipeline_depth"] == 2
    assert line["roofline"]["minmax_kernel"]["ms"] > 0


def test_smoke_runs_against_the_emulation():
    """__graft_entry__.smoke() -- what the driver runs first on the B200 -- executed here on the host emulation."""
    if shutil.which("g++") is None:
        pytest.skip("g++ not found")
    code = ("import sys; sys.path.insert(0, %r); from tests import fake_cuda; fake_cuda.install(); "
            "import __graft_entry__ as g; g.smoke()" % ROOT)
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "smoke OK" in r.stdout and r.stdout.count("bitwise=True") >= 6 and "bitwise=False" not in r.stdout


def test_two_ranks_replicas_only(tmp_path):
    """`--gpus 2` the way the driver launches it (torchrun, one rank per GPU): both ranks run their replica, the times
    are reduced with max over the ranks, rank 0 prints the one line.  gloo instead of NCCL, the emulation instead of GPUs."""
    if shutil.which("g++") is None:
        pytest.skip("g++ not found")
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    from tests.backends import EmuBackend
    EmuBackend().restore()                                   # the library is built before the ranks race for it
    script = tmp_path / "rank.py"
    src = DRIVER.format(root=ROOT, extra=["--gpus", "2", "--workload", "config1", "--no-variants", "--no-cpu-baseline"])
    # the process group is set up by bench.main(); gloo must be initialised before torch.cuda is replaced by the stand-in,
    # so the stand-in is installed lazily: right after init_process_group
    src = src.replace("from tests import fake_cuda\nfake_cuda.install()\n",
                      "import torch.distributed as dist\nfrom tests import fake_cuda\n"
                      "_init = dist.init_process_group\n"
                      "def _init_then_fake(*a, **k):\n    _init(*a, **k)\n    fake_cuda.install()\n"
                      "dist.init_process_group = _init_then_fake\n"
                      "import torch\ntorch.cuda.set_device = lambda d: None\n")
    script.write_text(src)
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)],
                       capture_output=True, text=True, timeout=1500, cwd=ROOT,
                       env={**os.environ, "VR_BENCH_DIST_BACKEND": "gloo", "VR_EMU_THREADS": "2", "VR_EMU_DEVICES": "2"})
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["scaling"] == "weak" and line["config"]["parallelism"] == "replicas only"
    assert line["value"] > 0 and line["e2e"]["value"] > 0
