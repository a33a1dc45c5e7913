"""bench.py host logic that needs no GPU: the roofline arithmetic, the max-over-ranks reduction of the
multi-GPU ("replicas only") path on world_size 2 over gloo, and the reference arm
(the CPU oracle) launched the way the driver launches it, single process and under torchrun."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_roofline_picks_the_binding_bound():
    pk = {"hbm_gbs": 6534.8, "sm_max_mhz": 1965.0, "source": "test"}
    # configs[1]: 4.2 samples per voxel -> issue-bound; numbers of profiles/r01c_bench_lines.md
    r = bench.resident_roofline("config1", "tex", "raycast_kernel", 512 * 512 * 1024, 1920, 1080, 148, pk,
                                5.656, 2.7286, 1123229967.25, 550676801.0)
    assert r["bound"] == "alu" and r["unit"] == "Tlane-op/s"
    assert abs(r["peak"] - 148 * 128 * 1.965e9 / 1e12) < 1e-9
    assert abs(r["achieved"] - 1123229967.25 * 55 / 5.656e-3 / 1e12) < 1e-9
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and 0.29 < r["frac"] < 0.30
    assert r["traffic"] is not None and r["hbm"]["bound"] == "hbm"
    assert r["hbm"]["algorithmic_bytes_per_launch"] == 512 * 512 * 1024 * 4 + 1920 * 1080 * 16
    # configs[2] at 1080p, step 1: 0.25 samples per voxel -> HBM-bound
    r = bench.resident_roofline("config2", "tex", "raycast_kernel", 2048 ** 3, 1920, 1080, 148, pk,
                                21.592, 2.897, 2179925166.875, 354730695.875)
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["peak"] == 6534.8
    assert abs(r["achieved"] - (2048 ** 3 * 4 + 1920 * 1080 * 16) / 21.592e-3 / 1e9) < 1e-6
    assert 0.24 < r["frac"] < 0.25 and r["traffic"] is None and r["alu"]["bound"] == "alu"
    assert r["ideal_ms"]["hbm"] > r["ideal_ms"]["alu"]


WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
got = bench.max_over_ranks([1.0 + rank, 10.0 - rank], world, "cpu")
assert got == [2.0, 10.0], got
assert bench.max_over_ranks([3.5], 1, "cpu") == [3.5]
dist.barrier()
dist.destroy_process_group()
sys.stdout.write("rank%dok\n" % rank)
"""


def test_max_over_ranks_gloo_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", str(free_port()), str(script)],
                       capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "rank0ok" in r.stdout and "rank1ok" in r.stdout


def check_reference_line(line, gpus):
    assert line["impl"] == "reference" and line["metric"] == "Gsamples/s" and line["unit"] == "Gsamples/s"
    assert line["n_gpus"] == gpus and line["higher_is_better"] is True and line["vs_baseline"] is None
    assert line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": "Gsamples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in line["config"] and line["dtype"] == "f32"


def test_reference_arm_single_process():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "config0",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    check_reference_line(json.loads(lines[0]), 1)


def test_reference_arm_under_torchrun_prints_one_line():
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", str(free_port()),
                        os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "config0", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stdout + r.stderr
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone runs and prints
    check_reference_line(json.loads(lines[0]), 2)
