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
    # the ALU peak counts the 22 pairable operations of MIP's 55 two to an instruction: 55 / 44 of one op per lane and clock
    assert abs(r["peak"] - 148 * 128 * 1.965e9 / 1e12 * 55 / 44) < 1e-9
    assert abs(r["achieved"] - 1123229967.25 * 55 / 5.656e-3 / 1e12) < 1e-9
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and 0.23 < r["frac"] < 0.24
    assert r["hbm"]["bound"] == "hbm"
    assert r["hbm"]["algorithmic_bytes_per_launch"] == 512 * 512 * 1024 * 4 + 1920 * 1080 * 16
    # dram traffic of that kernel: parsed from the committed ncu summary (1.03-1.08 GB read + 33 MB written per launch)
    assert 1.05e9 < r["traffic"] < 1.15e9 and "profiles/r01b_tex_mip_views012.md" in r["traffic_source"]
    assert r["traffic"] / r["hbm"]["algorithmic_bytes_per_launch"] < 1.05          # no wasted re-reads
    # configs[2] at 1080p, step 1: 0.25 samples per voxel -> HBM-bound
    r = bench.resident_roofline("config2", "tex", "raycast_kernel", 2048 ** 3, 1920, 1080, 148, pk,
                                21.592, 2.897, 2179925166.875, 354730695.875)
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["peak"] == 6534.8
    assert abs(r["achieved"] - (2048 ** 3 * 4 + 1920 * 1080 * 16) / 21.592e-3 / 1e9) < 1e-6
    assert 0.24 < r["frac"] < 0.25 and r["traffic"] is None and "no ncu capture" in r["traffic_source"]
    assert r["alu"]["bound"] == "alu" and r["ideal_ms"]["hbm"] > r["ideal_ms"]["alu"]
    # a kernel at the issue limit with every pairable operation paired sits at 1.0, not above
    n = 1e9
    t = n * (55 - 11) / (148 * 128 * 1.965e9)
    r = bench.resident_roofline("config1", "linear", "x", 512 * 512 * 1024, 1920, 1080, 148, pk, t * 1e3, 1.0, n, n)
    assert abs(r["frac"] - 1.0) < 1e-9


def test_default_line_carries_every_cube_size():
    sub = lambda v: {"metric": "Gsamples/s", "value": v, "unit": "Gsamples/s", "ms_per_step": 1.0, "config": {"workload": "w"},
                     "roofline": {"frac": 0.5}, "e2e": {"value": v / 2}, "gpu_launches": 16, "n_gpus": 1}
    line = bench.assemble({"config1": sub(200.0), "config2": sub(100.0), "stream": sub(4.0)}, 1, 5, 3)
    assert line["value"] == 100.0 and "config2" in line["config"]["headline"]
    assert set(line["per_config"]) == {"config1", "config2", "stream"} and line["gpu_launches"] == 48
    assert line["per_config"]["stream"]["e2e"]["value"] == 2.0
    # a cube that failed leaves its error and hands the headline on
    line = bench.assemble({"config1": sub(200.0), "config2": {"error": "OOM"}, "stream": sub(4.0)}, 1, 5, 3)
    assert line["value"] == 200.0 and line["per_config"]["config2"] == {"error": "OOM"} and line["gpu_launches"] == 32
    assert bench.assemble({"config2": {"error": "x"}}, 1, 5, 3)["value"] is None


def test_gpus_must_match_the_launch():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--no-cpu-baseline"],
                       capture_output=True, text=True, timeout=120, cwd=ROOT, env={**os.environ, "WORLD_SIZE": "1"})
    assert r.returncode == 2 and "WORLD_SIZE" in r.stderr and not r.stdout.strip()


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
