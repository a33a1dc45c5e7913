"""sort-last rendering across ranks, world_size 2 and 3 over gloo on the CPU.  Every
rank runs the PRODUCT's code -- paper_1001_2049_b200.sortlast.SortLast over the package's Volume wrapper, libvr's
vr_volume_create_part / vr_render / vr_composite / vr_mip_finish -- with the library replaced by the host emulation of
tests/hostemu and torch.cuda by tests/fake_cuda.py (there is no GPU here, and the driver's GPU box has one).  Rank 0
holds the final frame against the oracle: bitwise its compositor mode S13 with the slabs as bricks, and the resident
frame up to re-association of `over`."""
import os
import shutil
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import sys
sys.path.insert(0, {root!r})
import numpy as np
import torch
import torch.distributed as dist
dist.init_process_group("gloo")                 # (before torch.cuda is replaced by the stand-in)
rank, world = dist.get_rank(), dist.get_world_size()
from tests import fake_cuda
fake_cuda.install()
import oracle
import vr_inputs as vi
import paper_1001_2049_b200 as vr
from paper_1001_2049_b200.sortlast import SortLast

B = 16
dims = (17, 15, 16 * world + 1)                 # bricks of 16 cells = the z slabs of `world` equal ranks
V = np.random.RandomState(9).randn(dims[2], dims[1], dims[0]).astype(np.float32)       # same seed on every rank
lut, vmin, vmax = vi.lut_a()
lut = lut.copy(); lut[:, 3] *= 4.0
W, H = 40, 32
cams = [vi.orbit_camera(dims, 30.0), vi.orbit_camera(dims, 210.0, elevation_deg=-50.0), vi.ortho_axis_camera(dims, axis=2)]
inside = dict(cams[0]); inside["eye"] = np.float32([8.0, 7.0, dims[2] * 0.6]); cams.append(inside)
for layout in (vr.VR_LAYOUT_LINEAR, vr.VR_LAYOUT_TEX):
    with SortLast(dims, layout=layout) as sl:
        assert sl.slabs[rank] == (16 * rank, 16)
        sl.upload(np.ascontiguousarray(V[sl.part_slices()]))
        sl.set_transfer_function(lut, vmin, vmax)
        sl.set_option(vr.VR_OPT_ERT_TAU, 2.0)
        for cam in cams:
            for mode in (0, 1):
                got = sl.render(cam, W, H, 0.5, mode).cpu().numpy()
                oc, _, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, tau=2.0, bricked=B, compositor=True)
                ref, _, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, tau=2.0)
                assert np.array_equal(got, oc), (rank, layout, mode)          # every rank holds the final frame
                assert np.abs(got - ref).max() < 1e-5
        # with early termination: each slab stops its own rays; what differs from the single-GPU frame is bounded by 1 - tau
        sl.set_option(vr.VR_OPT_ERT_TAU, 0.99)
        got = sl.render(cams[0], W, H, 0.5, 0).cpu().numpy()
        ref, _, _ = oracle.render(V, lut, vmin, vmax, cams[0], W, H, 0.5, 0)
        assert np.abs(got - ref).max() <= 0.0101
# unequal slabs (capability-weighted partition, PAPER.md:45): same frame up to re-association
with SortLast(dims, layout=vr.VR_LAYOUT_LINEAR, weights=[2.0] + [1.0] * (world - 1)) as sl:
    sl.upload(np.ascontiguousarray(V[sl.part_slices()]))
    sl.set_transfer_function(lut, vmin, vmax)
    sl.set_option(vr.VR_OPT_ERT_TAU, 2.0)
    for mode in (0, 1):
        got = sl.render(cams[1], W, H, 0.5, mode).cpu().numpy()
        ref, ref_aux, _ = oracle.render(V, lut, vmin, vmax, cams[1], W, H, 0.5, mode, tau=2.0)
        assert np.abs(got - ref).max() < 1e-5
        if mode == 1:
            assert np.array_equal(got, ref)                   # max is exact whatever the partition
# voxels 2.5 world units apart along the partition axis (R23): the slab of the eye is found in index space
sp = (1.0, 1.0, 2.5)
world_dims = (dims[0], dims[1], int(np.ceil((dims[2] - 1) * 2.5)) + 1)
wcams = [vi.orbit_camera(world_dims, 30.0)]
inside = dict(wcams[0]); inside["eye"] = np.float32([8.0, 7.0, (dims[2] - 1) * 2.5 * 0.3]); wcams.append(inside)
with SortLast(dims, layout=vr.VR_LAYOUT_TEX) as sl:
    sl.upload(np.ascontiguousarray(V[sl.part_slices()]))
    sl.set_transfer_function(lut, vmin, vmax)
    sl.set_option(vr.VR_OPT_ERT_TAU, 2.0)
    sl.set_option(vr.VR_OPT_SPACING_Z, 2.5)
    for cam in wcams:
        for mode in (0, 1):
            got = sl.render(cam, W, H, 0.5, mode).cpu().numpy()
            with oracle.voxel_spacing(sp):
                oc, _, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, tau=2.0, bricked=B, compositor=True)
            assert np.array_equal(got, oc), (rank, "spacing", mode)
dist.barrier()
dist.destroy_process_group()
sys.stdout.write("rank%dok\n" % rank)
"""


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 3])
def test_sort_last_over_gloo(tmp_path, world):
    if shutil.which("g++") is None:
        pytest.skip("g++ not found")
    from tests.backends import EmuBackend
    EmuBackend().restore()                       # builds libvr_hostemu.so once, before the ranks race for it
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
                        "--master-addr", "127.0.0.1", "--master-port", str(free_port()), str(script)],
                       capture_output=True, text=True, timeout=900, cwd=ROOT, env={**os.environ, "VR_EMU_THREADS": "2"})
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    for k in range(world):
        assert f"rank{k}ok" in r.stdout
