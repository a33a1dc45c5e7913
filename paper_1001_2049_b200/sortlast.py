"""Sort-last rendering of one cube across GPUs -- the paper's own architecture (Figure 1): the
cube is partitioned into sub-cubes, every GPU ray casts its sub-cube into a full-resolution partial image (step 3-4),
and a scene-integration step combines the N images (step 5).  SURVEY.md Sec. 8(f)2.

One process per GPU, `torch.distributed` for the plumbing (NCCL over NVLink 5 / NVSwitch on the B200 node; any backend
torch offers works, the tests use gloo).  Argument marshalling and the exchange only: the ray casting
(vr_volume_create_part + vr_render), the compositing operator S13 (vr_composite) and the final LUT pass of MIP
(vr_mip_finish) all run in libvr.so's kernels.

Partition (step 1-2): contiguous slabs of cells along one axis (frequency by default), sized in proportion to
`weights` -- the paper's scheduler "maps tasks to resources by capability"; equal weights by default.
Neighbouring slabs share one voxel layer (S10).  View order (S11 for one-dimensional bricks): slabs sorted by
|slab - slab of the eye| (perspective) or by the sign of the view direction (orthographic); two slabs at equal distance
lie on opposite sides of the eye and share no ray.
Exchange: every rank gathers all partial images (all_gather: W*H*16 B per rank and GPU -- 33 MB at 1080p, a fraction of
a millisecond at NVLink rates) and composites them itself in view order, so every rank ends with the final image and no
second exchange is needed.  (A compositor that reads the peers' partial images through NVLink peer mappings inside
vr_composite's kernel would save the gather's staging copy; it needs a multi-GPU box to be validated and is not built.)

The result equals the single-GPU frame up to the re-association of `over` (<= 1e-5) when no ray terminates early, and
is bitwise the oracle's compositor mode S13 with the slabs as bricks; with early termination each slab stops its own
rays at tau, and what lies behind a saturated slab is composited with weight <= 1 - tau.
"""
import numpy as np

from . import (VR_LAYOUT_TEX, VR_MODE_EA, VR_OPT_SPACING_X, VR_OPT_SPACING_Z, VR_PROJ_PERSPECTIVE, Volume, vr_composite,
               vr_mip_finish)


def partition(n_cells, world, weights=None):
    """[(first cell, cells)] per rank: contiguous, covering [0, n_cells), every rank at least one cell."""
    if world < 1 or n_cells < world:
        raise ValueError("need at least one cell per rank")
    w = np.ones(world) if weights is None else np.asarray(weights, dtype=np.float64)
    if w.shape != (world,) or np.any(w <= 0):
        raise ValueError("weights: one positive number per rank")
    edges = np.rint(np.cumsum(w) / w.sum() * n_cells).astype(np.int64)
    edges = np.concatenate([[0], edges])
    for r in range(1, world + 1):                       # at least one cell each, monotone, ending at n_cells
        edges[r] = min(max(edges[r], edges[r - 1] + 1), n_cells - (world - r))
    edges[world] = n_cells
    return [(int(edges[r]), int(edges[r + 1] - edges[r])) for r in range(world)]


def view_order(slabs, cam, axis, spacing=1.0):
    """Ranks front to back for this camera (S11 along one axis); spacing: world units per voxel along that axis (R23)."""
    if int(cam["projection"]) == VR_PROJ_PERSPECTIVE:
        e = np.float32(cam["eye"][axis])
        if np.float32(spacing) != np.float32(1.0):
            e = e * (np.float32(1.0) / np.float32(spacing))          # the eye in index space, as the kernels compute it
        cell = int(np.floor(float(e)))
        e = -1
        for r, (c0, nc) in enumerate(slabs):
            if cell >= c0:
                e = r if cell < c0 + nc else r + 1          # beyond the last slab: e = world
        keys = [abs(r - e) for r in range(len(slabs))]
    else:
        d = float(np.float32(cam["forward"][axis]))
        sgn = (d > 0) - (d < 0)
        keys = [sgn * r for r in range(len(slabs))]
    return sorted(range(len(slabs)), key=lambda r: (keys[r], r))


class SortLast:
    """One rank of a sort-last renderer.  dims: the whole cube (nx, ny, nz)."""

    def __init__(self, dims, rank=None, world=None, group=None, device=0, layout=VR_LAYOUT_TEX, axis=2, weights=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank = dist.get_rank(group) if rank is None else int(rank)
        self.world = dist.get_world_size(group) if world is None else int(world)
        self.dims = tuple(int(v) for v in dims)
        self.axis = int(axis)
        self.slabs = partition(self.dims[self.axis] - 1, self.world, weights)
        c0, nc = self.slabs[self.rank]
        origin, pdims = [0, 0, 0], list(self.dims)
        origin[self.axis], pdims[self.axis] = c0, nc + 1          # nc cells = nc + 1 voxel layers (one shared, S10)
        self.origin, self.part_dims = tuple(origin), tuple(pdims)
        self.vol = Volume(self.dims, device=device, layout=layout, part=(self.origin, self.part_dims))
        self.spacing = [1.0, 1.0, 1.0]

    def close(self):
        self.vol.close()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def part_slices(self):
        """numpy / torch slices [z, y, x] of the whole cube that this rank must upload."""
        return tuple(slice(self.origin[a], self.origin[a] + self.part_dims[a]) for a in (2, 1, 0))

    def upload(self, V_part, stream=None):
        """V_part: this rank's voxels, [sz, sy, sx] = the cube cut by part_slices()."""
        self.vol.upload(V_part, stream)

    def set_transfer_function(self, lut, vmin, vmax):
        self.vol.set_transfer_function(lut, vmin, vmax)

    def set_option(self, key, value):
        self.vol.set_option(key, value)
        if VR_OPT_SPACING_X <= key <= VR_OPT_SPACING_Z:
            self.spacing[key - VR_OPT_SPACING_X] = float(value)

    def render(self, cam, W, H, step, mode, stream=None):
        """The final frame [H, W, 4], on every rank."""
        torch = self.vol._torch
        partial = self.vol.render(cam, W, H, step, mode, stream=stream)
        if self.world == 1:
            parts = [partial]
        else:
            torch.cuda.current_stream(self.vol.device).synchronize()
            parts = [torch.empty_like(partial) for _ in range(self.world)]
            self.dist.all_gather(parts, partial, group=self.group)
        order = view_order(self.slabs, cam, self.axis, self.spacing[self.axis])
        s = self.vol._stream(stream)
        if mode == VR_MODE_EA:
            running = torch.zeros_like(partial)
            rest = order
        else:
            running = parts[order[0]].clone()
            rest = order[1:]
        for r in rest:
            vr_composite(running.data_ptr(), parts[r].data_ptr(), W, H, mode, s)
        if mode != VR_MODE_EA:
            vr_mip_finish(self.vol.handle, running.data_ptr(), W, H, s)
        self._keep = parts                                  # until the stream has consumed them
        return running
