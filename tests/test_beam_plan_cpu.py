"""Host logic of the beam kernel (VR_OPT_KERNEL = 2), checked without a GPU.

vr_beam_plan() runs, on the host, the functions thread 0 of the kernel's CTA runs on the device
(csrc/vr_beam_plan.h): the slab axis of a 16 x 8 pixel tile, the slabs it marches through, and
the voxel box staged for each.  The property that makes the kernel exact is geometric: every
sample of every ray of the tile must find its cell -- and the cell's far corner -- inside the
box of the slab that owns the cell, and consecutive slabs must tile the cells the rays cross.
The sample positions here are an independent float64 restatement of S1-S5;
the boxes carry a quarter-voxel margin, far more than binary32 rounding moves a position.
"""
import numpy as np
import pytest

import vr_inputs as vi

vr = pytest.importorskip("paper_1001_2049_b200")

TW, TH = 16, 8


def rays_f64(cam, W, H, i, j):
    """S1, S2 in float64 for pixel arrays i, j -> origins, unit directions."""
    f = lambda k: np.asarray(cam[k], dtype=np.float64)
    sx = ((2 * i + 1) / W - 1.0) * (W / H)
    sy = 1.0 - (2 * j + 1) / H
    if int(cam["projection"]) == vr.VR_PROJ_PERSPECTIVE:
        th = float(cam["tan_half_fovy"])
        D = f("forward")[None] + (sx * th)[:, None] * f("right")[None] + (sy * th)[:, None] * f("up")[None]
        d = D / np.linalg.norm(D, axis=1, keepdims=True)
        o = np.broadcast_to(f("eye"), d.shape).copy()
    else:
        hh = float(cam["ortho_half_height"])
        o = f("eye")[None] + (sx * hh)[:, None] * f("right")[None] + (sy * hh)[:, None] * f("up")[None]
        d = np.broadcast_to(f("forward"), o.shape).copy()
    return o, d


def clip_f64(o, d, dims):
    hi = np.asarray(dims, dtype=np.float64) - 1.0
    tn, tf, ok = 0.0, np.inf, True
    for c in range(3):
        if d[c] == 0.0:
            ok = ok and (0.0 <= o[c] <= hi[c])
        else:
            t0, t1 = (0.0 - o[c]) / d[c], (hi[c] - o[c]) / d[c]
            tn, tf = max(tn, min(t0, t1)), min(tf, max(t0, t1))
    return tn, tf, ok and tn < tf


def check_tile(dims, cam, W, H, ti, tj, step):
    info, slabs = vr.vr_beam_plan(dims, cam, W, H, ti, tj)
    ax = info["axis"]
    n = np.asarray(dims)
    ii, jj = np.meshgrid(np.arange(ti * TW, min(ti * TW + TW, W)), np.arange(tj * TH, min(tj * TH + TH, H)))
    o, d = rays_f64(cam, W, H, ii.ravel().astype(np.float64), jj.ravel().astype(np.float64))
    n_hit = n_samples = 0
    for q in range(len(o)):
        tn, tf, hit = clip_f64(o[q], d[q], dims)
        # a ray that grazes the cube within rounding may be clipped differently in binary32
        if not hit or tf - tn < 1e-3:
            continue
        n_hit += 1
        k = np.arange(int(np.ceil((tf - tn) / step)) + 1)
        t = tn + (k + 0.5) * step
        t = t[t < tf]
        if len(t) == 0:
            continue
        p = np.clip(o[q][None] + t[:, None] * d[q][None], 0.0, n - 1.0)
        cell = np.minimum(np.floor(p).astype(np.int64), n - 2)
        n_samples += len(t)
        assert info["cmin"] <= cell[:, ax].min() and cell[:, ax].max() <= info["cmax"], "cell range misses samples"
        if info["all_direct"]:
            continue
        # the slab that owns each sample's cell along the slab axis
        lo, depth = slabs[:, 1], slabs[:, 2]
        order = np.argsort(lo, kind="stable")                  # check_plan_shape: the slabs tile the axis, no overlap
        owner = order[np.clip(np.searchsorted(lo[order], cell[:, ax], side="right") - 1, 0, len(lo) - 1)]
        assert np.all((cell[:, ax] >= lo[owner]) & (cell[:, ax] < lo[owner] + depth[owner])), \
            "a sample belongs to no slab"
        # slabs are visited in marching order
        assert np.all(np.diff(owner) >= 0), "slab order is not the order along the ray"
        for s in np.unique(owner):
            kind, org, dim = slabs[s, 0], slabs[s, 3:6], slabs[s, 6:9]
            if kind != 1:
                continue
            c = cell[owner == s]
            assert np.all(c >= org[None]) and np.all(c + 1 <= org[None] + dim[None] - 1), \
                f"box {org}+{dim} does not cover cells {c.min(0)}..{c.max(0) + 1} (tile {ti},{tj}, slab {s})"
    if abs(n_hit - info["rays_hit"]) > 0:
        assert abs(n_hit - info["rays_hit"]) <= 4      # grazing rays only
    return info, slabs, n_samples


def check_plan_shape(info, slabs, dims):
    """Slabs tile [cmin, cmax] without gaps in marching order; staged boxes fit the stage, stay inside the
    cube, start on a 16-byte boundary of their x rows, and their strides address the box injectively."""
    if info["rays_hit"] == 0:
        assert info["n_slabs"] == 0
        return
    assert info["n_slabs"] == len(slabs) >= 1
    if info["all_direct"]:
        assert len(slabs) == 1 and slabs[0, 0] == 2
        assert slabs[0, 1] == info["cmin"] and slabs[0, 1] + slabs[0, 2] - 1 == info["cmax"]
        return
    ax, fast = info["axis"], info["fast"]
    mid = 3 - ax - fast
    n = np.asarray(dims)
    if info["pos"]:
        assert slabs[0, 1] == info["cmin"]
        assert np.all(slabs[1:, 1] == slabs[:-1, 1] + slabs[:-1, 2])
        assert slabs[-1, 1] + slabs[-1, 2] > info["cmax"]
    else:
        assert slabs[0, 1] + slabs[0, 2] - 1 == info["cmax"]
        assert np.all(slabs[1:, 1] + slabs[1:, 2] == slabs[:-1, 1])
        assert slabs[-1, 1] <= info["cmin"]
    assert np.all(slabs[:, 1] >= 0) and np.all(slabs[:, 2] >= 1)
    st = slabs[slabs[:, 0] == 1]
    org, dim, stride = st[:, 3:6], st[:, 6:9], st[:, 9:12]
    assert np.all(org >= 0) and np.all(org + dim <= n[None])
    if fast == 0:                                             # whole 16-byte chunks of x rows are stored
        assert np.all(org[:, 0] % 4 == 0) and np.all(dim[:, 0] % 4 == 0) and np.all(st[:, 14] * 4 == dim[:, 0])
    else:                                                     # x slabs store exactly the slab's x range
        assert np.all(org[:, 0] == st[:, 1]) and np.all(st[:, 14] * 4 >= dim[:, 0])
    assert np.all(org[:, ax] == st[:, 1])
    assert np.all(org[:, ax] + dim[:, ax] - 1 >= np.minimum(st[:, 1] + st[:, 2], n[ax] - 1))
    if ax != 0:
        assert fast == 0
        assert np.all(stride[:, 1:] % 4 == 0)                      # 16-byte chunks: strides of y and z are multiples of 4
    assert np.all(stride[:, fast] == 1)
    assert np.all(stride[:, mid] >= dim[:, fast])
    assert np.all(stride[:, ax] >= stride[:, mid] * dim[:, mid])
    assert np.all(st[:, 12] == stride[:, ax] * dim[:, ax])
    assert np.all(st[:, 12] * 4 <= info["stage_bytes"])
    assert np.all(st[:, 13] == info["stage_bytes"] // 4 - 1 - stride.sum(axis=1))


CASES = [
    # dims, camera, W, H, step
    ((64, 64, 64), "c0v0", 256, 256, 0.5),
    ((64, 64, 64), "c0v1", 256, 256, 0.5),
    ((512, 512, 1024), "orbit0", 1920, 1080, 0.5),
    ((512, 512, 1024), "orbit1", 1920, 1080, 0.5),
    ((512, 512, 1024), "orbit2", 1920, 1080, 0.5),
    ((512, 512, 1024), "orbit5", 1920, 1080, 0.5),
    ((2048, 2048, 2048), "orbit3", 1920, 1080, 1.0),
    ((2048, 2048, 2048), "orbit6", 3840, 2160, 0.5),
    ((1024, 1024, 8192), "orbit1", 7680, 4320, 0.25),
    ((36, 29, 23), "inside", 50, 37, 0.5),
    ((132, 3, 66), "ortho_x", 33, 65, 0.3),
    ((24, 150, 31), "ortho_y", 50, 37, 1.0),
    ((4, 2, 2), "orbit4", 16, 8, 0.25),
]


def camera_for(name, dims):
    if name == "c0v0":
        return vi.config0_views()[0]
    if name == "c0v1":
        return vi.config0_views()[1]
    if name.startswith("orbit"):
        return vi.orbit_views(dims, 8)[int(name[5:])]
    if name == "inside":
        cam = dict(vi.orbit_camera(dims, 30.0))
        cam["eye"] = np.float32([(d - 1) * 0.4 for d in dims])
        return cam
    return vi.ortho_axis_camera(dims, axis={"ortho_x": 0, "ortho_y": 1}[name])


@pytest.mark.parametrize("dims,camname,W,H,step", CASES)
def test_boxes_cover_every_sample(dims, camname, W, H, step):
    cam = camera_for(camname, dims)
    rng = np.random.RandomState(abs(hash((dims, camname))) % (2 ** 31))
    tiles_x, tiles_y = (W + TW - 1) // TW, (H + TH - 1) // TH
    n_tiles = min(12 if max(dims) < 2048 else 4, tiles_x * tiles_y)
    picks = rng.choice(tiles_x * tiles_y, size=n_tiles, replace=False)
    # always include the image centre and the last (ragged) tile
    picks = list(picks) + [(tiles_y // 2) * tiles_x + tiles_x // 2, tiles_x * tiles_y - 1]
    total = staged = 0
    for tidx in picks:
        ti, tj = int(tidx % tiles_x), int(tidx // tiles_x)
        info, slabs, ns = check_tile(dims, cam, W, H, ti, tj, step)
        check_plan_shape(info, slabs, dims)
        total += ns
        staged += int((slabs[:, 0] == 1).sum()) if len(slabs) else 0
    assert total > 0


def test_dense_views_are_staged():
    """configs[1] (4 samples per voxel): the plan stages every slab of a central tile in shared memory."""
    dims = (512, 512, 1024)
    for view in range(8):
        cam = vi.orbit_views(dims, 8)[view]
        info, slabs = vr.vr_beam_plan(dims, cam, 1920, 1080, 60, 67)
        assert info["rays_hit"] == TW * TH and not info["all_direct"]
        assert np.all(slabs[:, 0] == 1), f"view {view}: {np.sum(slabs[:, 0] != 1)} direct slabs"


def test_plan_rejects_bad_arguments():
    cam = vi.config0_views()[0]
    with pytest.raises(vr.VrError):
        vr.vr_beam_plan((64, 64, 64), cam, 256, 256, 16, 0)       # tile column 16 starts at pixel 256
    with pytest.raises(vr.VrError):
        vr.vr_beam_plan((1, 64, 64), cam, 256, 256, 0, 0)


def test_stage_is_chosen_per_frame():
    """VR_OPT_BEAM_STAGE = 0: dense views (configs[1], configs[4]) get the small stage, the sparse 1080p views of
    configs[2] (two voxels per pixel) a larger one in the diagonal views; the choice is one of the candidates."""
    cand = {16384, 24576, 32768, 49152, 65536}
    dense = [vr.vr_beam_plan((512, 512, 1024), cam, 1920, 1080, 0, 0)[0]["stage_bytes"]
             for cam in vi.orbit_views((512, 512, 1024), 8)]
    assert set(dense) == {16384}
    sparse = [vr.vr_beam_plan((2048, 2048, 2048), cam, 1920, 1080, 0, 0)[0]["stage_bytes"]
              for cam in vi.orbit_views((2048, 2048, 2048), 8)]
    assert set(sparse) <= cand and max(sparse) > 16384
    # an explicit stage is taken as given
    info, _ = vr.vr_beam_plan((512, 512, 1024), vi.orbit_camera((512, 512, 1024), 0.0), 1920, 1080, 0, 0, stage_bytes=40000)
    assert info["stage_bytes"] == 40000


def test_chosen_stage_stages_the_sparse_views():
    """With the per-frame stage every slab of central and corner tiles of configs[2] at 1080p is staged."""
    dims = (2048, 2048, 2048)
    for view, cam in enumerate(vi.orbit_views(dims, 8)):
        for ti, tj in [(60, 67), (30, 30), (90, 100), (45, 80)]:
            info, slabs = vr.vr_beam_plan(dims, cam, 1920, 1080, ti, tj)
            if info["rays_hit"] == 0:
                continue
            assert not info["all_direct"]
            assert np.mean(slabs[:, 0] == 1) > 0.95, f"view {view} tile {ti},{tj}: {np.sum(slabs[:, 0] != 1)} direct slabs"
