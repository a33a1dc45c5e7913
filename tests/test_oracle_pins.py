"""Pins for the CPU oracle: closed forms, invariants, library
special cases and float64 brute force.  None of the expected values comes from
oracle/ itself or from the CUDA path."""
import json
import math
import os

import numpy as np
import pytest
from scipy.ndimage import map_coordinates

import oracle
import vr_inputs as vi
from tests import f64_bruteforce as bf

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.json")))
EA, MIP = oracle.MODE_EA, oracle.MODE_MIP


def const_lut(alpha, grey=0.5, n=16):
    lut = np.empty((n, 4), dtype=np.float32)
    lut[:, :3] = grey
    lut[:, 3] = alpha
    return lut


# ---- C1: constant cube, alpha = 1-(1-a)^n, step independent -----------------
@pytest.mark.parametrize("step", [0.25, 0.5, 1.0])
def test_constant_cube_closed_form(step):
    g = GOLD["constant_cube"]
    V = np.ones((64, 64, 64), dtype=np.float32)
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[0]
    img, aux, cnt = oracle.render(V, lut, vmin, vmax, cam, 256, 256, step, EA)
    n = g["samples"][str(step)]
    assert cnt["rays_hit"] == 256 * 256
    assert cnt["samples"] == 256 * 256 * n          # fence posts: exactly chord/step samples
    assert cnt["nominal"] == cnt["samples"]         # tau never reached
    tol = n * 2.0 ** -24 * 2
    assert np.abs(img[..., 3] - g["A"]).max() <= tol
    for ch in range(3):
        assert np.abs(img[..., ch] - g["grey"] * g["A"]).max() <= tol
    # all rays identical
    assert np.ptp(img[..., 3]) == 0.0


# ---- C2: early ray termination, integer closed form -------------------------
def test_ert_closed_form():
    g = GOLD["ert_constant_cube"]
    V = np.full((64, 64, 64), 0.25, dtype=np.float32)
    lut = const_lut(g["alpha_per_voxel"])
    cam = vi.config0_views()[0]
    img, _, cnt = oracle.render(V, lut, -1.0, 1.0, cam, 32, 32, g["step"], EA, tau=0.99)
    assert cnt["samples"] == 32 * 32 * g["n_terminate"]
    assert cnt["nominal"] == 32 * 32 * 126 or cnt["nominal"] == 32 * 32 * g["n_terminate"]
    assert np.abs(img[..., 3] - g["A"]).max() < 1e-5       # NOT renormalised to 1
    assert np.abs(img[..., 0] - 0.5 * g["A"]).max() < 1e-5
    # tau > 1 disables termination: all 126 samples, alpha = 1-0.7^63
    img2, _, cnt2 = oracle.render(V, lut, -1.0, 1.0, cam, 32, 32, g["step"], EA, tau=2.0)
    assert cnt2["samples"] == 32 * 32 * 126
    assert np.abs(img2[..., 3] - (1 - 0.7 ** 63)).max() < 1e-5


def test_opacity_correction_values():
    for a, step, want in GOLD["opacity_correction"]["cases"]:
        got = oracle.opacity_correct(const_lut(a, n=2), step)
        assert abs(float(got[0]) - want) < 1e-7, (a, step)


# ---- C3: trilinear is exact on a linear ramp, incl. the far faces -----------
def test_linear_ramp_exact():
    nx, ny, nz = 17, 12, 9
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    a, b, c, d = 0.37, -1.25, 2.5, 0.75
    V = (a * x + b * y + c * z + d).astype(np.float32)
    rng = np.random.RandomState(1)
    P = rng.rand(500, 3) * [nx - 1, ny - 1, nz - 1]
    P[:20] = np.round(P[:20])                       # on nodes
    P[20:30] = [nx - 1, ny - 1, nz - 1]             # p = hi on every axis
    P[30:40, 0] = nx - 1
    P[40:50, 2] = 0.0
    ulp = np.spacing(np.float32(np.abs(V).max()))
    for p in P:
        p32 = p.astype(np.float32)
        want = a * float(p32[0]) + b * float(p32[1]) + c * float(p32[2]) + d
        got = oracle.sample_at(V, p32)
        assert abs(got - want) <= 6 * ulp, (p, got, want)


def test_trilinear_matches_scipy_order1():
    rng = np.random.RandomState(2)
    V = rng.randn(7, 9, 11).astype(np.float32)
    P = (rng.rand(400, 3) * [10, 8, 6]).astype(np.float32)
    want = map_coordinates(V.astype(np.float64), [P[:, 2], P[:, 1], P[:, 0]], order=1, mode="nearest")
    got = np.array([oracle.sample_at(V, p) for p in P])
    assert np.abs(got - want).max() < 2e-6
    # a transposed operand or swapped weight would show here:
    V2 = np.zeros((3, 3, 3), dtype=np.float32)
    V2[2, 1, 0] = 1.0                                # x=0, y=1, z=2
    assert oracle.sample_at(V2, (0.25, 1.0, 2.0)) == pytest.approx(0.75)
    assert oracle.sample_at(V2, (0.0, 0.5, 2.0)) == pytest.approx(0.5)
    assert oracle.sample_at(V2, (0.0, 1.0, 1.25)) == pytest.approx(0.25)


# ---- C4: ramp under MIP = analytic value at the far (or near) end ------------
def test_ramp_mip():
    n = 64
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    V = (0.5 * x - 0.25 * y + 1.0 * z).astype(np.float32)
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[0]                      # along +z: samples at z = 0.25 + 0.5k
    W = H = 64
    img, aux, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, MIP)
    i = np.arange(W); j = np.arange(H)
    X = 31.5 + ((2 * i + 1) / W - 1.0) * 31.5
    Y = 31.5 + (1.0 - (2 * j + 1) / H) * 31.5
    want = 0.5 * X[None, :] - 0.25 * Y[:, None] + 1.0 * (0.25 + 0.5 * 125)
    assert np.abs(aux - want).max() < 2e-4
    assert cnt["samples"] == W * H * 126             # MIP never terminates early
    # decreasing ramp: maximum at the first sample
    img, aux2, _ = oracle.render(-V, lut, vmin, vmax, cam, W, H, 0.5, MIP)
    want2 = -(0.5 * X[None, :] - 0.25 * Y[:, None] + 0.25)
    assert np.abs(aux2 - want2).max() < 2e-4
    assert np.all(img[..., 3] == 1.0)


# ---- C5: single bright voxel under MIP --------------------------------------
def test_bright_voxel_mip():
    g = GOLD["bright_voxel_mip"]
    n = 64
    cx, cy, cz = 20, 41, 33
    V = np.zeros((n, n, n), dtype=np.float32)
    V[cz, cy, cx] = 1.0
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[0]
    W = H = 256
    img, aux, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, MIP)
    i = np.arange(W); j = np.arange(H)
    X = 31.5 + ((2 * i + 1) / W - 1.0) * 31.5        # +right = +x with increasing column
    Y = 31.5 + (1.0 - (2 * j + 1) / H) * 31.5        # row 0 is the top (+up = +y)
    fx = np.clip(1.0 - np.abs(X - cx), 0.0, None)
    fy = np.clip(1.0 - np.abs(Y - cy), 0.0, None)
    want = fy[:, None] * fx[None, :] * g["z_factor"]
    assert np.abs(aux - want).max() < 1e-5
    assert aux.max() > 0.6                           # the voxel is actually seen
    for dx, dy, val in g["examples"]:
        assert max(0, 1 - abs(dx)) * max(0, 1 - abs(dy)) * 0.75 == pytest.approx(val, abs=1e-9)
    # LUT colour of the maximum, alpha = 1 wherever the ray has samples
    grey = (want - vmin) / (vmax - vmin)
    assert np.abs(img[..., 0] - grey).max() < 1e-5
    assert np.all(img[..., 3] == 1.0)
    # x/y transposition or a flipped row order would break this:
    jmax, imax = np.unravel_index(np.argmax(aux), aux.shape)
    assert abs(X[imax] - cx) < 0.2 and abs(Y[jmax] - cy) < 0.2


# ---- C6: float64 brute force on tiny cubes -----------------------------------
def _rand_cam(rng, dims, perspective):
    n = np.asarray(dims, dtype=np.float64)
    c = (n - 1) / 2
    v = rng.randn(3); v /= np.linalg.norm(v)
    R = 1.6 * np.linalg.norm(n - 1) / 2 if perspective else 2.0 * np.linalg.norm(n)
    eye = c + R * v
    f = (c - eye) / np.linalg.norm(c - eye)
    upw = rng.randn(3)
    r = np.cross(upw, f); r /= np.linalg.norm(r)
    u = np.cross(f, r)
    f32 = lambda a: np.asarray(a, dtype=np.float32)
    return {"eye": f32(eye), "right": f32(r), "up": f32(u), "forward": f32(f),
            "projection": 0 if perspective else 1, "tan_half_fovy": float(np.float32(0.45)),
            "ortho_half_height": float(np.float32(0.7 * np.linalg.norm(n) / 2))}


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
@pytest.mark.parametrize("perspective", [True, False])
def test_float64_brute_force(seed, perspective):
    rng = np.random.RandomState(100 + seed)
    dims = [(16, 16, 16), (9, 14, 11), (16, 5, 8), (3, 2, 4)][seed]
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    lut = rng.rand(8, 4).astype(np.float32)
    lut[:, 3] *= 0.4
    lut[2, 3] = 0.0
    vmin, vmax = -1.5, 2.0                          # values outside the range are clamped
    cam = _rand_cam(rng, dims, perspective)
    W, H = 32, 24
    for step in (0.5, 0.3):
        # emission-absorption, termination disabled: smooth in every input
        got, _, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, step, EA, tau=2.0)
        want, _, ns = bf.render(V, lut, vmin, vmax, cam, W, H, step, 0, 2.0)
        assert np.abs(got - want).max() < 2e-5
        assert abs(cnt["samples"] - ns) <= max(4, ns // 2000)   # grazing rays may differ by a sample
        # with termination: a 1-ulp difference in A can move the stop by one sample
        got, _, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, step, EA, tau=0.9)
        want, _, _ = bf.render(V, lut, vmin, vmax, cam, W, H, step, 0, 0.9)
        err = np.abs(got - want).max(axis=-1)
        assert np.mean(err < 2e-5) > 0.99 and err.max() < 0.05
        assert got[..., 3].max() < 0.9 + 0.1 * 0.4 + 1e-6        # A is not renormalised
        # MIP
        got, aux, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, step, MIP)
        want, M, _ = bf.render(V, lut, vmin, vmax, cam, W, H, step, 1, 2.0)
        both = np.isfinite(aux) & np.isfinite(M)
        assert np.mean(np.isfinite(aux) == np.isfinite(M)) > 0.995
        # fp32 sample positions are off by a few ulp(t) ~ 1e-5 voxel; noise gradients are O(5)/voxel
        assert np.abs(aux[both] - M[both]).max() < 1e-4
        assert np.abs(got[both] - want[both]).max() < 1e-4


# ---- C7: bricked == unbricked -------------------------------------------------
@pytest.mark.parametrize("dims,B", [((16, 16, 16), 5), ((40, 33, 27), 8), ((64, 64, 64), 32)])
@pytest.mark.parametrize("mode", [EA, MIP])
def test_bricked_equals_unbricked(dims, B, mode):
    rng = np.random.RandomState(7)
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    lut, vmin, vmax = vi.lut_a()
    lut = lut.copy(); lut[:, 3] *= 8.0               # saturates inside the cube: ERT fires mid-brick
    W, H = (48, 40) if dims[0] < 64 else (64, 64)
    for cam in (_rand_cam(rng, dims, True), _rand_cam(rng, dims, False)):
        ref, ref_aux, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode)
        got, got_aux, cntb = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, bricked=B)
        assert np.array_equal(ref, got)              # fused carry-in: bitwise
        assert np.array_equal(ref_aux, got_aux)
        assert cnt["samples"] == cntb["samples"] and cnt["rays_hit"] == cntb["rays_hit"]
        # partial images + over operator: equal up to re-association, ERT disabled
        ref2, _, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, tau=2.0)
        got2, aux2, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, tau=2.0,
                                      bricked=B, compositor=True)
        assert np.abs(ref2 - got2).max() < 1e-5
        if mode == MIP:
            assert np.array_equal(aux2, ref_aux)     # max is exactly associative


@pytest.mark.parametrize("dims,B", [((16, 16, 16), 5), ((41, 33, 27), 8), ((33, 17, 9), 8)])
def test_brick_store_reader_equals_one_array(dims, B):
    """S10: the cube read from its brick store (bricks with a ghost layer on the high side) is the
    same cube -- the brick slices are cut here with plain numpy indexing, independent of oracle/."""
    rng = np.random.RandomState(17)
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    nz, ny, nx = V.shape
    bricks = []
    for z0 in range(0, nz - 1, B):                     # linear brick index bx + nbx*(by + nby*bz)
        for y0 in range(0, ny - 1, B):
            for x0 in range(0, nx - 1, B):
                bricks.append(np.ascontiguousarray(
                    V[z0:min(z0 + B, nz - 1) + 1, y0:min(y0 + B, ny - 1) + 1, x0:min(x0 + B, nx - 1) + 1]))
    ptrs = [b.ctypes.data for b in bricks]
    lut, vmin, vmax = vi.lut_a()
    lut = lut.copy(); lut[:, 3] *= 4.0
    W, H = 40, 32
    jj, ii = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    ij = np.stack([ii.ravel(), jj.ravel()], 1).astype(np.int32)
    for cam in (_rand_cam(rng, dims, True), _rand_cam(rng, dims, False), vi.ortho_axis_camera(dims, axis=0)):
        for mode in (EA, MIP):
            ref, ref_aux, cnt = oracle.render_pixels(V, lut, vmin, vmax, cam, W, H, 0.5, mode, ij)
            got, got_aux, cntb = oracle.render_pixels_bricks(ptrs, B, dims, lut, vmin, vmax, cam, W, H, 0.5,
                                                            mode, ij)
            assert np.array_equal(ref, got) and np.array_equal(ref_aux, got_aux)
            assert cnt == cntb


def test_brick_order_is_front_to_back():
    """S11: along any ray the wavefront key strictly increases from brick to brick."""
    dims, B = (40, 33, 27), 6
    rng = np.random.RandomState(11)
    nb = [oracle.n_bricks(n, B) for n in dims]
    for trial in range(6):
        cam = _rand_cam(rng, dims, perspective=trial % 2 == 0)
        if trial == 4:                               # eye inside the cube
            cam["eye"] = np.float32([20.3, 11.1, 9.7])
        order, keys = oracle.brick_order(dims, B, cam)
        assert sorted(order.tolist()) == list(range(nb[0] * nb[1] * nb[2]))
        assert np.all(np.diff(keys) >= 0)
        key_of = dict(zip(order.tolist(), keys.tolist()))
        O, D = bf.rays(cam, 24, 24)
        tn, tf, hit = bf.clip(O, D, dims)
        for (jj, ii) in zip(*np.nonzero(hit)):
            t = np.arange(tn[jj, ii] + 1e-6, tf[jj, ii], 0.05)
            P = np.clip(O[jj, ii] + t[:, None] * D[jj, ii], 0, np.array(dims) - 1.0)
            cell = np.minimum(np.floor(P).astype(int), np.array(dims) - 2)
            b = cell // B
            lin = b[:, 0] + nb[0] * (b[:, 1] + nb[1] * b[:, 2])
            seq = lin[np.concatenate([[True], np.diff(lin) != 0])]
            ks = [key_of[int(s)] for s in seq]
            assert all(k1 > k0 for k0, k1 in zip(ks, ks[1:])), (trial, ii, jj, ks)


def test_brick_minmax_definition_and_safety():
    rng = np.random.RandomState(5)
    dims, B = (21, 18, 30), 8
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    mn, mx = oracle.brick_minmax(V, B)
    assert mn.shape == (4, 3, 3)
    # corner brick by hand: cells [16, 20) in x -> voxels [15, 20]; y [16,17) -> [15,17]; z [24,29) -> [23,29]
    blk = V[23:30, 15:18, 15:21]
    assert mn[3, 2, 2] == blk.min() and mx[3, 2, 2] == blk.max()
    blk0 = V[0:10, 0:10, 0:10]
    assert mn[0, 0, 0] == blk0.min() and mx[0, 0, 0] == blk0.max()
    # safety: any sample whose cell lies in the brick is inside [mn, mx] up to fma rounding
    P = (rng.rand(4000, 3) * (np.array(dims) - 1)).astype(np.float32)
    for p in P:
        cell = np.minimum(np.floor(p).astype(int), np.array(dims) - 2) // B
        v = oracle.sample_at(V, p)
        lo, hi = mn[cell[2], cell[1], cell[0]], mx[cell[2], cell[1], cell[0]]
        guard = 8 * np.spacing(np.float32(max(abs(lo), abs(hi))))
        assert lo - guard <= v <= hi + guard


# ---- C9: invariants -------------------------------------------------------------
def test_invariants_config0(cube0):
    lut, vmin, vmax = vi.lut_a()
    views = vi.config0_views()
    for cam in views:
        img, aux, cnt = oracle.render(cube0, lut, vmin, vmax, cam, 128, 128, 0.5, EA)
        A = img[..., 3]
        assert A.min() >= 0.0 and A.max() <= 1.0
        assert np.all(img[..., :3] <= A[..., None] * lut[:, :3].max() + 1e-6)
        assert np.all(img[..., :3] >= 0.0)
        mimg, maux, _ = oracle.render(cube0, lut, vmin, vmax, cam, 128, 128, 0.5, MIP)
        has = np.isfinite(maux)
        assert has.sum() == cnt["rays_hit"]
        assert maux[has].max() <= cube0.max() + 1e-5 and maux[has].min() >= cube0.min() - 1e-5
        assert np.all(mimg[~has] == 0.0)
    # view 1 looks down the whole frequency axis: every ray 126 samples, none saturates
    _, _, cnt = oracle.render(cube0, lut, vmin, vmax, views[0], 256, 256, 0.5, EA)
    assert cnt["samples"] == 256 * 256 * 126


def test_step_halving_converges(cube0):
    """Opacity correction makes images at different steps comparable: O(step)."""
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[1]
    # smooth field so the Riemann sum converges quickly
    from scipy.ndimage import gaussian_filter
    V = gaussian_filter(cube0.astype(np.float64), 3.0).astype(np.float32) * 4.0
    imgs = [oracle.render(V, lut, vmin, vmax, cam, 64, 64, s, EA, tau=2.0)[0] for s in (1.0, 0.5, 0.25)]
    e1 = np.abs(imgs[0] - imgs[2]).max()
    e2 = np.abs(imgs[1] - imgs[2]).max()
    assert e2 < e1 and e1 < 0.02


def test_camera_roll_rotates_image():
    """A 90 degree camera roll of a cubic volume gives the rotated image."""
    rng = np.random.RandomState(3)
    V = rng.randn(12, 12, 12).astype(np.float32)
    lut, vmin, vmax = vi.lut_a()
    cam = vi.ortho_axis_camera((12, 12, 12), axis=2, half_height=8.0)
    img0, _, _ = oracle.render(V, lut, vmin, vmax, cam, 40, 40, 0.5, EA)
    rolled = dict(cam)
    rolled["right"] = cam["up"].copy()
    rolled["up"] = -cam["right"]
    img1, _, _ = oracle.render(V, lut, vmin, vmax, rolled, 40, 40, 0.5, EA)
    assert np.abs(np.rot90(img1, k=-1, axes=(0, 1)) - img0).max() < 1e-6 or \
           np.abs(np.rot90(img1, k=1, axes=(0, 1)) - img0).max() < 1e-6


def test_miss_and_degenerate_rays():
    V = np.ones((4, 4, 4), dtype=np.float32)
    lut, vmin, vmax = vi.lut_a()
    cam = vi.ortho_axis_camera((4, 4, 4), axis=2, half_height=6.0)   # wider than the cube
    img, aux, cnt = oracle.render(V, lut, vmin, vmax, cam, 16, 16, 0.5, MIP)
    assert cnt["rays_hit"] < 256 and cnt["rays_hit"] > 0
    miss = ~np.isfinite(aux)
    assert np.all(img[miss] == 0.0) and np.all(img[~miss][:, 3] == 1.0)
    with pytest.raises(ValueError):
        oracle.render(V, lut, vmin, vmax, cam, 16, 16, 0.0, EA)
    with pytest.raises(ValueError):
        oracle.render(V, lut, 1.0, 1.0, cam, 16, 16, 0.5, EA)
    with pytest.raises(ValueError):
        oracle.render(np.ones((1, 4, 4), np.float32), lut, vmin, vmax, cam, 16, 16, 0.5, EA)


def test_render_pixels_matches_full(cube0):
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[1]
    full, faux, _ = oracle.render(cube0, lut, vmin, vmax, cam, 96, 96, 0.5, EA)
    ij = vi.tile_subset(96, 96, n_tiles=4, tile=16, seed=3)
    sub, _, _ = oracle.render_pixels(cube0, lut, vmin, vmax, cam, 96, 96, 0.5, EA, ij)
    assert np.array_equal(sub, full[ij[:, 1], ij[:, 0]])


def test_far_face_never_reads_past_the_row():
    """p = hi must use cell n-2 with weight 1 (node-centred, no border mode): with
    NaN in column x = 0 a read of voxel x = n would pick up the next row's NaN."""
    V = np.random.RandomState(9).randn(5, 6, 7).astype(np.float32)
    V[:, :, 0] = np.nan
    for y, z in [(0.0, 0.0), (2.5, 1.25), (4.0, 3.0)]:
        got = oracle.sample_at(V, (6.0, y, z))
        assert np.isfinite(got)
    V = np.random.RandomState(9).randn(5, 6, 7).astype(np.float32)
    V[:, 0, :] = np.nan
    assert np.isfinite(oracle.sample_at(V, (3.3, 5.0, 2.0)))


# ---- S1: the aspect factor W/H multiplies the x screen coordinate ---------------------------------
def test_aspect_nonsquare_ortho():
    """Square pixels on a non-square image: a delta voxel's MIP footprint is 8 x 8 pixels at the predicted
    columns and rows.  asp divided instead of multiplied, or applied to y, changes the footprint (golden file)."""
    g = GOLD["aspect_nonsquare"]
    W, H = g["W"], g["H"]
    cx, cy, cz = g["voxel"]
    V = np.zeros((24, 48, 64), dtype=np.float32)
    V[cz, cy, cx] = 1.0
    lut, vmin, vmax = vi.lut_a()
    cam = {"eye": np.float32(g["eye"]), "right": np.float32([1, 0, 0]), "up": np.float32([0, 1, 0]),
           "forward": np.float32([0, 0, 1]), "projection": 1, "tan_half_fovy": 0.0, "ortho_half_height": g["hh"]}
    _, aux, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, MIP)
    lit = np.argwhere(aux > 0)                     # the cube is 0 elsewhere, rays outside it give -inf
    assert lit[:, 1].min() == g["cols"][0] and lit[:, 1].max() == g["cols"][1]
    assert lit[:, 0].min() == g["rows"][0] and lit[:, 0].max() == g["rows"][1]
    X = g["x_of_i"][0] * np.arange(W) + g["x_of_i"][1]
    Y = g["y_of_j"][0] * np.arange(H) + g["y_of_j"][1]
    want = (np.clip(1 - np.abs(Y - cy), 0, None)[:, None] * np.clip(1 - np.abs(X - cx), 0, None)[None, :]) * g["z_factor"]
    inside = np.isfinite(aux)
    assert np.abs(aux[inside] - want[inside]).max() < 1e-6
    assert aux.max() == pytest.approx(g["peak"], abs=1e-6)
    # the view window: 2 * hh * W / H = 64 voxels wide, so columns with x outside [0, 63] miss the cube
    assert np.array_equal(inside.any(axis=0), (X >= 0) & (X <= 63))
    assert np.array_equal(inside.any(axis=1), (Y >= 0) & (Y <= 47))


def test_aspect_nonsquare_perspective():
    """An off-axis voxel projects to the pixel the pinhole formula predicts on a 3:1 image."""
    g = GOLD["aspect_perspective"]
    W, H = g["W"], g["H"]
    cx, cy, cz = g["voxel"]
    V = np.zeros((40, 40, 60), dtype=np.float32)
    V[cz, cy, cx] = 1.0
    lut, vmin, vmax = vi.lut_a()
    cam = {"eye": np.float32(g["eye"]), "right": np.float32([1, 0, 0]), "up": np.float32([0, 1, 0]),
           "forward": np.float32([0, 0, 1]), "projection": 0, "tan_half_fovy": g["th"], "ortho_half_height": 0.0}
    _, aux, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.1, MIP)
    w = np.where(np.isfinite(aux), aux, 0.0).astype(np.float64)
    assert w.max() > 0.3                           # pixel pitch at the voxel is 0.75 voxel, centre between pixels
    jj, ii = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    ci, cj = (w * ii).sum() / w.sum(), (w * jj).sum() / w.sum()   # centroid of the (symmetric) footprint
    assert abs(ci - g["i"]) < 0.15 and abs(cj - g["j"]) < 0.15


# ---- W1: the display wall: K x L off-axis sub-frusta of one camera ---------------
@pytest.mark.parametrize("mode", [EA, MIP])
def test_wall_tiles_are_offaxis_subfrusta(mode):
    """Every tile of the wall against an INDEPENDENT float64 statement of the same thing: the camera's frustum cut to
    the window [a/K, (a+1)/K] x [b/L, (b+1)/L] of the image plane and sampled at the tile's own w x h pixel centres
    (tests/f64_bruteforce.py).  Swapped tile rows or columns, a tile sampled with its own aspect ratio, or pixel centres
    that do not line up across tiles all fail here."""
    rng = np.random.RandomState(5)
    V = rng.rand(10, 12, 14).astype(np.float32) * 2 - 1
    ramp = np.linspace(0, 1, 32)
    lut = np.stack([ramp, 1 - ramp, ramp ** 2, 0.3 * ramp], 1).astype(np.float32)
    W, H, K, L = 24, 18, 3, 2
    for cam in (vi.orbit_camera((14, 12, 10), 35.0, elevation_deg=25.0), vi.ortho_axis_camera((14, 12, 10), axis=1)):
        tiles, auxs, cnt = oracle.render_wall(V, lut, -1.0, 1.0, cam, W, H, K, L, 0.5, mode, tau=2.0)
        n = 0
        for b in range(L):
            for a in range(K):
                want, m, ns = bf.render(V, lut, -1.0, 1.0, cam, W // K, H // L, 0.5, mode, 2.0,
                                        window=(a / K, (a + 1) / K, b / L, (b + 1) / L, W / H))
                assert np.abs(tiles[b][a] - want).max() < 2e-5
                if mode == MIP:
                    has = np.isfinite(m)
                    assert np.array_equal(has, np.isfinite(auxs[b][a]))
                    assert np.abs(auxs[b][a][has] - m[has]).max() < 2e-5
                n += ns
        assert abs(cnt["samples"] - n) <= 0.002 * n          # grazing rays may differ by a sample between fp32 and fp64


def test_wall_is_the_frame_cut_into_tiles(cube0):
    """... and the tiles put side by side are the single frame, pixel for pixel (same rays, same arithmetic)."""
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[1]
    for (W, H, K, L) in [(96, 64, 4, 2), (60, 60, 1, 1), (30, 45, 5, 9), (16, 16, 16, 16)]:
        for mode in (EA, MIP):
            full, full_aux, c0 = oracle.render(cube0, lut, vmin, vmax, cam, W, H, 0.5, mode)
            tiles, auxs, c1 = oracle.render_wall(cube0, lut, vmin, vmax, cam, W, H, K, L, 0.5, mode)
            assert np.array_equal(np.block([[t for t in row] for row in [[x.reshape(H // L, -1) for x in r] for r in tiles]]),
                                  full.reshape(H, -1))
            assert np.array_equal(np.block(auxs), full_aux)
            assert c0 == c1
    with pytest.raises(ValueError):
        oracle.render_wall(cube0, lut, vmin, vmax, cam, 50, 40, 3, 2, 0.5, EA)      # 50 % 3 != 0


# ---- C1: which sub-cubes a frame needs (saturation culling of the out-of-core path) ----------
def test_needed_bricks_closed_form():
    """Constant cube, rays along z, alpha per voxel 0.3: every ray stops after 26 samples = 13 voxels (closed form C2),
    so of the 4 x 4 x 4 bricks of 16^3 cells only the 16 of the first z layer hold an evaluated sample -- 26 samples of
    each of the rays that cross them -- and the frame is the unbricked one bit for bit."""
    g = GOLD["ert_constant_cube"]
    V = np.full((64, 64, 64), 0.25, dtype=np.float32)
    lut = const_lut(g["alpha_per_voxel"])
    cam = vi.config0_views()[0]
    ref, _, _ = oracle.render(V, lut, -1.0, 1.0, cam, 32, 32, g["step"], EA)
    img, _, cnt, bs = oracle.render_bricked_needed(V, lut, -1.0, 1.0, cam, 32, 32, g["step"], EA, 16)
    assert np.array_equal(img, ref)
    assert bs.shape == (4, 4, 4) and bs.sum() == cnt["samples"] == 32 * 32 * g["n_terminate"]
    assert np.all(bs[0] == 8 * 8 * g["n_terminate"]) and np.all(bs[1:] == 0)        # 8 x 8 rays per brick column
    # without termination every brick is needed: 126 samples per ray, 16 voxels = 32 samples per brick (30 in the last:
    # 63 voxels of chord)
    _, _, cnt2, bs2 = oracle.render_bricked_needed(V, lut, -1.0, 1.0, cam, 32, 32, g["step"], EA, 16, tau=2.0)
    assert np.all(bs2[:3] == 64 * 32) and np.all(bs2[3] == 64 * 30) and bs2.sum() == cnt2["samples"] == 32 * 32 * 126
    # MIP never saturates
    _, _, _, bs3 = oracle.render_bricked_needed(V, lut, -1.0, 1.0, cam, 32, 32, g["step"], MIP, 16)
    assert np.array_equal(bs3, bs2)


def test_needed_bricks_are_exactly_those_with_samples(cube0):
    """The per-brick counts against an independent count: the samples of the unbricked render, binned by the brick
    that owns their cell (float64 positions from tests/f64_bruteforce.py's rays), for rays that never saturate."""
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[1]
    W = H = 24
    B = 32
    _, _, cnt, bs = oracle.render_bricked_needed(cube0, lut, vmin, vmax, cam, W, H, 1.0, MIP, B)
    O, D = bf.rays(cam, W, H)
    tn, tf, hit = bf.clip(O, D, (64, 64, 64))
    want = np.zeros((2, 2, 2), dtype=np.int64)
    for k in range(200):
        t = tn + (k + 0.5) * 1.0
        act = hit & (t < tf)
        P = np.clip(O + t[..., None] * D, 0.0, 63.0)
        cell = np.minimum(np.floor(P).astype(int), 62) // B
        for c in cell[act]:
            want[c[2], c[1], c[0]] += 1
    assert abs(int(bs.sum()) - int(want.sum())) <= 4                       # grazing rays: fp32 vs fp64 chord ends
    assert np.abs(bs.astype(np.int64) - want).max() <= 8                   # samples within rounding of a brick face
    assert cnt["samples"] == bs.sum()


# ---- R23: anisotropic voxel spacing (RA / Dec and frequency have different units) -------------------
def test_spacing_constant_cube_closed_form():
    """Voxels 2 world units apart along z: the same 64 channels are a 126-unit chord, so with alpha = 0.025 per unit
    length A = 1 - 0.975^126 whatever the step, with 126 / step samples -- and with spacing (1, 1, 1) nothing changes."""
    V = np.ones((64, 64, 64), dtype=np.float32)
    lut, vmin, vmax = vi.lut_a()
    cam = dict(vi.config0_views()[0])
    cam["eye"] = np.float32([31.5, 31.5, -32.0])
    want = 1.0 - 0.975 ** 126
    for step in (0.5, 1.0):
        with oracle.voxel_spacing((1.0, 1.0, 2.0)):
            img, _, cnt = oracle.render(V, lut, vmin, vmax, cam, 32, 32, step, EA, tau=2.0)
        assert cnt["samples"] == 32 * 32 * int(126 / step)
        assert np.abs(img[..., 3] - want).max() < 1e-5 and np.abs(img[..., 0] - 0.5 * want).max() < 1e-5
    base, _, c0 = oracle.render(V, lut, vmin, vmax, cam, 32, 32, 0.5, EA, tau=2.0)
    with oracle.voxel_spacing((1.0, 1.0, 1.0)):
        same, _, c1 = oracle.render(V, lut, vmin, vmax, cam, 32, 32, 0.5, EA, tau=2.0)
    assert np.array_equal(base, same) and c0 == c1
    with pytest.raises(ValueError):
        with oracle.voxel_spacing((1.0, 0.0, 1.0)):
            pass


def test_spacing_stretches_the_footprint_of_a_voxel():
    """A single bright voxel under MIP, voxels 3 world units apart along x: its footprint is three times as wide in
    world units -- the value at world position X is (1 - |X / 3 - cx|)+ -- and unchanged along y."""
    cx, cy, cz = 5, 7, 4
    V = np.zeros((9, 16, 12), dtype=np.float32)
    V[cz, cy, cx] = 1.0
    lut, vmin, vmax = vi.lut_a()
    W, H, hh = 96, 64, 8.0
    # ortho along +z; the window is 24 x 16 world units, centred on world (16.5, 7.5): pixel pitch 0.25
    cam = {"eye": np.float32([16.5, 7.5, -5.0]), "right": np.float32([1, 0, 0]), "up": np.float32([0, 1, 0]),
           "forward": np.float32([0, 0, 1]), "projection": 1, "tan_half_fovy": 0.0, "ortho_half_height": hh}
    with oracle.voxel_spacing((3.0, 1.0, 1.0)):
        _, aux, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, MIP)
    X = 16.5 + ((2 * np.arange(W) + 1) / W - 1.0) * (W / H) * hh
    Y = 7.5 + (1.0 - (2 * np.arange(H) + 1) / H) * hh
    want = np.clip(1 - np.abs(Y - cy), 0, None)[:, None] * np.clip(1 - np.abs(X / 3.0 - cx), 0, None)[None, :] * 0.75
    inside = np.isfinite(aux)
    assert inside.sum() > 0.5 * W * H
    assert np.abs(aux[inside] - want[inside]).max() < 2e-6
    assert (aux > 0).sum() > 2.5 * 8 * 8                      # ~ 24 x 8 pixels lit instead of 8 x 8


def test_spacing_against_float64_bruteforce():
    rng = np.random.RandomState(17)
    V = rng.rand(9, 11, 13).astype(np.float32) * 2 - 1
    ramp = np.linspace(0, 1, 32)
    lut = np.stack([ramp, 1 - ramp, ramp ** 2, 0.2 * ramp], 1).astype(np.float32)
    sp = (1.5, 0.75, 2.5)
    world = tuple(int(np.ceil((n - 1) * s)) + 1 for n, s in zip((13, 11, 9), sp))       # the cube's extent in world units
    for cam in (vi.orbit_camera(world, 35.0, elevation_deg=25.0), vi.orbit_camera(world, 250.0, elevation_deg=-40.0),
                vi.ortho_axis_camera(world, axis=1)):
        for mode in (EA, MIP):
            with oracle.voxel_spacing(sp):
                img, aux, cnt = oracle.render(V, lut, -1.0, 1.0, cam, 20, 16, 0.4, mode, tau=2.0)
            want, m, ns = bf.render(V, lut, -1.0, 1.0, cam, 20, 16, 0.4, mode, 2.0, spacing=sp)
            assert cnt["rays_hit"] > 40
            assert np.abs(img - want).max() < 3e-5
            assert abs(cnt["samples"] - ns) <= 0.01 * ns + 4


# ---- R17b: blanked (non-finite) voxels -------------------------------------------------------------------------
def test_blanking_replaces_exactly_the_nonfinite_voxels():
    rng = np.random.RandomState(2)
    V = rng.randn(6, 7, 8).astype(np.float32)
    V[1, 2, 3] = np.nan; V[0, 0, 0] = np.inf; V[5, 6, 7] = -np.inf; V[3, 3, 3] = np.float32(3.4e38); V[2, 2, 2] = -0.0
    out, n = oracle.blank_nonfinite(V, -3.0)
    assert n == 3 and np.isnan(V[1, 2, 3])                      # the input is left alone
    want = V.copy()
    want[1, 2, 3] = want[0, 0, 0] = want[5, 6, 7] = -3.0
    assert np.array_equal(out, want) and np.signbit(out[2, 2, 2])
    # a blank under LUT-A's vmin contributes nothing: a column of NaNs leaves a constant cube's closed form untouched
    # where the ray does not cross it, and lowers the opacity where it does
    C = np.ones((64, 64, 64), dtype=np.float32)
    C[20:40, 32, 32] = np.nan
    B, _ = oracle.blank_nonfinite(C, -3.0)
    lut, vmin, vmax = vi.lut_a()
    img, _, _ = oracle.render(B, lut, vmin, vmax, vi.config0_views()[0], 64, 64, 0.5, EA)
    g = GOLD["constant_cube"]
    assert abs(img[0, 0, 3] - g["A"]) < 1e-5 and np.isfinite(img).all()
    assert img[..., 3].min() < g["A"] - 0.05
