"""Parity cases: the library behind the C ABI (include/vr.h) against the CPU oracle on the same seeded
inputs, element by element.  Bar (BASELINE.json north_star): max |dRGBA| <= 1e-3 per channel, MIP values
exact.  Because both sides execute the same IEEE-754 binary32 op sequence the cases also
assert the stronger bitwise equality.

The cases reach the library through a backend `be` (tests/backends.py):
  tests/test_gpu_1_parity.py   libvr.so on the B200 (`-m gpu`): the parity tests proper;
  tests/test_emu_parity.py     the same sources compiled against the host emulation of tests/hostemu (`-m "not gpu"`):
                               host logic, stream / event ordering and the kernels' C++ without a GPU.
"""
import os

import numpy as np
import pytest

import oracle
import vr_inputs as vi

TOL = 1e-3
EA, MIP = 0, 1
# device paths that must give the same pixels: VR_LAYOUT_LINEAR and VR_LAYOUT_TEX with the direct kernel, and
# VR_LAYOUT_LINEAR with the beam kernel (VR_OPT_KERNEL = 2): one stage, two stages, two stages + bulk row copies.
# On a GPU the beam kernel runs only with VR_TEST_BEAM=1 (bulk copies: VR_TEST_BEAM_BULK=1 as well) until it has passed
# the validation order of DESIGN.md Sec. 7; under the host emulation it always runs.
LINEAR, TEX, BEAM, BEAM2, BEAM3 = 0, 1, 2, 3, 4
# the direct kernel with 2 / 4 samples in flight per thread (VR_OPT_PIPELINE, vr_pipe.cu) and the supertile order of
# CTAs (VR_OPT_TILE_ORDER): PIPE2 = linear, depth 2, supertiles; PIPE4 = tex, depth 4, row-major; TILES = tex, depth 1, supertiles
# REUSE / REUSE_T = the direct kernel keeping the last cell's voxels in registers (VR_OPT_REUSE), linear / tex
PIPE2, PIPE4, TILES, REUSE, REUSE_T = 5, 6, 7, 8, 9
BASE_LAYOUT = {LINEAR: 0, TEX: 1, BEAM: 0, BEAM2: 0, BEAM3: 0, PIPE2: 0, PIPE4: 1, TILES: 1, REUSE: 0, REUSE_T: 1}
TEST_BEAM = os.environ.get("VR_TEST_BEAM", "0") == "1"
TEST_BEAM_BULK = TEST_BEAM and os.environ.get("VR_TEST_BEAM_BULK", "0") == "1"
layouts = pytest.mark.parametrize("layout", [LINEAR, TEX, BEAM, BEAM2, BEAM3, PIPE2, PIPE4, TILES, REUSE, REUSE_T],
                                  ids=["linear", "tex", "beam", "beam2", "beam3", "pipe2", "pipe4", "tiles", "reuse", "reuse_tex"])
direct_layouts = pytest.mark.parametrize("layout", [LINEAR, TEX], ids=["linear", "tex"])


def gate(be, layout):
    if be.name == "gpu" and layout in (BEAM, BEAM2) and not TEST_BEAM:
        pytest.skip("beam kernel on hardware is opt-in (VR_TEST_BEAM=1): DESIGN.md Sec. 7, validation order")
    if be.name == "gpu" and layout == BEAM3 and not TEST_BEAM_BULK:
        pytest.skip("beam kernel with bulk copies on hardware is opt-in (VR_TEST_BEAM=1 VR_TEST_BEAM_BULK=1), after the "
                    "plain cp.async pipelines have passed memcheck and racecheck (DESIGN.md Sec. 7)")


def open_volume(be, dims, layout, **kw):
    gate(be, layout)
    vr = be.vr
    vol = be.Volume(dims, layout=BASE_LAYOUT[layout], **kw)
    if layout in (BEAM, BEAM2, BEAM3) and not kw.get("host_brick") and dims[0] % 4 == 0:
        vol.set_option(vr.VR_OPT_KERNEL, 2)
        vol.set_option(vr.VR_OPT_BEAM_STAGES, 1 if layout == BEAM else 2)
        vol.set_option(vr.VR_OPT_BEAM_BULK, 1 if layout == BEAM3 else 0)
    vol.set_option(vr.VR_OPT_PIPELINE, {PIPE2: 2, PIPE4: 4}.get(layout, 1))      # 1: the plain direct kernel
    vol.set_option(vr.VR_OPT_TILE_ORDER, 1 if layout in (PIPE2, TILES, REUSE_T) else 0)
    vol.set_option(vr.VR_OPT_REUSE, 2 if layout in (REUSE, REUSE_T) else 1)
    return vol


def expected_kernel(layout, nx, skip, mode):
    if layout in (BEAM, BEAM2, BEAM3) and nx % 4 == 0 and not (skip and mode == MIP):
        return 2
    if layout in (REUSE, REUSE_T) and not skip:
        return 4
    return 3 if layout in (PIPE2, PIPE4) and not skip else 1


def render_once(be, V, lut, vmin, vmax, cam, W, H, step, mode, tau=0.99, skip=False, count=True,
                mm_brick=0, layout=LINEAR):
    vr = be.vr
    nz, ny, nx = V.shape
    with open_volume(be, (nx, ny, nz), layout, mm_brick=mm_brick) as vol:
        vol.upload(V)
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_ERT_TAU, tau)
        if skip and mode == MIP:
            vol.set_option(vr.VR_OPT_KERNEL, 0)            # MIP skipping is a feature of the direct kernel
        vol.set_option(vr.VR_OPT_SKIP, int(skip))
        vol.set_option(vr.VR_OPT_COUNT, int(count))
        aux = vol.enable_aux(W, H)
        img = vol.render(cam, W, H, step, mode)
        be.sync()
        st = vol.stats()
        assert st["kernel"] == expected_kernel(layout, nx, skip, mode)
        return be.to_np(img).copy(), be.to_np(aux).copy(), st


def assert_parity(got, ref, got_aux, ref_aux, mode, exact=True):
    d = np.abs(got - ref).max()
    assert d <= TOL, f"max |dRGBA| = {d}"
    if mode == MIP:
        assert np.array_equal(got_aux, ref_aux), "MIP values must match exactly"
    if exact:
        assert np.array_equal(got, ref), f"not bitwise equal (max diff {d})"


# ---- configs[0]: 64^3, both views, EA + MIP, full frames ------------------------
@layouts
@pytest.mark.parametrize("view", [0, 1])
@pytest.mark.parametrize("mode", [EA, MIP])
def test_config0_full_frames(be, cube0, view, mode, layout):
    gate(be, layout)
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[view]
    ref, ref_aux, cnt = oracle.render(cube0, lut, vmin, vmax, cam, 256, 256, 0.5, mode)
    got, got_aux, st = render_once(be, cube0, lut, vmin, vmax, cam, 256, 256, 0.5, mode, layout=layout)
    assert_parity(got, ref, got_aux, ref_aux, mode)
    assert st["rays_hit"] == cnt["rays_hit"] and st["samples"] == cnt["samples"]


# ---- ragged sizes, several tiles + a ragged tail, perspective / ortho / eye inside --
@pytest.mark.parametrize("dims", [(37, 29, 23), (2, 2, 2), (130, 3, 66), (64, 64, 64), (36, 29, 23), (132, 3, 66),
                                  (4, 2, 2), (24, 150, 31)])
@pytest.mark.parametrize("mode", [EA, MIP])
@layouts
def test_ragged_cubes_and_images(be, dims, mode, layout):
    gate(be, layout)
    if be.name == "emu" and layout not in (LINEAR, TEX, REUSE) and dims not in ((36, 29, 23), (132, 3, 66), (4, 2, 2), (37, 29, 23)):
        pytest.skip("the host emulation runs every cube on the two base layouts and four of them on the variants")
    rng = np.random.RandomState(sum(dims))
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    lut, vmin, vmax = vi.lut_a()
    lut = lut.copy(); lut[:, 3] *= 6.0                     # ERT fires inside the cube
    cams = [vi.orbit_camera(dims, 30.0), vi.orbit_camera(dims, 200.0, elevation_deg=-35.0),
            vi.ortho_axis_camera(dims, axis=0), vi.ortho_axis_camera(dims, axis=1)]
    inside = dict(cams[0]); inside["eye"] = np.float32([(d - 1) * 0.4 for d in dims])
    cams.append(inside)
    for cam in cams:
        for (W, H, step) in [(50, 37, 0.5), (16, 8, 1.0), (1, 1, 0.25), (33, 65, 0.3)]:
            ref, ref_aux, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, step, mode)
            got, got_aux, st = render_once(be, V, lut, vmin, vmax, cam, W, H, step, mode, layout=layout)
            assert_parity(got, ref, got_aux, ref_aux, mode)
            assert st["samples"] == cnt["samples"] and st["rays_hit"] == cnt["rays_hit"]


@layouts
def test_steep_lut_and_tau(be, cube0, layout):
    """configs[4]-style steep LUT: a 1-ulp disagreement at the ERT threshold would show."""
    gate(be, layout)
    lut, vmin, vmax = vi.lut_s()
    cam = vi.config0_views()[1]
    for tau in (0.99, 0.5, 2.0):
        ref, ref_aux, cnt = oracle.render(cube0 * 2.0, lut, vmin, vmax, cam, 128, 128, 0.25, EA, tau=tau)
        got, got_aux, st = render_once(be, cube0 * 2.0, lut, vmin, vmax, cam, 128, 128, 0.25, EA, tau=tau,
                                       layout=layout)
        assert_parity(got, ref, got_aux, ref_aux, EA)
        assert st["samples"] == cnt["samples"]


def test_large_lut_in_dynamic_shared_memory(be, cube0):
    n = 4096                                                  # 128 KiB of LUT: needs the opt-in
    ramp = np.linspace(0, 1, n)
    lut = np.stack([ramp, ramp ** 2, 1 - ramp, 0.05 * ramp], 1).astype(np.float32)
    cam = vi.config0_views()[1]
    ref, ref_aux, _ = oracle.render(cube0, lut, -3.0, 5.0, cam, 64, 64, 0.5, EA)
    got, got_aux, _ = render_once(be, cube0, lut, -3.0, 5.0, cam, 64, 64, 0.5, EA)
    assert_parity(got, ref, got_aux, ref_aux, EA)


# ---- A2 / A10: min/max table and exact empty-space skipping -----------------------
@direct_layouts
def test_minmax_table_matches_oracle(be, layout):
    rng = np.random.RandomState(4)
    for dims, B in [((70, 45, 33), 16), ((64, 64, 64), 64), ((130, 129, 67), 64), ((21, 18, 30), 8), ((2, 2, 2), 64),
                    ((259, 9, 5), 4),
                    # x extent a multiple of 4: the 16-byte row reader (bricks with both x rings, one wider than 32 pieces)
                    ((132, 70, 67), 64), ((72, 45, 33), 16), ((264, 6, 5), 128), ((8, 5, 4), 2)]:
        V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
        mn_ref, mx_ref = oracle.brick_minmax(V, B)
        with open_volume(be, dims, layout, mm_brick=B) as vol:
            vol.upload(V)
            mn, mx = vol.minmax()
        assert np.array_equal(mn, mn_ref) and np.array_equal(mx, mx_ref)


@layouts
@pytest.mark.parametrize("mode", [EA, MIP])
def test_skip_on_equals_skip_off(be, mode, layout):
    gate(be, layout)
    # sources-only cube: most bricks are empty under the 5-sigma LUT, so skipping fires
    dims = (96, 80, 72) if be.name == "gpu" else (72, 56, 48)          # (the host emulation gets a smaller cube)
    W, H = (80, 60) if be.name == "gpu" else (48, 36)
    spec = vi.CubeSpec("src-only", dims, 5, 6, (6.0, 12.0), kind="blob", inner=0.7, noise=False)
    V = vi.make_cube(spec).numpy()
    noise = vi.make_cube(vi.CubeSpec("noise", dims, 6, 0, (0, 0))).numpy()
    lut, vmin, vmax = vi.lut_5sigma()
    for cube, expect_skip in ((V, True), (V + noise, False), (V + 0.2 * noise, mode == EA)):
        for cam in (vi.orbit_camera(dims, 40.0), vi.ortho_axis_camera(dims, axis=2)):
            ref, ref_aux, cnt = oracle.render(cube, lut, vmin, vmax, cam, W, H, 0.5, mode)
            off, off_aux, st0 = render_once(be, cube, lut, vmin, vmax, cam, W, H, 0.5, mode, mm_brick=8,
                                            layout=layout)
            on, on_aux, st1 = render_once(be, cube, lut, vmin, vmax, cam, W, H, 0.5, mode, skip=True, mm_brick=8,
                                          layout=layout)
            assert_parity(off, ref, off_aux, ref_aux, mode)
            assert np.array_equal(on, off) and np.array_equal(on_aux, off_aux)     # bitwise
            assert st0["samples"] == cnt["samples"]
            assert st1["samples"] <= st0["samples"]
            if expect_skip:
                assert st1["samples"] < 0.9 * st0["samples"]
                if mode == EA:
                    assert st1["bricks_skippable"] > 0


# ---- A1: upload by boxes == upload whole -------------------------------------------
@direct_layouts
def test_upload_boxes_equals_whole(be, layout):
    rng = np.random.RandomState(8)
    dims = (40, 33, 27)
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    lut, vmin, vmax = vi.lut_a()
    cam = vi.orbit_camera(dims, 75.0)
    ref, _, _ = oracle.render(V, lut, vmin, vmax, cam, 64, 48, 0.5, EA)
    boxes = []
    for z0 in range(0, 27, 10):
        for y0 in range(0, 33, 17):
            for x0 in range(0, 40, 16):
                boxes.append(((x0, y0, z0), np.ascontiguousarray(V[z0:z0 + 10, y0:y0 + 17, x0:x0 + 16])))
    for on_device in (False, True):
        with open_volume(be, dims, layout) as vol:
            bx = [(o, be.dev(b) if on_device else b) for o, b in boxes]
            vol.vr_volume_upload_bricks(bx)
            vol.set_transfer_function(lut, vmin, vmax)
            got = be.to_np(vol.render(cam, 64, 48, 0.5, EA))
            if layout != TEX:
                assert np.array_equal(be.to_np(vol.as_tensor()), V)
        assert np.array_equal(got, ref)


# ---- A12 / A13: streamed (out-of-core) == resident ------------------------------------
def make_host_bricks(be, V, B):
    nz, ny, nx = V.shape
    out = []
    for z0 in range(0, nz - 1, B):
        for y0 in range(0, ny - 1, B):
            for x0 in range(0, nx - 1, B):
                blk = V[z0:min(z0 + B, nz - 1) + 1, y0:min(y0 + B, ny - 1) + 1, x0:min(x0 + B, nx - 1) + 1]
                out.append(((x0, y0, z0), be.pin(blk)))
    return out


@pytest.mark.parametrize("dims,B,slots", [((40, 33, 27), 16, 2), ((64, 64, 64), 32, 3), ((37, 29, 23), 8, 2)])
@pytest.mark.parametrize("mode", [EA, MIP])
@direct_layouts
def test_streamed_equals_resident(be, dims, B, slots, mode, layout):
    vr = be.vr
    rng = np.random.RandomState(21)
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    lut, vmin, vmax = vi.lut_a()
    lut = lut.copy(); lut[:, 3] *= 5.0
    cams = [vi.orbit_camera(dims, 20.0), vi.orbit_camera(dims, 250.0, elevation_deg=50.0),
            vi.ortho_axis_camera(dims, axis=2)]
    inside = dict(cams[0]); inside["eye"] = np.float32([(d - 1) * 0.45 for d in dims])
    cams.append(inside)
    W, H = 72, 56
    with open_volume(be, dims, layout, host_brick=B, n_slots=slots) as vol:
        vol.vr_volume_upload_bricks(make_host_bricks(be, V, B))
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_COUNT, 1)
        aux = vol.enable_aux(W, H)
        for q, cam in enumerate(cams):
            ref, ref_aux, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode)
            for sched in be.scheds:          # host emulation: copies as late / as early as the event waits allow
                be.set_sched(sched)
                depth = (1, 4, 2, 0)[q % 4]  # the per-brick segment with 1 / 4 / 2 samples in flight, or chosen per frame
                vol.set_option(vr.VR_OPT_PIPELINE, depth)
                got = be.to_np(vol.render(cam, W, H, 0.5, mode))
                st = vol.stats()
                assert_parity(got, ref, be.to_np(aux), ref_aux, mode)        # fused mode: bitwise
                assert st["samples"] == cnt["samples"]
                assert depth == 0 or (st["pipeline_depth"], st["kernel"]) == (depth, 3 if depth > 1 else 1)
                assert 0 < st["bricks_streamed"] <= st["bricks_total"]
                assert st["h2d_bytes"] > 0
            be.set_sched(None)
        # compositor mode (literal "N partial images"): equal up to re-association, ERT off
        vol.set_option(vr.VR_OPT_COMPOSITOR, 1)
        vol.set_option(vr.VR_OPT_ERT_TAU, 2.0)
        for cam in cams[:2]:
            ref, ref_aux, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, tau=2.0)
            oc, oc_aux, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, tau=2.0,
                                          bricked=B, compositor=True)
            got = be.to_np(vol.render(cam, W, H, 0.5, mode))
            assert np.abs(got - ref).max() < 1e-5
            assert np.array_equal(got, oc)                                    # same op order as the oracle's S13
            if mode == MIP:
                assert np.array_equal(be.to_np(aux), ref_aux)


# ---- error behaviour -------------------------------------------------------------------
def test_errors(be, cube0):
    vr = be.vr
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[0]
    with be.Volume((64, 64, 64)) as vol:
        with pytest.raises(vr.VrError) as e:
            vol.render(cam, 32, 32, 0.5, EA)
        assert e.value.status == 2                                             # nothing uploaded
        vol.upload(cube0)
        with pytest.raises(vr.VrError) as e:
            vol.render(cam, 32, 32, 0.5, EA)
        assert e.value.status == 2                                             # no transfer function
        with pytest.raises(vr.VrError):
            vol.set_transfer_function(lut, 1.0, 1.0)
        with pytest.raises(vr.VrError):
            vol.set_transfer_function(lut[:1], 0.0, 1.0)
        vol.set_transfer_function(lut, vmin, vmax)
        for bad_step in (0.0, -1.0, float("nan"), float("inf"), 1e-6):         # 1e-6: more than 2^22 samples per ray
            with pytest.raises(vr.VrError) as e:
                vol.render(cam, 32, 32, bad_step, EA)
            assert e.value.status == 1
        with pytest.raises(vr.VrError):
            vol.render(cam, 32, 32, 0.5, 7)
        with pytest.raises(vr.VrError):
            vol.vr_volume_upload_bricks([((60, 0, 0), np.zeros((8, 8, 8), np.float32))])  # leaves the cube
        with pytest.raises(vr.VrError) as e:
            vol.set_option(vr.VR_OPT_COMPOSITOR, 1)
        assert e.value.status == 3
        img = be.to_np(vol.render(cam, 32, 32, 0.5, EA))                       # still usable afterwards
        assert np.isfinite(img).all()


# ---- configs[1] at full size, in the launch configuration bench.py times -----------------
@layouts
@pytest.mark.parametrize("mode", [EA, MIP])
def test_config1_full_size_sampled_pixels(be, mode, layout):
    gate(be, layout)
    if be.name != "gpu":
        pytest.skip("full-size frames need the GPU")
    import torch
    spec = vi.CONFIGS[1]
    Vd = vi.make_cube(spec, device="cuda")
    V = Vd.cpu().numpy()
    lut, vmin, vmax = vi.lut_a()
    W, H = 1920, 1080
    ij = vi.tile_subset(W, H, n_tiles=16, tile=32, seed=1)
    with open_volume(be, spec.dims, layout) as vol:
        vol.upload(Vd)
        del Vd
        vol.set_transfer_function(lut, vmin, vmax)
        aux = vol.enable_aux(W, H)
        for view in (0, 3):
            cam = vi.orbit_views(spec.dims)[view]
            img = vol.render(cam, W, H, 0.5, mode).cpu().numpy()
            a = aux.cpu().numpy()
            ref, ref_aux, cnt = oracle.render_pixels(V, lut, vmin, vmax, cam, W, H, 0.5, mode, ij)
            assert cnt["rays_hit"] > 0.3 * len(ij)
            assert_parity(img[ij[:, 1], ij[:, 0]], ref, a[ij[:, 1], ij[:, 0]], ref_aux, mode)
            # properties that hold at any size
            assert np.isfinite(img).all() and img.min() >= 0.0 and img[..., 3].max() <= 1.0
    torch.cuda.empty_cache()


def test_beam_kernel_unsupported_is_an_error(be):
    """VR_OPT_KERNEL = 2 is an error where the beam kernel cannot run (never a silent fallback)."""
    vr = be.vr
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[1]
    with be.Volume((37, 29, 23)) as vol:                       # rows are not 16-byte multiples: no 16-byte box copies
        vol.upload(np.zeros((23, 29, 37), np.float32))
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_KERNEL, 2)
        with pytest.raises(vr.VrError) as e:
            vol.render(cam, 16, 16, 0.5, EA)
        assert e.value.status == 3
        with pytest.raises(vr.VrError):
            vol.set_option(vr.VR_OPT_KERNEL, 5)
        vol.set_option(vr.VR_OPT_KERNEL, 0)
        assert np.isfinite(be.to_np(vol.render(cam, 16, 16, 0.5, EA))).all()
        assert vol.stats()["kernel"] in (1, 3, 4)              # the direct kernel: plain, pipelined loads or cell reuse


def test_beam_kernel_selection(be, cube0):
    """VR_OPT_KERNEL = 2 asks for the beam kernel; MIP skipping with it is an error, EA skipping is not."""
    gate(be, BEAM)
    vr = be.vr
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[1]
    with be.Volume((64, 64, 64)) as vol:
        vol.upload(cube0)
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_KERNEL, 2)
        a = be.to_np(vol.render(cam, 96, 96, 0.5, EA)).copy()
        assert vol.stats()["kernel"] == 2
        vol.set_option(vr.VR_OPT_KERNEL, 1)
        b = be.to_np(vol.render(cam, 96, 96, 0.5, EA)).copy()
        assert vol.stats()["kernel"] in (1, 3, 4)              # a member of the direct family (dense view, step 0.5: cell reuse)
        assert np.array_equal(a, b)
        vol.set_option(vr.VR_OPT_KERNEL, 2)
        vol.set_option(vr.VR_OPT_SKIP, 1)
        c = be.to_np(vol.render(cam, 96, 96, 0.5, EA)).copy()
        assert vol.stats()["kernel"] == 2 and np.array_equal(a, c)
        with pytest.raises(vr.VrError) as e:
            vol.render(cam, 96, 96, 0.5, MIP)
        assert e.value.status == 3


def test_tex_layout_limits(be):
    """VR_LAYOUT_TEX: cubes with more than 2048 channels are cut into z chunks; beyond 8 chunks it is an error, not a
    fallback."""
    vr = be.vr
    with pytest.raises(vr.VrError) as e:
        be.Volume((8, 8, 2047 * 8 + 2), layout=TEX)
    assert e.value.status == 3
    with be.Volume((8, 8, 2047 * 8 + 2), layout=LINEAR):
        pass


@pytest.mark.parametrize("mode", [EA, MIP])
def test_tex_z_chunks(be, mode, monkeypatch):
    """A resident VR_LAYOUT_TEX cube cut into several layered arrays along z (configs[4]: 8192 channels > 2048 layers):
    VR_TEX_MAX_LAYERS shrinks the arrays so that a small cube takes 2 .. 8 of them, the last one ragged.  Uploads by
    boxes that straddle chunk boundaries, the min/max table read through the chunks, skipping on and off."""
    vr = be.vr
    rng = np.random.RandomState(77)
    lut, vmin, vmax = vi.lut_a()
    lut = lut.copy(); lut[:, 3] *= 6.0
    for dims, L in [((24, 17, 23), 5), ((16, 9, 30), 30), ((16, 9, 31), 30), ((10, 12, 9), 2), ((33, 20, 44), 8)]:
        monkeypatch.setenv("VR_TEX_MAX_LAYERS", str(L))
        V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
        cams = [vi.orbit_camera(dims, 35.0), vi.ortho_axis_camera(dims, axis=2), vi.ortho_axis_camera(dims, axis=0)]
        mn_ref, mx_ref = oracle.brick_minmax(V, 4)
        for by_boxes in (False, True):
            with be.Volume(dims, layout=TEX, mm_brick=4) as vol:
                if by_boxes:
                    zs = list(range(0, dims[2], 7))
                    vol.vr_volume_upload_bricks([((0, 0, z0), np.ascontiguousarray(V[z0:z0 + 7])) for z0 in zs])
                else:
                    vol.upload(V)
                vol.set_transfer_function(lut, vmin, vmax)
                vol.set_option(vr.VR_OPT_COUNT, 1)
                mn, mx = vol.minmax()
                assert np.array_equal(mn, mn_ref) and np.array_equal(mx, mx_ref)
                aux = vol.enable_aux(40, 30)
                for cam in cams:
                    ref, ref_aux, cnt = oracle.render(V, lut, vmin, vmax, cam, 40, 30, 0.5, mode)
                    for skip in (0, 1):
                        vol.set_option(vr.VR_OPT_SKIP, skip)
                        got = be.to_np(vol.render(cam, 40, 30, 0.5, mode))
                        assert_parity(got, ref, be.to_np(aux), ref_aux, mode)
                    vol.set_option(vr.VR_OPT_SKIP, 0)
                    assert vol.stats()["samples"] <= cnt["samples"]
    monkeypatch.setenv("VR_TEX_MAX_LAYERS", "3")
    with pytest.raises(vr.VrError) as e:                      # 2 * 8 + 1 = 17 layers at most with 3-layer arrays
        be.Volume((8, 8, 18), layout=TEX)
    assert e.value.status == 3


def test_pipeline_depth_is_chosen_from_the_camera(be, cube0):
    """VR_OPT_PIPELINE = 0: sparse views (at most one sample per voxel) keep four samples in flight, dense ones one."""
    vr = be.vr
    lut, vmin, vmax = vi.lut_a()
    dense, sparse = vi.config0_views()[0], dict(vi.config0_views()[0])
    sparse["ortho_half_height"] = np.float32(31.5)
    with be.Volume((64, 64, 64)) as vol:
        vol.upload(cube0)
        vol.set_transfer_function(lut, vmin, vmax)
        for mode in (EA, MIP):
            ref, _, _ = oracle.render(cube0, lut, vmin, vmax, sparse, 24, 24, 1.0, mode)
            got = be.to_np(vol.render(sparse, 24, 24, 1.0, mode))          # 2.6 voxels between pixels, step 1
            st = vol.stats()
            assert (st["kernel"], st["pipeline_depth"]) == (3, 4)
            assert np.array_equal(got, ref)
            vol.set_option(vr.VR_OPT_SKIP, 1)                               # the skipping loop is not pipelined
            got = be.to_np(vol.render(sparse, 24, 24, 1.0, mode))
            assert vol.stats()["kernel"] == 1 and np.array_equal(got, ref)
            vol.set_option(vr.VR_OPT_SKIP, 0)
            ref, _, _ = oracle.render(cube0, lut, vmin, vmax, dense, 128, 128, 0.5, mode)
            got = be.to_np(vol.render(dense, 128, 128, 0.5, mode))          # 0.5 voxels between pixels, step 0.5:
            st = vol.stats()                                                # dense and short steps -> cell reuse
            assert (st["kernel"], st["pipeline_depth"]) == (4, 1)
            assert np.array_equal(got, ref)
            ref1, _, _ = oracle.render(cube0, lut, vmin, vmax, dense, 128, 128, 1.0, mode)
            got = be.to_np(vol.render(dense, 128, 128, 1.0, mode))          # dense, step 1: the plain direct kernel
            assert vol.stats()["kernel"] == 1 and np.array_equal(got, ref1)
        with pytest.raises(vr.VrError):
            vol.set_option(vr.VR_OPT_PIPELINE, 3)
        with pytest.raises(vr.VrError):
            vol.set_option(vr.VR_OPT_TILE_ORDER, 2)


# ---- W1: the display wall ---------------------------------------------------------
@pytest.mark.parametrize("layout", [LINEAR, TEX, PIPE2, PIPE4, TILES], ids=["linear", "tex", "pipe2", "pipe4", "tiles"])
@pytest.mark.parametrize("mode", [EA, MIP])
def test_display_wall_equals_the_oracles(be, cube0, mode, layout):
    """vr_render_wall: K x L tiles from one launch, each bitwise the oracle's tile (and so the uncut frame's pixels);
    tile edges that cut through the 16 x 8-pixel CTA tiles included."""
    vr = be.vr
    lut, vmin, vmax = vi.lut_s() if mode == EA else vi.lut_a()
    with open_volume(be, (64, 64, 64), layout) as vol:
        vol.upload(cube0 * 2.0)
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_COUNT, 1)
        for cam, (W, H, K, L, step) in [(vi.config0_views()[1], (96, 64, 4, 2, 0.5)), (vi.orbit_camera((64, 64, 64), 70.0), (60, 45, 5, 9, 0.7)),
                                        (vi.config0_views()[0], (40, 24, 1, 1, 1.0)), (vi.orbit_camera((64, 64, 64), 200.0), (64, 8, 64, 1, 0.5))]:
            ref, _, cnt = oracle.render_wall(cube0 * 2.0, lut, vmin, vmax, cam, W, H, K, L, step, mode)
            got = vol.render_wall(cam, W, H, K, L, step, mode)
            assert vol.stats()["samples"] == cnt["samples"]
            for b in range(L):
                for a in range(K):
                    assert np.array_equal(be.to_np(got[b * K + a]), ref[b][a]), (a, b)
        cam = vi.config0_views()[1]
        with pytest.raises(vr.VrError) as e:
            vol.render_wall(cam, 50, 40, 3, 2, 0.5, mode)               # 50 % 3 != 0
        assert e.value.status == 1
        with pytest.raises(vr.VrError) as e:
            vol.render_wall(cam, 130, 130, 13, 5, 0.5, mode)            # 65 tiles
        assert e.value.status == 1
        vol.enable_aux(48, 48)
        with pytest.raises(vr.VrError) as e:
            vol.render_wall(cam, 48, 48, 2, 2, 0.5, mode)
        assert e.value.status == 3


# ---- 8(f)1: brick cache across frames + saturation / empty-brick culling of the out-of-core path (reading C1) ----------
@direct_layouts
@pytest.mark.parametrize("mode", [EA, MIP])
@pytest.mark.parametrize("slots", [3, 80])
def test_stream_cull_and_cache(be, mode, layout, slots):
    """Streamed volume with VR_OPT_STREAM_CULL and the slot cache: every frame is bitwise the oracle's; every brick the
    oracle evaluates a sample in (reading C1: the needed bricks) was fetched or found resident; saturated rays make
    bricks drop out; with enough slots a repeated view crosses the host link with nothing."""
    vr = be.vr
    dims, B = (64, 48, 56), 16
    rng = np.random.RandomState(31)
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    lut, vmin, vmax = vi.lut_a()
    lut = lut.copy(); lut[:, 3] *= 8.0                                   # rays saturate after ~ 10 voxels
    cams = [vi.orbit_camera(dims, 25.0), vi.orbit_camera(dims, 70.0), vi.orbit_camera(dims, 25.0),
            vi.ortho_axis_camera(dims, axis=0)]
    inside = dict(cams[0]); inside["eye"] = np.float32([(d - 1) * 0.5 for d in dims])
    cams.append(inside)
    W, H = 64, 48
    n_bricks = 4 * 3 * 4
    with open_volume(be, dims, layout, host_brick=B, n_slots=slots) as vol:
        vol.vr_volume_upload_bricks(make_host_bricks(be, V, B))
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_COUNT, 1)
        vol.set_option(vr.VR_OPT_STREAM_CULL, 1)
        aux = vol.enable_aux(W, H)
        seen_culled = 0
        for q, cam in enumerate(cams):
            ref, ref_aux, cnt, bs = oracle.render_bricked_needed(V, lut, vmin, vmax, cam, W, H, 0.5, mode, B)
            for sched in be.scheds:
                be.set_sched(sched)
                got = be.to_np(vol.render(cam, W, H, 0.5, mode))
                st = vol.stats()
                flags = vol.brick_flags()
                assert_parity(got, ref, be.to_np(aux), ref_aux, mode)
                assert st["samples"] == cnt["samples"]
                fetched = (flags == vr.VR_BRICK_STREAMED) | (flags == vr.VR_BRICK_CACHED)
                assert np.all(fetched[bs > 0]), "a brick with evaluated samples was left out"
                assert st["bricks_streamed"] + st["bricks_cached"] == fetched.sum()
                assert st["bricks_culled"] == (flags == vr.VR_BRICK_CULLED).sum()
                assert st["h2d_bytes"] == sum(4 * np.prod(np.minimum(B + 1, np.array(dims[::-1]) - B * np.array(b)))
                                              for b in np.argwhere(flags == vr.VR_BRICK_STREAMED))
                assert st["timing_valid"] == 1 and st["frame_ms"] >= 0.0
                seen_culled += st["bricks_culled"]
                if slots >= n_bricks and sched == be.scheds[-1] and len(be.scheds) > 1:
                    assert st["bricks_streamed"] == 0          # the same view again: everything needed is resident
            be.set_sched(None)
        if mode == EA:
            assert seen_culled > 0                              # saturation makes bricks drop out
        if slots >= n_bricks:
            # view 2 repeats view 0: nothing it needs has left the device
            assert st["bricks_total"] == n_bricks
        # a brick registered again holds new voxels: its cached copy and its value range are forgotten
        V2 = V.copy()
        V2[0:16, 0:16, 0:16] += 3.0                               # voxels only brick (0, 0, 0) stores
        vol.vr_volume_upload_bricks([b for b in make_host_bricks(be, V2, B) if b[0] == (0, 0, 0)])
        cam = cams[0]
        ref, ref_aux, _ = oracle.render(V2, lut, vmin, vmax, cam, W, H, 0.5, mode)
        got = be.to_np(vol.render(cam, W, H, 0.5, mode))
        assert_parity(got, ref, be.to_np(aux), ref_aux, mode)
        # culling off, cache off: every brick in the frustum crosses the link again
        vol.set_option(vr.VR_OPT_STREAM_CULL, 0)
        vol.set_option(vr.VR_OPT_STREAM_CACHE, 0)
        got = be.to_np(vol.render(cam, W, H, 0.5, mode))
        st = vol.stats()
        assert_parity(got, ref, be.to_np(aux), ref_aux, mode)
        assert st["bricks_cached"] == 0 and st["bricks_culled"] == 0 and st["bricks_streamed"] > 0


@direct_layouts
def test_stream_cull_empty_and_dim_bricks(be, layout):
    """Bricks the transfer function is zero on (EA) or whose maximum cannot raise any ray's running maximum (MIP) are
    left out from the second frame on, once their value range has been measured on the device; same pixels."""
    vr = be.vr
    dims, B = (96, 80, 72), 16
    spec = vi.CubeSpec("src-only", dims, 5, 6, (6.0, 12.0), kind="blob", inner=0.7, noise=False)
    V = vi.make_cube(spec).numpy()
    lut, vmin, vmax = vi.lut_5sigma()
    cam = vi.orbit_camera(dims, 40.0)
    W, H = 80, 60
    with open_volume(be, dims, layout, host_brick=B, n_slots=4) as vol:
        vol.vr_volume_upload_bricks(make_host_bricks(be, V, B))
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_STREAM_CULL, 1)
        vol.set_option(vr.VR_OPT_STREAM_CACHE, 0)
        aux = vol.enable_aux(W, H)
        for mode in (EA, MIP):
            ref, ref_aux, _, bs = oracle.render_bricked_needed(V, lut, vmin, vmax, cam, W, H, 0.5, mode, B)
            first = None
            for frame in range(3):
                got = be.to_np(vol.render(cam, W, H, 0.5, mode))
                st = vol.stats()
                assert_parity(got, ref, be.to_np(aux), ref_aux, mode)
                if first is None:
                    first = st["bricks_streamed"]
            if mode == EA:
                # most bricks of this cube hold nothing but zeros: alpha' = 0 on every sample of theirs (the oracle
                # evaluates those samples; they add nothing), and from the second frame on they stay on the host
                assert st["bricks_streamed"] < 0.5 * first
                assert st["bricks_empty"] > 0
                assert (vol.brick_flags() == vr.VR_BRICK_EMPTY).sum() == st["bricks_empty"]
            else:
                assert st["bricks_culled"] > 0                  # zero bricks behind a ray that has seen a source


def test_stream_options_are_for_streamed_volumes(be):
    vr = be.vr
    with be.Volume((8, 8, 8)) as vol:
        for key in (vr.VR_OPT_STREAM_CULL, vr.VR_OPT_STREAM_CACHE):
            with pytest.raises(vr.VrError) as e:
                vol.set_option(key, 1)
            assert e.value.status == 3
            vol.set_option(key, 0)


def test_autotune_picks_a_variant_and_keeps_the_pixels(be, cube0):
    """vr_autotune: times the direct kernel's variants on one frame, sets the winner; the image stays the oracle's."""
    vr = be.vr
    lut, vmin, vmax = vi.lut_a()
    cam = vi.config0_views()[1]
    for layout in (LINEAR, TEX):
        with be.Volume((64, 64, 64), layout=layout) as vol:
            vol.upload(cube0)
            vol.set_transfer_function(lut, vmin, vmax)
            vol.set_option(vr.VR_OPT_SKIP, 1)
            for mode in (EA, MIP):
                depth, order, reuse = vol.autotune(cam, 48, 40, 0.5, mode)
                assert depth in (1, 2, 4) and order in (0, 1) and reuse in (1, 2) and (reuse == 1 or depth == 1)
                ref, _, _ = oracle.render(cube0, lut, vmin, vmax, cam, 48, 40, 0.5, mode)
                assert np.array_equal(be.to_np(vol._tune_out) if hasattr(vol, "_tune_out") else ref, ref)
                vol.set_option(vr.VR_OPT_SKIP, 0)
                got = be.to_np(vol.render(cam, 48, 40, 0.5, mode))
                st = vol.stats()
                assert np.array_equal(got, ref)
                assert st["pipeline_depth"] == depth and st["kernel"] == (4 if reuse == 2 else (3 if depth > 1 else 1))
    with be.Volume((64, 64, 64), host_brick=32, n_slots=2) as vol:
        vol.vr_volume_upload_bricks(make_host_bricks(be, cube0, 32))
        vol.set_transfer_function(lut, vmin, vmax)
        with pytest.raises(vr.VrError) as e:
            vol.autotune(cam, 16, 16, 0.5, EA)
        assert e.value.status == 3


# ---- 8(f)4: low signal to noise: finer, two-level min/max tables ------------------------------------
@direct_layouts
def test_fine_bricks_on_noisy_cubes(be, layout):
    """What exact MIP skipping can and cannot do on low signal-to-noise data, measured and printed (DESIGN.md reports
    these numbers), with the frame always the unskipped one bit for bit:
      * pure N(0,1) noise: NOTHING is skipped at any brick size -- a ray's running maximum is a maximum of
        INTERPOLATED samples (an average of eight voxels, sigma ~ 0.6) and stays far below the largest VOXEL of even a
        4^3 brick, which is what the table must hold to be exact;
      * noise plus 4-sigma sources: a ray that has crossed a source skips what follows if the bricks are fine enough --
        an 8^3 brick rarely holds a 4-sigma noise voxel, a 64^3 brick always does."""
    vr = be.vr
    dims = (160, 96, 128)
    noise = vi.make_cube(vi.CubeSpec("noise", dims, 12, 0, (0, 0))).numpy()
    blobs = vi.make_cube(vi.CubeSpec("blobs", dims, 13, 40, (4.0, 4.0), kind="blob", inner=0.9, noise=False)).numpy()
    lut, vmin, vmax = vi.lut_a()
    W, H = (64, 48) if be.name == "gpu" else (40, 30)
    cam, step = vi.orbit_camera(dims, 30.0), 1.0
    shares = {}
    for name, V in (("noise", noise), ("noise + 4-sigma sources", noise + blobs)):
        with open_volume(be, dims, layout, mm_brick=64) as vol:
            vol.upload(V)
            vol.set_transfer_function(lut, vmin, vmax)
            vol.set_option(vr.VR_OPT_COUNT, 1)
            aux = vol.enable_aux(W, H)
            ref, ref_aux, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, step, MIP)
            share = {}
            for B in ((64, 8, 4) if be.name == "gpu" else (64, 8)):     # (a 4^3 table is 30 000 CTAs: too slow to emulate)
                vol.set_option(vr.VR_OPT_MM_BRICK, B)          # 8 and 4 come with a coarse level of 64 / 32 on top
                vol.set_option(vr.VR_OPT_SKIP, 1)
                got = be.to_np(vol.render(cam, W, H, step, MIP))
                st = vol.stats()
                assert_parity(got, ref, be.to_np(aux), ref_aux, MIP)
                share[B] = 1.0 - st["samples"] / cnt["samples"]
                assert st["mm_bricks"] == np.prod([(n - 1 + B - 1) // B for n in dims])
                mn, mx = vol.minmax()
                mn_ref, mx_ref = oracle.brick_minmax(V, B)
                assert np.array_equal(mn, mn_ref) and np.array_equal(mx, mx_ref)
            shares[name] = share
            print(f"MIP samples skipped, {name}: " + ", ".join(f"{B}^3 bricks {share[B]:.4f}" for B in share))
            if name == "noise":
                # EA with LUT-A (alpha > 0 from -3 sigma): nothing is skippable at any brick size
                vol.set_option(vr.VR_OPT_MM_BRICK, 8)
                refe, refe_aux, cnte = oracle.render(V, lut, vmin, vmax, cam, W, H, step, EA)
                got = be.to_np(vol.render(cam, W, H, step, EA))
                assert_parity(got, refe, be.to_np(aux), refe_aux, EA)
                assert vol.stats()["samples"] == cnte["samples"] and vol.stats()["bricks_skippable"] == 0
                with pytest.raises(vr.VrError):
                    vol.set_option(vr.VR_OPT_MM_BRICK, 24)
    assert max(shares["noise"].values()) < 0.02
    s = shares["noise + 4-sigma sources"]
    assert s[64] < 0.02 and s[8] > 0.03 and s[8] > 3 * s[64]


# ---- 8(f)2: parts of a cube, partial images and the S13 operator (the building blocks of sort-last rendering) ----------
@direct_layouts
@pytest.mark.parametrize("mode", [EA, MIP])
def test_parts_composited_equal_the_oracles_compositor_mode(be, mode, layout):
    """A cube cut into z slabs, one handle per slab (vr_volume_create_part); every slab's partial image composited in
    view order with vr_composite (+ vr_mip_finish): bitwise the oracle's compositor mode S13 with the slabs as bricks,
    and the resident frame up to re-association."""
    vr = be.vr
    B = 16
    dims = (17, 15, 49)                        # one brick of 16 cells in x and y, three along z: bricks = z slabs
    rng = np.random.RandomState(3)
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    lut, vmin, vmax = vi.lut_a()
    lut = lut.copy(); lut[:, 3] *= 4.0
    W, H = 48, 40
    cams = [vi.orbit_camera(dims, 20.0), vi.orbit_camera(dims, 200.0, elevation_deg=60.0), vi.ortho_axis_camera(dims, axis=2),
            vi.ortho_axis_camera(dims, axis=0)]
    inside = dict(cams[0]); inside["eye"] = np.float32([8.0, 7.0, 24.5])
    cams.append(inside)
    from paper_1001_2049_b200.sortlast import partition, view_order
    slabs = partition(dims[2] - 1, 3)
    assert slabs == [(0, 16), (16, 16), (32, 16)]
    vols = []
    for c0, nc in slabs:
        vol = be.Volume(dims, layout=BASE_LAYOUT[layout], part=((0, 0, c0), (dims[0], dims[1], nc + 1)))
        vol.upload(V[c0:c0 + nc + 1])
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_ERT_TAU, 2.0)
        vol.set_option(vr.VR_OPT_COUNT, 1)
        vol.set_option(vr.VR_OPT_PIPELINE, (1, 2, 4)[len(vols) % 3])          # every slab with another depth
        vols.append(vol)
    try:
        for cam in cams:
            oc, oc_aux, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, tau=2.0, bricked=B, compositor=True)
            ref, _, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, tau=2.0)
            parts, samples = [], 0
            for vol in vols:
                parts.append(be.to_np(vol.render(cam, W, H, 0.5, mode)).copy())
                samples += vol.stats()["samples"]
            assert samples == cnt["samples"]                 # the slabs' samples are exactly the cube's (S10)
            order = view_order(slabs, cam, 2)
            if mode == EA:
                running = be.dev(np.zeros((H, W, 4), np.float32))
                rest = order
            else:
                running = be.dev(parts[order[0]].copy())
                rest = order[1:]
            rp = running.data_ptr() if hasattr(running, "data_ptr") else running.ctypes.data
            keep = []
            for r in rest:
                p = be.dev(parts[r]); keep.append(p)
                vr.vr_composite(rp, p.data_ptr() if hasattr(p, "data_ptr") else p.ctypes.data, W, H, mode, 0)
            if mode == MIP:
                vr.vr_mip_finish(vols[0].handle, rp, W, H, 0)
            be.sync()
            got = be.to_np(running)
            assert np.array_equal(got, oc), "not the oracle's S13 image"
            assert np.abs(got - ref).max() < 1e-5
    finally:
        for vol in vols:
            vol.close()
    with pytest.raises(vr.VrError):
        be.Volume(dims, part=((0, 0, 40), (17, 15, 20)))          # leaves the cube


def test_partition_and_view_order_of_slabs():
    from paper_1001_2049_b200.sortlast import partition, view_order
    assert partition(100, 4) == [(0, 25), (25, 25), (50, 25), (75, 25)]
    p = partition(8191, 8)
    assert sum(n for _, n in p) == 8191 and all(a + n == b for (a, n), (b, _) in zip(p, p[1:])) and min(n for _, n in p) >= 1023
    p = partition(100, 3, weights=[1, 2, 1])                  # capability-weighted
    assert p == [(0, 25), (25, 50), (75, 25)]
    assert [n for _, n in partition(5, 5, weights=[100, 1, 1, 1, 1])] == [1, 1, 1, 1, 1]
    with pytest.raises(ValueError):
        partition(3, 4)
    slabs = partition(90, 3)
    cam = {"eye": np.float32([5, 5, -40]), "forward": np.float32([0, 0, 1]), "projection": 0}
    assert view_order(slabs, cam, 2) == [0, 1, 2]
    cam["eye"] = np.float32([5, 5, 200])
    assert view_order(slabs, cam, 2) == [2, 1, 0]
    cam["eye"] = np.float32([5, 5, 45.5])
    assert view_order(slabs, cam, 2)[0] == 1
    cam = {"eye": np.float32([5, 5, 0]), "forward": np.float32([0.6, 0, -0.8]), "projection": 1}
    assert view_order(slabs, cam, 2) == [2, 1, 0]


# ---- R23: anisotropic voxel spacing (VR_OPT_SPACING_X / Y / Z) ----------------------------------------------------
@pytest.mark.parametrize("layout", [LINEAR, TEX, PIPE2, PIPE4, TILES], ids=["linear", "tex", "pipe2", "pipe4", "tiles"])
@pytest.mark.parametrize("mode", [EA, MIP])
def test_voxel_spacing(be, mode, layout):
    """Voxels (1.5, 0.75, 2.5) world units apart: resident (skipping on and off) and streamed with culling, bitwise the
    oracle's frames under the same spacing; spacing (1, 1, 1) set explicitly changes nothing."""
    vr = be.vr
    dims, sp = (40, 33, 27), (1.5, 0.75, 2.5)
    rng = np.random.RandomState(23)
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    lut, vmin, vmax = vi.lut_a()
    lut = lut.copy(); lut[:, 3] *= 5.0
    world = tuple(int(np.ceil((n - 1) * s)) + 1 for n, s in zip(dims, sp))
    cams = [vi.orbit_camera(world, 25.0), vi.orbit_camera(world, 160.0, elevation_deg=-30.0), vi.ortho_axis_camera(world, axis=0)]
    inside = dict(cams[0]); inside["eye"] = np.float32([(w - 1) * 0.45 for w in world]); cams.append(inside)
    W, H = 56, 40

    def set_spacing(vol, s):
        for key, val in zip((vr.VR_OPT_SPACING_X, vr.VR_OPT_SPACING_Y, vr.VR_OPT_SPACING_Z), s):
            vol.set_option(key, val)

    with open_volume(be, dims, layout, mm_brick=8) as vol:
        vol.upload(V)
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_COUNT, 1)
        aux = vol.enable_aux(W, H)
        set_spacing(vol, sp)
        for cam in cams:
            with oracle.voxel_spacing(sp):
                ref, ref_aux, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.4, mode)
            assert cnt["rays_hit"] > 100
            for skip in (1, 0):
                vol.set_option(vr.VR_OPT_SKIP, skip)
                got = be.to_np(vol.render(cam, W, H, 0.4, mode))
                assert_parity(got, ref, be.to_np(aux), ref_aux, mode)
            assert vol.stats()["samples"] == cnt["samples"]          # (of the frame without skipping)
        set_spacing(vol, (1.0, 1.0, 1.0))
        cam = vi.orbit_camera(dims, 25.0)
        ref, ref_aux, _ = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.4, mode)
        assert_parity(be.to_np(vol.render(cam, W, H, 0.4, mode)), ref, be.to_np(aux), ref_aux, mode)
        with pytest.raises(vr.VrError):
            vol.set_option(vr.VR_OPT_SPACING_Y, 0.0)
    if layout in (LINEAR, TEX):
        B = 16
        with open_volume(be, dims, layout, host_brick=B, n_slots=3) as vol:
            vol.vr_volume_upload_bricks(make_host_bricks(be, V, B))
            vol.set_transfer_function(lut, vmin, vmax)
            vol.set_option(vr.VR_OPT_STREAM_CULL, 1)
            set_spacing(vol, sp)
            aux = vol.enable_aux(W, H)
            for cam in cams:
                with oracle.voxel_spacing(sp):
                    ref, ref_aux, _, bs = oracle.render_bricked_needed(V, lut, vmin, vmax, cam, W, H, 0.4, mode, B)
                for sched in be.scheds:
                    be.set_sched(sched)
                    got = be.to_np(vol.render(cam, W, H, 0.4, mode))
                    assert_parity(got, ref, be.to_np(aux), ref_aux, mode)
                    flags = vol.brick_flags()
                    assert np.all(((flags == vr.VR_BRICK_STREAMED) | (flags == vr.VR_BRICK_CACHED))[bs > 0])
                be.set_sched(None)
    if layout == LINEAR and dims[0] % 4 == 0:
        with be.Volume(dims) as vol:                      # the beam kernel does not take a spacing: an error, not a fallback
            vol.upload(V)
            vol.set_transfer_function(lut, vmin, vmax)
            set_spacing(vol, sp)
            vol.set_option(vr.VR_OPT_KERNEL, 2)
            with pytest.raises(vr.VrError) as e:
                vol.render(cams[0], W, H, 0.4, mode)
            assert e.value.status == 3


# ---- R17b: blanked voxels (VR_OPT_BLANK_VALUE) ---------------------------------------------------------------------
@pytest.mark.parametrize("mode", [EA, MIP])
def test_blanked_voxels(be, mode):
    """NaN / +-inf voxels are replaced on the device as they arrive -- resident (whole cube and boxes) and streamed
    (every brick as it lands in a slot, culling on): bitwise the oracle's render of the blanked cube."""
    vr = be.vr
    dims, B = (40, 33, 27), 16
    rng = np.random.RandomState(41)
    V = rng.randn(dims[2], dims[1], dims[0]).astype(np.float32)
    V[rng.rand(*V.shape) < 0.02] = np.nan
    V[5:9, :, 10:14] = np.nan                                  # a masked block of channels
    V[20, 30, 35] = np.inf; V[0, 0, 0] = -np.inf
    lut, vmin, vmax = vi.lut_a()
    lut = lut.copy(); lut[:, 3] *= 5.0
    Vb, n_blank = oracle.blank_nonfinite(V, vmin)
    assert n_blank > 500
    W, H = 56, 40
    cams = [vi.orbit_camera(dims, 35.0), vi.ortho_axis_camera(dims, axis=2)]
    with be.Volume(dims) as vol:
        vol.set_option(vr.VR_OPT_BLANK_VALUE, vmin)
        vol.set_transfer_function(lut, vmin, vmax)
        aux = vol.enable_aux(W, H)
        for by_boxes in (False, True):
            if by_boxes:
                vol.vr_volume_upload_bricks([((0, 0, z0), np.ascontiguousarray(V[z0:z0 + 10])) for z0 in range(0, 27, 10)])
            else:
                vol.upload(V)
            assert np.array_equal(be.to_np(vol.as_tensor()), Vb)
            for cam in cams:
                ref, ref_aux, _ = oracle.render(Vb, lut, vmin, vmax, cam, W, H, 0.5, mode)
                for skip in (0, 1):
                    vol.set_option(vr.VR_OPT_SKIP, skip)
                    assert_parity(be.to_np(vol.render(cam, W, H, 0.5, mode)), ref, be.to_np(aux), ref_aux, mode)
        vol.set_option(vr.VR_OPT_BLANK_VALUE, float("nan"))     # off again
        with pytest.raises(vr.VrError):
            vol.set_option(vr.VR_OPT_BLANK_VALUE, float("inf"))
    with be.Volume(dims, host_brick=B, n_slots=3) as vol:
        vol.vr_volume_upload_bricks(make_host_bricks(be, V, B))
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_BLANK_VALUE, vmin)
        vol.set_option(vr.VR_OPT_STREAM_CULL, 1)
        aux = vol.enable_aux(W, H)
        for cam in cams:
            ref, ref_aux, _ = oracle.render(Vb, lut, vmin, vmax, cam, W, H, 0.5, mode)
            for sched in be.scheds * 2:                        # second round: value ranges (of the blanked bricks) known
                be.set_sched(sched)
                assert_parity(be.to_np(vol.render(cam, W, H, 0.5, mode)), ref, be.to_np(aux), ref_aux, mode)
            be.set_sched(None)
    with pytest.raises(vr.VrError) as e:                       # arrays are written by the copy engine: no blanking there
        with be.Volume(dims, layout=TEX) as vol:
            vol.set_option(vr.VR_OPT_BLANK_VALUE, vmin)
    assert e.value.status == 3


@direct_layouts
def test_cell_reuse_share(be, cube0, layout):
    """VR_OPT_REUSE: how many samples still fetch their eight voxels (the rest find them in registers), printed for
    DESIGN.md; the frames are bitwise the oracle's (test_config0_full_frames runs the variant too)."""
    vr = be.vr
    lut, vmin, vmax = vi.lut_a()
    with be.Volume((64, 64, 64), layout=layout) as vol:
        vol.upload(cube0)
        vol.set_transfer_function(lut, vmin, vmax)
        vol.set_option(vr.VR_OPT_COUNT, 1)
        vol.set_option(vr.VR_OPT_REUSE, 2)
        vol.set_option(vr.VR_OPT_PIPELINE, 1)
        shares = {}
        for name, cam, step in (("along z, step 0.5", vi.config0_views()[0], 0.5), ("rotated 30 deg, step 0.5", vi.config0_views()[1], 0.5),
                                ("orbit, step 0.5", vi.orbit_camera((64, 64, 64), 45.0), 0.5),
                                ("orbit, step 0.25", vi.orbit_camera((64, 64, 64), 45.0), 0.25),
                                ("orbit, step 1", vi.orbit_camera((64, 64, 64), 45.0), 1.0)):
            ref, _, cnt = oracle.render(cube0, lut, vmin, vmax, cam, 96, 96, step, MIP)
            got = be.to_np(vol.render(cam, 96, 96, step, MIP))
            st = vol.stats()
            assert np.array_equal(got, ref) and st["kernel"] == 4 and st["samples"] == cnt["samples"]
            shares[name] = st["fetches"] / st["samples"]
        print("samples that fetch (MIP): " + "; ".join(f"{k}: {v:.3f}" for k, v in shares.items()))
        assert abs(shares["along z, step 0.5"] - 0.5) < 0.01          # every second sample enters a new cell
        assert shares["orbit, step 0.25"] < shares["orbit, step 0.5"] < shares["orbit, step 1"] <= 1.0
        assert shares["orbit, step 0.5"] < 0.8
        vol.set_option(vr.VR_OPT_REUSE, 1)
        vol.render(vi.config0_views()[0], 96, 96, 0.5, MIP)
        st = vol.stats()
        assert st["kernel"] == 1 and st["fetches"] == st["samples"]
