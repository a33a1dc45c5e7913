"""GPU parity at BASELINE.json's full sizes (configs[2], [3], [4]), on the layouts bench.py times them on
(VR_LAYOUT_TEX for the resident cubes -- configs[4]'s 8192 channels as five z chunks -- and VR_LAYOUT_LINEAR besides;
linear slots for the streamed cube): the frames are rendered whole, and seeded pixel subsets are checked one by one
against the CPU oracle (bitwise -- both sides run the same binary32 op sequence); properties that
hold at any size are checked on the whole frame.  Sorted after test_gpu_1_parity.py: `pytest -x` reaches the 32 GiB
cubes last.

configs[3] (4096^3, 256 GiB) needs more pinned host memory than the GPU box has (206 GB): the test
keeps its 512^3 bricks, seed, generator and source density and takes the largest near-cubic brick
grid that fits in VR_TEST_OOC_GB (default 40 GB -> 2048^3 = 64 bricks), with the
device pool capped at 3 slots so that every brick is streamed.  The oracle reads the same pinned
brick store (oracle.render_pixels_bricks)."""
import os

import numpy as np
import pytest

import oracle
import vr_inputs as vi

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

EA, MIP = 0, 1
LINEAR, TEX = 0, 1
# the beam kernel (VR_OPT_KERNEL = 2) is opt-in until it has run on hardware
TEST_BEAM = os.environ.get("VR_TEST_BEAM", "0") == "1"
TEST_BEAM_BULK = TEST_BEAM and os.environ.get("VR_TEST_BEAM_BULK", "0") == "1"     # bulk copies: their own gate


def check_beam_frames(vr, vol, cam, W, H, step, frames, aux):
    """VR_TEST_BEAM=1: the whole frame of the beam kernel, one and two stages, is bitwise the direct kernel's."""
    if not TEST_BEAM:
        return
    vol.set_option(vr.VR_OPT_SKIP, 0)
    for stages, bulk in ((1, 0), (2, 0)) + (((2, 1),) if TEST_BEAM_BULK else ()):
        vol.set_option(vr.VR_OPT_KERNEL, 2)
        vol.set_option(vr.VR_OPT_BEAM_STAGES, stages)
        vol.set_option(vr.VR_OPT_BEAM_BULK, bulk)
        for mode in (EA, MIP):
            img = vol.render(cam, W, H, step, mode).cpu().numpy()
            assert vol.stats()["kernel"] == 2
            assert np.array_equal(img, frames[mode][0]), f"beam kernel, {stages} stage(s), bulk {bulk}, mode {mode}: frame differs"
            assert np.array_equal(aux.cpu().numpy(), frames[mode][1])
    vol.set_option(vr.VR_OPT_KERNEL, 0)


@pytest.fixture(scope="module")
def vr():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_1001_2049_b200 as m
    m.lib()
    return m


def mem_available_bytes():
    for line in open("/proc/meminfo"):
        if line.startswith("MemAvailable:"):
            return int(line.split()[1]) * 1024
    return 0


def check_pixels(img, aux, ref, ref_aux, ij, mode):
    got = img[ij[:, 1], ij[:, 0]]
    d = float(np.abs(got - ref).max())
    assert d <= 1e-3, f"max |dRGBA| = {d}"
    assert np.array_equal(got, ref), f"not bitwise equal (max diff {d})"
    if mode == MIP:
        assert np.array_equal(aux[ij[:, 1], ij[:, 0]], ref_aux), "MIP values must match exactly"


def check_frame_properties(img, mode):
    assert np.isfinite(img).all() and img.min() >= 0.0 and img[..., 3].max() <= 1.0
    if mode == MIP:
        a = img[..., 3]
        assert np.all((a == 0.0) | (a == 1.0))


# ---- configs[2]: 2048^3 resident (32 GiB), 1080p / 4K, step 1.0 / 0.5, skipping on / off ----------
def test_config2_full_size(vr):
    spec = vi.CONFIGS[2]
    free, _ = torch.cuda.mem_get_info()
    if free < 110 * 2 ** 30 or mem_available_bytes() < 48 * 2 ** 30:
        pytest.skip("needs 110 GiB of HBM and 48 GiB of host memory")
    lut, vmin, vmax = vi.lut_a()
    Vd = vi.make_cube(spec, device="cuda")
    torch.cuda.synchronize()
    V = Vd.cpu().numpy()
    views = vi.orbit_views(spec.dims)
    cases = [(1920, 1080, 1.0, 1), (3840, 2160, 0.5, 6)]
    refs = {}
    for (W, H, step, view) in cases:
        ij = vi.tile_subset(W, H, n_tiles=16, tile=32, seed=2)
        for mode in (EA, MIP):
            ref, ref_aux, cnt = oracle.render_pixels(V, lut, vmin, vmax, views[view], W, H, step, mode, ij)
            assert cnt["rays_hit"] > 0.3 * len(ij)
            refs[(W, mode)] = (ij, ref, ref_aux)
    # TEX first: the layout bench.py times this cube on (2048 layers = the most one array holds)
    for layout in (TEX, LINEAR):
        with vr.Volume(spec.dims, layout=layout) as vol:
            vol.upload(Vd)
            torch.cuda.synchronize()
            vol.set_transfer_function(lut, vmin, vmax)
            for (W, H, step, view) in cases:
                cam = views[view]
                aux = vol.enable_aux(W, H)
                frames = {}
                for mode, skip in [(EA, 0), (EA, 1), (MIP, 0), (MIP, 1)]:
                    vol.set_option(vr.VR_OPT_SKIP, skip)
                    img = vol.render(cam, W, H, step, mode).cpu().numpy()
                    frames[(mode, skip)] = (img, aux.cpu().numpy())
                    check_frame_properties(img, mode)
                for mode in (EA, MIP):
                    ij, ref, ref_aux = refs[(W, mode)]
                    check_pixels(*frames[(mode, 0)], ref, ref_aux, ij, mode)
                    # exact empty-space skipping: the whole frame is bitwise the frame without it
                    assert np.array_equal(frames[(mode, 0)][0], frames[(mode, 1)][0])
                    assert np.array_equal(frames[(mode, 0)][1], frames[(mode, 1)][1])
                if layout == LINEAR:
                    check_beam_frames(vr, vol, cam, W, H, step, {m: frames[(m, 0)] for m in (EA, MIP)}, aux)
                vol.disable_aux()
            st = vol.stats()
            assert st["mm_bricks"] == 32 ** 3
            # noise cube under LUT-A: no 64^3 brick is skippable -- reported, not assumed
            assert st["bricks_skippable"] == 0
    del Vd
    torch.cuda.empty_cache()


# ---- configs[4]: 1024 x 1024 x 8192 (32 GiB), one 7680 x 4320 frame, step 0.25, steep LUT ---------
def test_config4_full_size(vr):
    spec = vi.CONFIGS[4]
    free, _ = torch.cuda.mem_get_info()
    if free < 110 * 2 ** 30 or mem_available_bytes() < 48 * 2 ** 30:
        pytest.skip("needs 110 GiB of HBM and 48 GiB of host memory")
    lut, vmin, vmax = vi.lut_s()
    W, H, step = 7680, 4320, 0.25
    cam = vi.orbit_views(spec.dims)[1]
    ij = vi.tile_subset(W, H, n_tiles=16, tile=32, seed=4)
    Vd = vi.make_cube(spec, device="cuda")
    torch.cuda.synchronize()
    V = Vd.cpu().numpy()
    refs = {}
    for mode in (EA, MIP):
        refs[mode] = oracle.render_pixels(V, lut, vmin, vmax, cam, W, H, step, mode, ij)
        assert refs[mode][2]["rays_hit"] >= 2048      # the elongated cube covers about a quarter of this frame
    for layout in (TEX, LINEAR):                      # TEX: 8192 channels = five z chunks of <= 2048 layers
        with vr.Volume(spec.dims, layout=layout) as vol:
            vol.upload(Vd)
            torch.cuda.synchronize()
            vol.set_transfer_function(lut, vmin, vmax)
            aux = vol.enable_aux(W, H)
            frames = {}
            for mode in (EA, MIP):
                img = vol.render(cam, W, H, step, mode).cpu().numpy()
                a = aux.cpu().numpy()
                frames[mode] = (img, a)
                check_frame_properties(img, mode)
                check_pixels(img, a, refs[mode][0], refs[mode][1], ij, mode)
            if layout == LINEAR:
                check_beam_frames(vr, vol, cam, W, H, step, frames, aux)
            # W1: the same frame as a 4 x 4 display wall of 1920 x 1080 tiles, one launch
            vol.disable_aux()
            for mode in (EA, MIP):
                tiles = vol.render_wall(cam, W, H, 4, 4, step, mode)
                for b in range(4):
                    for a in range(4):
                        assert np.array_equal(tiles[b * 4 + a].cpu().numpy(),
                                              frames[mode][0][b * 1080:(b + 1) * 1080, a * 1920:(a + 1) * 1920]), (a, b)
                del tiles
    del Vd
    torch.cuda.empty_cache()


# ---- configs[3]: out-of-core, 512^3 bricks streamed from pinned host memory ------------------------
def test_config3_streamed_full_bricks(vr):
    budget = float(os.environ.get("VR_TEST_OOC_GB", "40")) * 1e9
    if mem_available_bytes() < 1.6 * budget:
        pytest.skip("not enough host memory for the pinned brick store")
    spec = vi.ooc_spec(budget)
    B = 512
    lut, vmin, vmax = vi.lut_a()
    W, H, step = 1920, 1080, 0.5
    params = vi.source_params(spec)
    boxes = vi.brick_boxes(spec.dims, B)
    store = []
    for origin, size in boxes:                                   # generated brick by brick from the seed
        pb = vr.PinnedBrick((size[2], size[1], size[0]))
        blk = vi.make_box(spec, origin, size, device="cuda", params=vi.sources_in_box(spec, params, origin, size))
        torch.from_numpy(pb.array).copy_(blk)
        del blk
        store.append(pb)
    ptrs = [pb.data_ptr() for pb in store]
    ij = vi.tile_subset(W, H, n_tiles=16, tile=32, seed=3)
    try:
        with vr.Volume(spec.dims, host_brick=B, n_slots=3) as vol:
            vol.vr_volume_upload_bricks([(o, pb) for (o, _), pb in zip(boxes, store)])
            vol.set_transfer_function(lut, vmin, vmax)
            aux = vol.enable_aux(W, H)
            for view in (1, 4):
                cam = vi.orbit_views(spec.dims)[view]
                for mode in (EA, MIP):
                    img = vol.render(cam, W, H, step, mode).cpu().numpy()
                    a = aux.cpu().numpy()
                    st = vol.stats()
                    assert st["bricks_total"] == len(boxes) and st["n_slots"] == 3
                    assert 0 < st["bricks_streamed"] <= st["bricks_total"]
                    check_frame_properties(img, mode)
                    ref, ref_aux, cnt = oracle.render_pixels_bricks(ptrs, B, spec.dims, lut, vmin, vmax, cam, W, H,
                                                                    step, mode, ij)
                    assert cnt["rays_hit"] > 0.3 * len(ij)
                    check_pixels(img, a, ref, ref_aux, ij, mode)
                    if view == 1:
                        # 8(f)1: the same frame with brick culling (VR_OPT_STREAM_CULL) -- the whole frame is bitwise
                        # the unculled one, and with LUT-A on noise the rays saturate long before the far bricks
                        vol.set_option(vr.VR_OPT_STREAM_CULL, 1)
                        for rep in range(2):            # second pass: value ranges known (MIP culling by maximum)
                            img2 = vol.render(cam, W, H, step, mode).cpu().numpy()
                            st2 = vol.stats()
                            assert np.array_equal(img2, img) and np.array_equal(aux.cpu().numpy(), a)
                            assert st2["bricks_streamed"] + st2["bricks_cached"] + st2["bricks_culled"] + st2["bricks_empty"] <= len(boxes)
                        if mode == EA:
                            assert st2["bricks_culled"] > 0
                        assert st2["timing_valid"] == 1 and st2["h2d_gbs"] > 1.0
                        vol.set_option(vr.VR_OPT_STREAM_CULL, 0)
    finally:
        for pb in store:
            pb.close()
