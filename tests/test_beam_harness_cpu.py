"""The beam kernel's per-thread code, run on the host and compared with the oracle (no GPU).

tests/beam_harness.cu compiles the host + device phases of the beam kernel (csrc/vr_beam_plan.h,
csrc/vr_beam_core.cuh: the slab plan, the box copy, the sample march) for the host and walks the
128 threads of every CTA through them exactly as raycast_beam_kernel's barriers order them.  The
image must equal the oracle's bit for bit (same samples, same order, same binary32 ops), no stage
or cube index may leave its array, every 16-byte copy must be aligned, and every voxel a sample
reads must have been copied by its own slab (the harness poisons the stage with NaN before each
copy).

The CTA body that orders those phases (csrc/vr_beam_cta.cuh: beam_cta, the function the kernel runs, written
against a context of barrier / vote / atomic operations) is run too: 128 OS threads per CTA with pthread
barriers, against the oracle here and under ThreadSanitizer in a stand-alone build, where a missing or
misplaced __syncthreads() shows up as a data race on the "shared memory".  What stays untested without a
GPU is only the binding of that context to the hardware (vr_beam.cu: __syncthreads, __any_sync,
__reduce_*_sync, shared atomics, the cp.async PTX) and the intrinsics behind the VR_* macros.
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

import oracle
import vr_inputs as vi

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "beam_harness.cu")
LIB = os.path.join(HERE, "libbeam_harness.so")
CSRC = os.path.join(HERE, "..", "paper_1001_2049_b200", "csrc")
STATS = ["rays_hit", "samples", "bad_read", "bad_write", "bad_global", "misaligned", "slabs_staged", "slabs_direct",
         "tiles", "tiles_direct", "floats_staged", "chunks16", "lds", "lds_wavefronts", "samples_staged", "box_floats",
         "lut_lds", "lut_wavefronts", "lut_skipped", "samples_interior", "slabs_empty"]


class _Camera(C.Structure):
    _fields_ = [("eye", C.c_float * 3), ("right", C.c_float * 3), ("up", C.c_float * 3),
                ("forward", C.c_float * 3), ("projection", C.c_int),
                ("tan_half_fovy", C.c_float), ("ortho_half_height", C.c_float)]


@pytest.fixture(scope="module")
def harness():
    deps = [SRC] + [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    if not os.path.exists(LIB) or any(os.path.getmtime(LIB) < os.path.getmtime(d) for d in deps):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        if not os.path.exists(nvcc):
            pytest.skip("nvcc not found")
        subprocess.run([nvcc, "-x", "cu", "-std=c++17", "-O1", "-fmad=false", "-gencode", "arch=compute_100a,code=sm_100a",
                        "-Xcompiler", "-fPIC,-fopenmp,-ffp-contract=off,-fno-fast-math,-Wno-unknown-pragmas",
                        "-diag-suppress", "550,20011,20014", "-shared", "-o", LIB, SRC, "-lpthread"], check=True)
    L = C.CDLL(LIB)
    fp = C.POINTER(C.c_float)
    L.beam_harness_render.argtypes = [fp, C.c_int, C.c_int, C.c_int, C.POINTER(_Camera), C.c_int, C.c_int, C.c_float,
                                      C.c_int, fp, C.c_int, C.c_float, C.c_float, C.c_float, C.c_int, C.c_int, C.c_int,
                                      fp, fp, C.POINTER(C.c_ulonglong)]
    L.beam_harness_render_threads.argtypes = L.beam_harness_render.argtypes
    L.beam_harness_check_div_magic.restype = C.c_ulonglong
    L.beam_harness_set_skip.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int]
    L.beam_harness_set_skip.restype = None
    assert L.beam_harness_n_stats() == len(STATS)
    return L


def run(L, V, cam, W, H, step, mode, lut, vmin, vmax, tau=0.99, stage=0, pad=-1, stride=1):
    V = np.ascontiguousarray(V, dtype=np.float32)
    nz, ny, nx = V.shape
    c = _Camera()
    for k in ("eye", "right", "up", "forward"):
        getattr(c, k)[:] = [float(x) for x in np.asarray(cam[k], dtype=np.float32)]
    c.projection = int(cam["projection"])
    c.tan_half_fovy = float(np.float32(cam.get("tan_half_fovy", 0.0)))
    c.ortho_half_height = float(np.float32(cam.get("ortho_half_height", 0.0)))
    lut = np.ascontiguousarray(lut, dtype=np.float32)
    out = np.zeros((H, W, 4), dtype=np.float32)
    aux = np.zeros((H, W), dtype=np.float32)
    st = (C.c_ulonglong * len(STATS))()
    fp = C.POINTER(C.c_float)
    rc = L.beam_harness_render(V.ctypes.data_as(fp), nx, ny, nz, C.byref(c), W, H, step, mode, lut.ctypes.data_as(fp),
                               lut.shape[0], vmin, vmax, tau, stage, pad, stride, out.ctypes.data_as(fp),
                               aux.ctypes.data_as(fp), st)
    assert rc == 0
    return out, aux, dict(zip(STATS, [int(v) for v in st]))


def run_threads(L, V, cam, W, H, step, mode, lut, vmin, vmax, tau=0.99, stage=0, pad=-1, teams=2):
    """The frame rendered by beam_cta itself, 128 threads per CTA.  Returns (rgba, aux, stats)."""
    V = np.ascontiguousarray(V, dtype=np.float32)
    nz, ny, nx = V.shape
    c = _Camera()
    for k in ("eye", "right", "up", "forward"):
        getattr(c, k)[:] = [float(x) for x in np.asarray(cam[k], dtype=np.float32)]
    c.projection = int(cam["projection"])
    c.tan_half_fovy = float(np.float32(cam.get("tan_half_fovy", 0.0)))
    c.ortho_half_height = float(np.float32(cam.get("ortho_half_height", 0.0)))
    lut = np.ascontiguousarray(lut, dtype=np.float32)
    out = np.zeros((H, W, 4), dtype=np.float32)
    aux = np.zeros((H, W), dtype=np.float32)
    st = (C.c_ulonglong * 6)()
    fp = C.POINTER(C.c_float)
    rc = L.beam_harness_render_threads(V.ctypes.data_as(fp), nx, ny, nz, C.byref(c), W, H, step, mode,
                                       lut.ctypes.data_as(fp), lut.shape[0], vmin, vmax, tau, stage, pad, teams,
                                       out.ctypes.data_as(fp), aux.ctypes.data_as(fp), st)
    assert rc == 0
    return out, aux, dict(zip(STATS[:6], [int(v) for v in st]))


def check_clean(st):
    assert st["bad_read"] == 0, "a sample formed a stage index outside the stage"
    assert st["bad_write"] == 0, "a copy wrote outside the stage"
    assert st["bad_global"] == 0, "a copy read outside the cube"
    assert st["misaligned"] == 0, "a 16-byte copy was not 16-byte aligned"


def check_against_oracle(L, V, cam, W, H, step, lut, vmin, vmax, tau=0.99, stage=0, pad=-1, want_staged=True):
    stats = {}
    for mode in (oracle.MODE_EA, oracle.MODE_MIP):
        ref, ref_aux, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, step, mode, tau=tau)
        got, aux, st = run(L, V, cam, W, H, step, mode, lut, vmin, vmax, tau=tau, stage=stage, pad=pad)
        check_clean(st)
        assert not np.isnan(got).any(), "a sample read a voxel its slab's copy did not bring"
        assert np.array_equal(got, ref), f"mode {mode}: max |dRGBA| = {np.abs(got - ref).max()}"
        assert np.array_equal(aux, ref_aux)
        assert st["samples"] == cnt["samples"] and st["rays_hit"] == cnt["rays_hit"]
        if want_staged and cnt["samples"]:
            assert st["samples_staged"] > 0.5 * st["samples"], "most samples should come from staged boxes"
        stats[mode] = st
    return stats


@pytest.fixture(scope="module")
def cube0():
    return vi.make_cube(0).numpy()


@pytest.fixture(scope="module")
def ragged():
    rng = np.random.default_rng(7)
    return rng.standard_normal((90, 50, 64)).astype(np.float32)      # V[z][y][x]: nx = 64, ny = 50, nz = 90


@pytest.mark.parametrize("view", [0, 1])
def test_config0_bitwise(harness, cube0, view):
    """configs[0]: 64^3, ortho 256 x 256 along the frequency axis and rotated 30 degrees, step 0.5."""
    lut, vmin, vmax = vi.lut_a()
    st = check_against_oracle(harness, cube0, vi.config0_views()[view], 256, 256, 0.5, lut, vmin, vmax)
    assert st[oracle.MODE_MIP]["slabs_direct"] == 0 and st[oracle.MODE_MIP]["tiles_direct"] == 0


@pytest.mark.parametrize("pad", [0, 1])
@pytest.mark.parametrize("azimuth", [0, 45, 90, 135, 180, 225, 270, 315])
def test_orbit_views_ragged_cube(harness, ragged, azimuth, pad):
    """Perspective orbit views (the configs[1]-[4] camera recipe) of a 64 x 50 x 90 cube, ragged 160 x 90 frame:
    z slabs, x slabs (transposing copy) and both marching senses."""
    lut, vmin, vmax = vi.lut_a()
    cam = vi.orbit_camera((64, 50, 90), azimuth)
    check_against_oracle(harness, ragged, cam, 165, 93, 0.5, lut, vmin, vmax, pad=pad)


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("flip", [False, True])
def test_axis_aligned_ortho(harness, ragged, axis, flip):
    """Views straight down each axis, both senses: rays with zero direction components, x / y / z slabs."""
    lut, vmin, vmax = vi.lut_a()
    dims = (64, 50, 90)
    cam = vi.ortho_axis_camera(dims, axis=axis)
    if flip:
        c = (np.asarray(dims, dtype=np.float64) - 1.0) / 2.0
        cam = dict(cam)
        cam["forward"] = -np.asarray(cam["forward"])
        cam["right"] = -np.asarray(cam["right"])
        cam["eye"] = (2.0 * c - np.asarray(cam["eye"], dtype=np.float64)).astype(np.float32)
    check_against_oracle(harness, ragged, cam, 96, 72, 0.5, lut, vmin, vmax)


@pytest.mark.parametrize("step", [0.25, 1.0, 0.7])
def test_steps_and_no_ert(harness, ragged, step):
    lut, vmin, vmax = vi.lut_a()
    cam = vi.orbit_camera((64, 50, 90), 30.0, elevation_deg=35.0)
    check_against_oracle(harness, ragged, cam, 128, 72, step, lut, vmin, vmax, tau=2.0)


@pytest.mark.parametrize("stage", [4096, 8192, 65536])
def test_stage_sizes(harness, ragged, stage):
    """A small stage forces the thinner depth sets and direct slabs; the pixels must not change."""
    lut, vmin, vmax = vi.lut_s()
    cam = vi.orbit_camera((64, 50, 90), 60.0)
    st = check_against_oracle(harness, ragged, cam, 80, 45, 0.5, lut, vmin, vmax, stage=stage, want_staged=False)
    if stage == 4096:
        assert st[oracle.MODE_MIP]["slabs_direct"] > 0, "the test should exercise direct slabs"


def test_eye_inside_and_wide_fov(harness, ragged):
    """Eye inside the cube with a wide field of view: tiles whose rays do not share a slab axis or sense go direct."""
    lut, vmin, vmax = vi.lut_a()
    cam = vi.orbit_camera((64, 50, 90), 20.0)
    cam = dict(cam)
    cam["eye"] = np.asarray([30.3, 22.1, 40.7], dtype=np.float32)
    cam["tan_half_fovy"] = 1.5
    check_against_oracle(harness, ragged, cam, 128, 96, 0.5, lut, vmin, vmax, tau=2.0, want_staged=False)
    cam["tan_half_fovy"] = 6.0                           # a 16 x 8 tile now spans tens of degrees
    st = check_against_oracle(harness, ragged, cam, 40, 24, 0.5, lut, vmin, vmax, tau=2.0, want_staged=False)
    assert st[oracle.MODE_MIP]["tiles_direct"] > 0


def test_tiny_cubes(harness):
    rng = np.random.default_rng(3)
    lut, vmin, vmax = vi.lut_a()
    for dims in [(4, 2, 2), (4, 3, 5), (8, 2, 3)]:
        V = rng.standard_normal((dims[2], dims[1], dims[0])).astype(np.float32)
        for az in (10.0, 100.0, 200.0):
            cam = vi.orbit_camera(dims, az)
            check_against_oracle(harness, V, cam, 40, 24, 0.25, lut, vmin, vmax, want_staged=False)


def test_miss_everything(harness, ragged):
    lut, vmin, vmax = vi.lut_a()
    cam = dict(vi.orbit_camera((64, 50, 90), 0.0))
    cam["forward"] = -np.asarray(cam["forward"])          # looks away from the cube
    got, aux, st = run(harness, ragged, cam, 64, 32, 0.5, oracle.MODE_EA, lut, vmin, vmax)
    assert st["rays_hit"] == 0 and st["samples"] == 0 and not got.any()


@pytest.mark.parametrize("azimuth", [0.0, 45.0, 90.0])
def test_config1_geometry_statistics(harness, azimuth):
    """configs[1] geometry (512 x 512 x 1024, 1920 x 1080, step 0.5) on every 8th tile of an all-zero cube:
    the plan must stage every slab in the default 32 KiB stage, and the modelled shared-memory traffic
    must stay near one wavefront per warp-wide load."""
    dims = (512, 512, 1024)
    V = np.zeros((dims[2], dims[1], dims[0]), dtype=np.float32)
    lut, vmin, vmax = vi.lut_a()
    cam = vi.orbit_camera(dims, azimuth)
    got, aux, st = run(harness, V, cam, 1920, 1080, 0.5, oracle.MODE_MIP, lut, vmin, vmax, stride=8)
    check_clean(st)
    assert not np.isnan(got).any()
    assert st["samples"] > 1e7 and st["slabs_direct"] == 0 and st["tiles_direct"] == 0
    wf = st["lds_wavefronts"] / st["lds"]
    staged_bytes_per_sample = 4.0 * st["floats_staged"] / st["samples"]
    print(f"azimuth {azimuth}: {st['samples']} samples, {wf:.2f} wavefronts / LDS, "
          f"{staged_bytes_per_sample:.2f} B staged / sample, {st['slabs_staged']} slabs")
    assert wf < 2.5
    assert staged_bytes_per_sample < 16.0


CTA_CASES = [(c, s) for c in ("config0_rotated", "orbit_x_slabs", "orbit_z_slabs", "wide_fov_inside", "small_stage")
             for s in (1, 2)] + [("orbit_z_slabs", 1 + 128), ("orbit_z_slabs", 2 + 128), ("small_stage", 2 + 128)]


@pytest.mark.parametrize("case,stages", CTA_CASES,
                         ids=[f"{c}-{s & 3}stage{'-bulk' if s & 128 else ''}" for c, s in CTA_CASES])
def test_cta_body_with_threads(harness, cube0, ragged, case, stages):
    """beam_cta -- the code raycast_beam_kernel runs, barriers, votes and atomics included -- with 128 threads per
    CTA: bitwise the oracle's image, aux values and sample counts, no bad index."""
    lut, vmin, vmax = vi.lut_a()
    kw = {}
    if case == "config0_rotated":
        V, cam, W, H = cube0, vi.config0_views()[1], 96, 96
    elif case == "orbit_x_slabs":
        V, cam, W, H = ragged, vi.orbit_camera((64, 50, 90), 90.0), 100, 60
    elif case == "orbit_z_slabs":
        V, cam, W, H = ragged, vi.orbit_camera((64, 50, 90), 200.0), 100, 60
    elif case == "wide_fov_inside":
        cam = dict(vi.orbit_camera((64, 50, 90), 20.0))
        cam["eye"] = np.asarray([30.3, 22.1, 40.7], dtype=np.float32)
        cam["tan_half_fovy"] = 6.0
        V, W, H = ragged, 40, 24
        kw = dict(tau=2.0)
    else:
        V, cam, W, H = ragged, vi.orbit_camera((64, 50, 90), 60.0), 80, 45
        kw = dict(stage=4096)
    for mode in (oracle.MODE_EA, oracle.MODE_MIP):
        ref, ref_aux, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, 0.5, mode, tau=kw.get("tau", 0.99))
        got, aux, st = run_threads(harness, V, cam, W, H, 0.5, mode, lut, vmin, vmax, pad=1 + (64 if stages & 2 else 0) + (stages & 128),
                                   **{k: v for k, v in kw.items() if k != "pad"})
        check_clean(st)
        assert np.array_equal(got, ref), f"mode {mode}: max |dRGBA| = {np.abs(got - ref).max()}"
        assert np.array_equal(aux, ref_aux)
        assert st["samples"] == cnt["samples"] and st["rays_hit"] == cnt["rays_hit"]


def test_cta_body_under_thread_sanitizer():
    """The stand-alone ThreadSanitizer build of the harness: the threaded CTA body against the sequential harness
    on five views x two modes; any unsynchronised access to the CTA's shared memory is a reported data race."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not found")
    exe = os.path.join(HERE, "beam_harness_tsan")
    deps = [SRC] + [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    if not os.path.exists(exe) or any(os.path.getmtime(exe) < os.path.getmtime(d) for d in deps):
        r = subprocess.run([nvcc, "-x", "cu", "-std=c++17", "-O1", "-g", "-fmad=false", "-gencode",
                            "arch=compute_100a,code=sm_100a", "-DBEAM_HARNESS_MAIN", "-Xcompiler",
                            "-fPIE,-ffp-contract=off,-fno-fast-math,-Wno-unknown-pragmas,-fsanitize=thread",
                            "-diag-suppress", "550,20011,20014", "-o", exe, SRC, "-lpthread"],
                           capture_output=True, text=True)
        if r.returncode != 0:
            pytest.skip("ThreadSanitizer build not available: " + r.stderr[-300:])
    env = dict(os.environ, TSAN_OPTIONS="halt_on_error=1 exitcode=66")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=900)
    if r.returncode != 0 and "FATAL: ThreadSanitizer" in r.stderr:
        pytest.skip("ThreadSanitizer cannot run here: " + r.stderr[-200:])
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert "beam_cta threads OK" in r.stdout


def coloured_lut(n=256):
    """A transfer function whose three colour channels differ (the general two-read classification),
    with a stretch of zero alpha in the middle and a single zero-alpha entry elsewhere."""
    rng = np.random.default_rng(11)
    ramp = np.arange(n, dtype=np.float64) / (n - 1)
    lut = np.stack([ramp, 1.0 - 0.5 * ramp, 0.25 + 0.5 * np.sin(6.0 * ramp) ** 2, 0.2 * rng.random(n)], axis=1)
    lut[100:140, 3] = 0.0
    lut[200, 3] = 0.0
    return lut.astype(np.float32), -3.0, 5.0


@pytest.mark.parametrize("lutname", ["coloured", "grey_steep", "grey_ramp"])
@pytest.mark.parametrize("flags", [0, 16, 32, 48])
def test_classification_shortcuts_are_exact(harness, ragged, lutname, flags):
    """EA with and without the grey-LUT table (flag 16 off) and the zero-alpha bits (flag 32 off): the same
    image as the oracle, bit for bit, for a coloured LUT (never grey), the steep LUT-S (93 % of noise samples
    fall into zero-alpha cells) and LUT-A (alpha > 0 everywhere: the bits are empty)."""
    lut, vmin, vmax = {"coloured": coloured_lut, "grey_steep": vi.lut_s, "grey_ramp": vi.lut_a}[lutname]()
    cam = vi.orbit_camera((64, 50, 90), 115.0, elevation_deg=25.0)
    W, H = 96, 54
    ref, ref_aux, cnt = oracle.render(ragged, lut, vmin, vmax, cam, W, H, 0.5, oracle.MODE_EA)
    got, aux, st = run(harness, ragged, cam, W, H, 0.5, oracle.MODE_EA, lut, vmin, vmax, pad=1 + flags)
    check_clean(st)
    assert np.array_equal(got, ref), f"max |dRGBA| = {np.abs(got - ref).max()}"
    assert st["samples"] == cnt["samples"]
    got2, _, st2 = run_threads(harness, ragged, cam, W, H, 0.5, oracle.MODE_EA, lut, vmin, vmax, pad=1 + flags)
    assert np.array_equal(got2, ref) and st2["samples"] == cnt["samples"]


def test_lut_traffic_model(harness, ragged):
    """What the shortcuts buy, in modelled shared-memory wavefronts of the classification reads per warp-sample
    (a 16-byte load of 32 random LUT entries costs ~9 wavefronts, 4 if conflict-free): the grey table halves them,
    the zero bits of the steep LUT-S remove nearly all of them on noise."""
    cam = vi.orbit_camera((64, 50, 90), 30.0)
    res = {}
    for name, (lut, vmin, vmax) in {"a": vi.lut_a(), "s": vi.lut_s()}.items():
        for flags in (0, 16):
            _, _, st = run(harness, ragged, cam, 160, 90, 0.5, oracle.MODE_EA, lut, vmin, vmax, tau=2.0, pad=1 + flags)
            res[name, flags] = st
    warp_samples = res["a", 0]["lds"] / 8
    grey, general = res["a", 0]["lut_wavefronts"] / warp_samples, res["a", 16]["lut_wavefronts"] / warp_samples
    print(f"LUT-A: {grey:.1f} (grey table) vs {general:.1f} (two reads) LUT wavefronts per warp-sample; "
          f"LUT-S skips {res['s', 0]['lut_skipped'] / res['s', 0]['samples']:.3f} of the samples")
    assert res["a", 0]["lut_skipped"] == 0
    assert abs(general - 2.0 * grey) < 1e-6 and 4.0 <= grey <= 12.0
    assert res["s", 0]["lut_skipped"] > 0.9 * res["s", 0]["samples"]


def test_division_by_multiplication_is_exact(harness):
    """copy_box splits a chunk index with umulhi(e, 2^32 / d + 1): exact for every divisor and index a stage can hold."""
    assert harness.beam_harness_check_div_magic() == 0


def random_camera(rng, dims):
    """Any orthonormal basis (rolled, tilted), eye inside or outside the cube, perspective or orthographic."""
    n = np.asarray(dims, dtype=np.float64)
    c = (n - 1.0) / 2.0
    q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    right, up, fwd = q[:, 0], q[:, 1], q[:, 2]
    dist = rng.choice([0.2, 0.9, 1.6, 3.0]) * float(np.linalg.norm(n))
    eye = c - fwd * dist + rng.standard_normal(3) * 0.15 * n
    f32 = lambda v: np.asarray(v, dtype=np.float64).astype(np.float32)
    if rng.random() < 0.7:
        return {"eye": f32(eye), "right": f32(right), "up": f32(up), "forward": f32(fwd), "projection": 0,
                "tan_half_fovy": float(np.float32(rng.choice([0.15, 0.4, 0.9, 2.5]))), "ortho_half_height": 0.0}
    return {"eye": f32(eye), "right": f32(right), "up": f32(up), "forward": f32(fwd), "projection": 1,
            "tan_half_fovy": 0.0, "ortho_half_height": float(np.float32(rng.choice([0.3, 0.6, 1.1]) * n.max()))}


@pytest.mark.parametrize("seed", range(24))
def test_random_cameras(harness, seed):
    """Seeded random cubes, cameras (any roll and tilt, eye anywhere), steps and stage sizes: the beam code gives the
    oracle's image bit for bit and never forms a bad index, whatever the plan decides (staged, thinner sets, direct)."""
    rng = np.random.default_rng(1000 + seed)
    dims = (int(rng.choice([4, 8, 20, 36, 64])), int(rng.integers(2, 40)), int(rng.integers(2, 48)))
    V = rng.standard_normal((dims[2], dims[1], dims[0])).astype(np.float32)
    cam = random_camera(rng, dims)
    step = float(rng.choice([0.25, 0.5, 0.8, 1.0]))
    stage = int(rng.choice([4096, 8192, 16384, 32768]))
    lut, vmin, vmax = (vi.lut_a, vi.lut_s, coloured_lut)[seed % 3]()
    W, H = int(rng.integers(20, 72)), int(rng.integers(12, 44))
    check_against_oracle(harness, V, cam, W, H, step, lut, vmin, vmax, tau=float(rng.choice([0.99, 0.6, 2.0])),
                         stage=stage, want_staged=False)


def skip_bytes(V, lut, vmin, vmax, step, shift):
    """EA skip byte of every min/max brick (edge 2^shift cells), restated from DESIGN.md S9b in numpy: min / max over the
    brick's voxels plus a one-voxel ring, guard band 2^-20 * max(|min|, |max|), and alpha' = 0 on every LUT node from
    one below the cell of the guarded minimum to two above the cell of the guarded maximum."""
    nz, ny, nx = V.shape
    B = 1 << shift
    n = lut.shape[0]
    alpha = oracle.opacity_correct(lut, step)
    scale = np.float32((n - 1) / (float(vmax) - float(vmin)))
    nb = [(d - 1 + B - 1) // B for d in (nx, ny, nz)]
    out = np.zeros((nb[2], nb[1], nb[0]), dtype=np.uint8)
    for bz in range(nb[2]):
        for by in range(nb[1]):
            for bx in range(nb[0]):
                blk = V[max(B * bz - 1, 0):B * bz + B + 2, max(B * by - 1, 0):B * by + B + 2, max(B * bx - 1, 0):B * bx + B + 2]
                mn, mx = np.float32(blk.min()), np.float32(blk.max())
                guard = np.float32(max(abs(mn), abs(mx))) * np.float32(2.0 ** -20)
                xlo = np.clip((np.float32(mn - guard) - np.float32(vmin)) * scale, 0, n - 1)
                xhi = np.clip((np.float32(mx + guard) - np.float32(vmin)) * scale, 0, n - 1)
                qlo = max(min(int(xlo), n - 2) - 1, 0)
                qhi = min(min(int(xhi), n - 2) + 2, n - 1)
                out[bz, by, bx] = 1 if not alpha[qlo:qhi + 1].any() else 0
    return out, nb


@pytest.mark.parametrize("azimuth", [20.0, 110.0, 250.0])
def test_empty_slabs_are_skipped_exactly(harness, azimuth):
    """A10 in the beam kernel: on a noise-free cube (two blobs) under a LUT with alpha = 0 below a threshold most slabs
    are empty; skipping them leaves the EA image bit for bit the oracle's (which samples everything)."""
    dims = (64, 48, 72)
    z, y, x = np.meshgrid(np.arange(dims[2]), np.arange(dims[1]), np.arange(dims[0]), indexing="ij")
    V = (3.0 * np.exp(-((x - 20) ** 2 + (y - 18) ** 2 + (z - 25) ** 2) / 30.0)
         + 2.0 * np.exp(-((x - 45) ** 2 + (y - 30) ** 2 + (z - 55) ** 2) / 50.0)).astype(np.float32)
    lut, vmin, vmax = vi.lut_s()
    cam = vi.orbit_camera(dims, azimuth)
    W, H, step, shift = 120, 68, 0.5, 3
    skip, nb = skip_bytes(V, lut, vmin, vmax, step, shift)
    assert 0.3 < skip.mean() < 1.0
    ref, ref_aux, cnt = oracle.render(V, lut, vmin, vmax, cam, W, H, step, oracle.MODE_EA)
    harness.beam_harness_set_skip(skip.ctypes.data, nb[0], nb[1], nb[2], shift)
    try:
        got, aux, st = run(harness, V, cam, W, H, step, oracle.MODE_EA, lut, vmin, vmax)
        got2, _, st2 = run_threads(harness, V, cam, W, H, step, oracle.MODE_EA, lut, vmin, vmax, pad=1 + 64)
    finally:
        harness.beam_harness_set_skip(None, 0, 0, 0, 0)
    check_clean(st)
    assert st["slabs_empty"] > 0 and st["samples"] < cnt["samples"]
    assert np.array_equal(got, ref), f"max |dRGBA| = {np.abs(got - ref).max()}"
    assert np.array_equal(got2, ref)
    assert ref[..., 3].max() > 0.1, "the blobs must be visible for the test to mean anything"
