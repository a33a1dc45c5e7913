"""CPU oracle for the spectral-cube ray caster -- TEST INFRASTRUCTURE ONLY.

ctypes binding of oracle/libvr_oracle.so (plain C99, see vr_oracle.h / .c).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package; it imports nothing from
paper_1001_2049_b200 and shares no code with the CUDA path.

Cameras are plain dicts (vr_inputs.cameras): eye/right/up/forward (3 floats
each), projection (0 perspective, 1 ortho), tan_half_fovy, ortho_half_height.
"""
import ctypes as C
import os

import numpy as np

MODE_EA, MODE_MIP = 0, 1


class _Camera(C.Structure):
    _fields_ = [("eye", C.c_float * 3), ("right", C.c_float * 3), ("up", C.c_float * 3),
                ("forward", C.c_float * 3), ("projection", C.c_int),
                ("tan_half_fovy", C.c_float), ("ortho_half_height", C.c_float)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        from .build import build as _build_lib
        path = _build_lib()
        L = C.CDLL(path)
        fp, ip, u64p = C.POINTER(C.c_float), C.POINTER(C.c_int), C.POINTER(C.c_ulonglong)
        cam = C.POINTER(_Camera)
        L.vro_set_voxel_spacing.argtypes = [C.POINTER(C.c_float * 3)]
        L.vro_blank_nonfinite.argtypes = [fp, C.c_long, C.c_float]
        L.vro_blank_nonfinite.restype = C.c_long
        L.vro_opacity_correct.argtypes = [fp, C.c_int, C.c_float, fp]
        L.vro_opacity_correct.restype = None
        common = [fp, C.c_int, C.c_int, C.c_int]
        tf = [fp, C.c_int, C.c_float, C.c_float]
        view = [cam, C.c_int, C.c_int, C.c_float, C.c_int, C.c_float]
        L.vro_render_pixels.argtypes = common + tf + view + [ip, C.c_long, fp, fp, u64p, C.c_int]
        L.vro_render_pixels_bricks.argtypes = ([C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_int] + tf + view
                                               + [ip, C.c_long, fp, fp, u64p, C.c_int])
        L.vro_render.argtypes = common + tf + view + [fp, fp, u64p, C.c_int]
        L.vro_render_wall.argtypes = (common + tf + [cam, C.c_int, C.c_int, C.c_int, C.c_int, C.c_float, C.c_int, C.c_float]
                                      + [C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), u64p, C.c_int])
        L.vro_render_bricked.argtypes = common + [C.c_int, C.c_int] + tf + view + [fp, fp, u64p, C.c_int]
        L.vro_render_bricked_needed.argtypes = common + [C.c_int] + tf + view + [fp, fp, u64p, u64p, C.c_int]
        L.vro_brick_order.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, cam, ip, ip]
        L.vro_brick_minmax.argtypes = common + [C.c_int, fp, fp]
        L.vro_sample_at.argtypes = common + [C.c_float, C.c_float, C.c_float]
        L.vro_sample_at.restype = C.c_float
        L.vro_classify_at.argtypes = [fp, fp, C.c_int, C.c_float, C.c_float, C.c_float, fp]
        L.vro_classify_at.restype = None
        _lib = L
    return _lib


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _cam(cam):
    c = _Camera()
    for k in ("eye", "right", "up", "forward"):
        v = np.asarray(cam[k], dtype=np.float32)
        getattr(c, k)[:] = [float(x) for x in v]
    c.projection = int(cam["projection"])
    c.tan_half_fovy = float(np.float32(cam.get("tan_half_fovy", 0.0)))
    c.ortho_half_height = float(np.float32(cam.get("ortho_half_height", 0.0)))
    return c


def _vol(V):
    V = np.ascontiguousarray(V, dtype=np.float32)
    assert V.ndim == 3, "volume is V[z][y][x]"
    nz, ny, nx = V.shape
    return V, nx, ny, nz


def _lut(lut):
    lut = np.ascontiguousarray(lut, dtype=np.float32)
    assert lut.ndim == 2 and lut.shape[1] == 4
    return lut


class voxel_spacing:
    """with oracle.voxel_spacing((sx, sy, sz)): ...   -- renders inside use that spacing (R23); (1, 1, 1) afterwards."""

    def __init__(self, s):
        self.s = tuple(float(v) for v in s)

    def __enter__(self):
        if lib().vro_set_voxel_spacing(C.byref((C.c_float * 3)(*self.s))):
            raise ValueError("oracle: spacing must be finite and > 0")
        return self

    def __exit__(self, *a):
        lib().vro_set_voxel_spacing(C.byref((C.c_float * 3)(1.0, 1.0, 1.0)))


def blank_nonfinite(V, value):
    """A copy of V with every non-finite voxel replaced by `value` (R17b), and how many there were."""
    out = np.array(V, dtype=np.float32, copy=True, order="C")
    n = lib().vro_blank_nonfinite(_fp(out), out.size, C.c_float(value))
    return out, int(n)


def n_bricks(n, B):
    return (n - 1 + B - 1) // B


def opacity_correct(lut, step):
    lut = _lut(lut)
    out = np.empty(lut.shape[0], dtype=np.float32)
    lib().vro_opacity_correct(_fp(lut), lut.shape[0], C.c_float(step), _fp(out))
    return out


def render(V, lut, vmin, vmax, cam, W, H, step, mode, tau=0.99, nthreads=0,
           bricked=0, compositor=False):
    """Full frame.  Returns (rgba[H,W,4], aux[H,W], counters dict)."""
    V, nx, ny, nz = _vol(V)
    lut = _lut(lut)
    out = np.empty((H, W, 4), dtype=np.float32)
    aux = np.empty((H, W), dtype=np.float32)
    cnt = (C.c_ulonglong * 3)()
    c = _cam(cam)
    if bricked:
        rc = lib().vro_render_bricked(_fp(V), nx, ny, nz, int(bricked), int(bool(compositor)),
                                      _fp(lut), lut.shape[0], vmin, vmax, C.byref(c), W, H,
                                      step, mode, tau, _fp(out), _fp(aux), cnt, nthreads)
    else:
        rc = lib().vro_render(_fp(V), nx, ny, nz, _fp(lut), lut.shape[0], vmin, vmax,
                              C.byref(c), W, H, step, mode, tau, _fp(out), _fp(aux), cnt, nthreads)
    if rc:
        raise ValueError(f"oracle: invalid argument (rc={rc})")
    return out, aux, {"rays_hit": cnt[0], "samples": cnt[1], "nominal": cnt[2]}


def render_bricked_needed(V, lut, vmin, vmax, cam, W, H, step, mode, B, tau=0.99, nthreads=0):
    """Fused brick-by-brick render (S12) plus the samples evaluated inside every brick:
    (rgba, aux, counters, brick_samples[nbz, nby, nbx]); a brick is needed for the frame iff its count is > 0 (C1)."""
    V, nx, ny, nz = _vol(V)
    lut = _lut(lut)
    out = np.empty((H, W, 4), dtype=np.float32)
    aux = np.empty((H, W), dtype=np.float32)
    cnt = (C.c_ulonglong * 3)()
    shape = (n_bricks(nz, B), n_bricks(ny, B), n_bricks(nx, B))
    bs = np.zeros(shape, dtype=np.uint64)
    c = _cam(cam)
    rc = lib().vro_render_bricked_needed(_fp(V), nx, ny, nz, int(B), _fp(lut), lut.shape[0], vmin, vmax, C.byref(c),
                                         W, H, step, mode, tau, _fp(out), _fp(aux), cnt,
                                         bs.ctypes.data_as(C.POINTER(C.c_ulonglong)), nthreads)
    if rc:
        raise ValueError(f"oracle: invalid argument (rc={rc})")
    return out, aux, {"rays_hit": cnt[0], "samples": cnt[1], "nominal": cnt[2]}, bs


def render_wall(V, lut, vmin, vmax, cam, W, H, K, L, step, mode, tau=0.99, nthreads=0):
    """The frame as a K x L display wall (W1).  Returns (rgba[L][K] of [h,w,4], aux[L][K] of [h,w], counters)."""
    V, nx, ny, nz = _vol(V)
    lut = _lut(lut)
    w, h = W // K, H // L
    outs = [[np.empty((h, w, 4), dtype=np.float32) for _ in range(K)] for _ in range(L)]
    auxs = [[np.empty((h, w), dtype=np.float32) for _ in range(K)] for _ in range(L)]
    po = (C.c_void_p * (K * L))(*[outs[b][a].ctypes.data for b in range(L) for a in range(K)])
    pa = (C.c_void_p * (K * L))(*[auxs[b][a].ctypes.data for b in range(L) for a in range(K)])
    cnt = (C.c_ulonglong * 3)()
    c = _cam(cam)
    rc = lib().vro_render_wall(_fp(V), nx, ny, nz, _fp(lut), lut.shape[0], vmin, vmax, C.byref(c), W, H, K, L,
                               step, mode, tau, po, pa, cnt, nthreads)
    if rc:
        raise ValueError(f"oracle: invalid argument (rc={rc})")
    return outs, auxs, {"rays_hit": cnt[0], "samples": cnt[1], "nominal": cnt[2]}


def render_pixels(V, lut, vmin, vmax, cam, W, H, step, mode, ij, tau=0.99, nthreads=0):
    """Only the pixels ij[npix,2] = (i, j).  Returns (rgba[npix,4], aux[npix], counters)."""
    V, nx, ny, nz = _vol(V)
    lut = _lut(lut)
    ij = np.ascontiguousarray(ij, dtype=np.int32)
    npix = ij.shape[0]
    out = np.empty((npix, 4), dtype=np.float32)
    aux = np.empty(npix, dtype=np.float32)
    cnt = (C.c_ulonglong * 3)()
    c = _cam(cam)
    rc = lib().vro_render_pixels(_fp(V), nx, ny, nz, _fp(lut), lut.shape[0], vmin, vmax,
                                 C.byref(c), W, H, step, mode, tau,
                                 ij.ctypes.data_as(C.POINTER(C.c_int)), npix,
                                 _fp(out), _fp(aux), cnt, nthreads)
    if rc:
        raise ValueError(f"oracle: invalid argument (rc={rc})")
    return out, aux, {"rays_hit": cnt[0], "samples": cnt[1], "nominal": cnt[2]}


def render_pixels_bricks(brick_ptrs, B, dims, lut, vmin, vmax, cam, W, H, step, mode, ij, tau=0.99, nthreads=0):
    """render_pixels with the cube read from its brick store: brick_ptrs[bx + nbx*(by + nby*bz)] is
    the host address of brick b (dense float32, voxels [B*b, min(B*b+B, n-1)] per axis)."""
    nx, ny, nz = (int(v) for v in dims)
    total = n_bricks(nx, B) * n_bricks(ny, B) * n_bricks(nz, B)
    assert len(brick_ptrs) == total
    ptrs = (C.c_void_p * total)(*[int(p) for p in brick_ptrs])
    lut = _lut(lut)
    ij = np.ascontiguousarray(ij, dtype=np.int32)
    npix = ij.shape[0]
    out = np.empty((npix, 4), dtype=np.float32)
    aux = np.empty(npix, dtype=np.float32)
    cnt = (C.c_ulonglong * 3)()
    c = _cam(cam)
    rc = lib().vro_render_pixels_bricks(ptrs, int(B), nx, ny, nz, _fp(lut), lut.shape[0], vmin, vmax,
                                        C.byref(c), W, H, step, mode, tau,
                                        ij.ctypes.data_as(C.POINTER(C.c_int)), npix,
                                        _fp(out), _fp(aux), cnt, nthreads)
    if rc:
        raise ValueError(f"oracle: invalid argument (rc={rc})")
    return out, aux, {"rays_hit": cnt[0], "samples": cnt[1], "nominal": cnt[2]}


def brick_order(dims, B, cam):
    nx, ny, nz = dims
    total = n_bricks(nx, B) * n_bricks(ny, B) * n_bricks(nz, B)
    order = np.empty(total, dtype=np.int32)
    keys = np.empty(total, dtype=np.int32)
    c = _cam(cam)
    ip = C.POINTER(C.c_int)
    rc = lib().vro_brick_order(nx, ny, nz, B, C.byref(c), order.ctypes.data_as(ip),
                               keys.ctypes.data_as(ip))
    if rc:
        raise ValueError("oracle: invalid argument")
    return order, keys


def brick_minmax(V, B):
    V, nx, ny, nz = _vol(V)
    shape = (n_bricks(nz, B), n_bricks(ny, B), n_bricks(nx, B))
    mn = np.empty(shape, dtype=np.float32)
    mx = np.empty(shape, dtype=np.float32)
    rc = lib().vro_brick_minmax(_fp(V), nx, ny, nz, B, _fp(mn), _fp(mx))
    if rc:
        raise ValueError("oracle: invalid argument")
    return mn, mx


def sample_at(V, p):
    V, nx, ny, nz = _vol(V)
    return float(lib().vro_sample_at(_fp(V), nx, ny, nz, C.c_float(p[0]), C.c_float(p[1]),
                                     C.c_float(p[2])))


def classify_at(lut, alpha_tab, vmin, vmax, v):
    lut = _lut(lut)
    alpha_tab = np.ascontiguousarray(alpha_tab, dtype=np.float32)
    out = np.empty(4, dtype=np.float32)
    lib().vro_classify_at(_fp(lut), _fp(alpha_tab), lut.shape[0], vmin, vmax, C.c_float(v), _fp(out))
    return out
