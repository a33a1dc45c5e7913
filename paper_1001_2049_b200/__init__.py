"""paper_1001_2049_b200 -- B200-native ray-cast volume rendering of spectral cubes.

Thin ctypes binding of the C-ABI library libvr.so (include/vr.h): argument
marshalling only, every step of the path runs in the CUDA kernels.  PyTorch is
used for device memory and streams, nothing else.  There is no CPU fallback:
importing works without a GPU (so the ABI can be inspected), but creating a
volume needs a CUDA device and a built libvr.so, and fails loudly otherwise.

The module-level functions carry the C names (vr_volume_create, ...); `Volume`
is a small convenience wrapper whose methods call exactly those.
Reference: PAPER.md:56-63 (Sec. 3.1, frame pipeline steps 1-5).
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvr.so")

VR_OK = 0
VR_MODE_EA, VR_MODE_MIP = 0, 1
VR_PROJ_PERSPECTIVE, VR_PROJ_ORTHO = 0, 1
VR_LAYOUT_LINEAR, VR_LAYOUT_TEX = 0, 1
(VR_OPT_ERT_TAU, VR_OPT_SKIP, VR_OPT_KERNEL, VR_OPT_COUNT, VR_OPT_COMPOSITOR, VR_OPT_STREAM_CULL,
 VR_OPT_BEAM_STAGE, VR_OPT_BEAM_PAD, VR_OPT_BEAM_STAGES, VR_OPT_BEAM_BULK, VR_OPT_PIPELINE,
 VR_OPT_TILE_ORDER, VR_OPT_STREAM_CACHE, VR_OPT_MM_BRICK, VR_OPT_SPACING_X, VR_OPT_SPACING_Y,
 VR_OPT_SPACING_Z, VR_OPT_BLANK_VALUE, VR_OPT_REUSE) = range(19)
VR_BRICK_OUTSIDE, VR_BRICK_EMPTY, VR_BRICK_CULLED, VR_BRICK_STREAMED, VR_BRICK_CACHED = 1, 2, 3, 4, 5
STATUS_NAMES = {0: "VR_OK", 1: "VR_ERR_INVALID_ARG", 2: "VR_ERR_STATE", 3: "VR_ERR_UNSUPPORTED",
                4: "VR_ERR_OOM_HOST", 5: "VR_ERR_OOM_DEVICE", 6: "VR_ERR_CUDA"}

# every symbol include/vr.h declares (tests check the library exports them all)
ABI_SYMBOLS = ["vr_volume_storage_bytes", "vr_volume_slot_bytes", "vr_volume_create", "vr_volume_create_part",
               "vr_composite", "vr_mip_finish",
               "vr_volume_destroy", "vr_volume_upload_bricks", "vr_set_transfer_function",
               "vr_set_option", "vr_set_aux_output", "vr_render", "vr_render_wall", "vr_autotune", "vr_render_host",
               "vr_get_minmax", "vr_get_stats", "vr_get_brick_flags", "vr_brick_order", "vr_last_error", "vr_version",
               "vr_host_alloc", "vr_host_free", "vr_beam_plan"]


class VrError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


class vr_camera(C.Structure):
    _fields_ = [("eye", C.c_float * 3), ("right", C.c_float * 3), ("up", C.c_float * 3),
                ("forward", C.c_float * 3), ("projection", C.c_int),
                ("tan_half_fovy", C.c_float), ("ortho_half_height", C.c_float)]


class vr_volume_desc(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("host_brick", C.c_int),
                ("mm_brick", C.c_int), ("device", C.c_int), ("d_storage", C.c_void_p),
                ("d_storage_bytes", C.c_size_t), ("layout", C.c_int), ("n_slots", C.c_int)]


class vr_stats(C.Structure):
    _fields_ = [("rays_hit", C.c_ulonglong), ("samples", C.c_ulonglong),
                ("bricks_total", C.c_ulonglong), ("bricks_streamed", C.c_ulonglong),
                ("bricks_skippable", C.c_ulonglong), ("h2d_bytes", C.c_ulonglong),
                ("mm_bricks", C.c_ulonglong), ("bricks_cached", C.c_ulonglong), ("bricks_culled", C.c_ulonglong),
                ("bricks_empty", C.c_ulonglong), ("fetches", C.c_ulonglong), ("frame_ms", C.c_double), ("h2d_ms", C.c_double),
                ("h2d_gbs", C.c_double), ("overlap_ratio", C.c_double), ("n_slots", C.c_int), ("kernel", C.c_int),
                ("beam_stage_bytes", C.c_int), ("pipeline_depth", C.c_int), ("timing_valid", C.c_int),
                ("reserved", C.c_int)]


_lib = None


def lib():
    """The loaded libvr.so with argument types set.  Raises if it was not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with "
                          "`python -m paper_1001_2049_b200.build` (there is no CPU fallback)")
    _lib = _bind(C.CDLL(LIB_PATH))
    return _lib


def _bind(L):
    """Sets the argument and result types of every include/vr.h entry point on a loaded library."""
    vp, i3 = C.c_void_p, C.POINTER(C.c_int * 3)
    fp, ip = C.POINTER(C.c_float), C.POINTER(C.c_int)
    L.vr_volume_storage_bytes.argtypes = [C.POINTER(vr_volume_desc)]
    L.vr_volume_storage_bytes.restype = C.c_size_t
    L.vr_volume_slot_bytes.argtypes = [C.POINTER(vr_volume_desc)]
    L.vr_volume_slot_bytes.restype = C.c_size_t
    L.vr_volume_create.argtypes = [C.POINTER(vr_volume_desc), C.POINTER(vp)]
    L.vr_volume_create_part.argtypes = [C.POINTER(vr_volume_desc), C.POINTER(C.c_int * 3), C.POINTER(C.c_int * 3), C.POINTER(vp)]
    L.vr_composite.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, vp]
    L.vr_mip_finish.argtypes = [vp, vp, C.c_int, C.c_int, vp]
    L.vr_volume_destroy.argtypes = [vp]
    L.vr_volume_destroy.restype = None
    L.vr_volume_upload_bricks.argtypes = [vp, C.c_int, i3, i3, C.POINTER(vp), C.c_int, vp]
    L.vr_set_transfer_function.argtypes = [vp, fp, C.c_int, C.c_float, C.c_float]
    L.vr_set_option.argtypes = [vp, C.c_int, C.c_double]
    L.vr_set_aux_output.argtypes = [vp, vp]
    L.vr_render.argtypes = [vp, C.POINTER(vr_camera), C.c_int, C.c_int, C.c_float, C.c_int, vp, vp]
    L.vr_render_wall.argtypes = [vp, C.POINTER(vr_camera), C.c_int, C.c_int, C.c_int, C.c_int, C.c_float, C.c_int,
                                 C.POINTER(vp), vp]
    L.vr_autotune.argtypes = [vp, C.POINTER(vr_camera), C.c_int, C.c_int, C.c_float, C.c_int, vp, vp, ip, ip, ip]
    L.vr_render_host.argtypes = [vp, C.POINTER(vr_camera), C.c_int, C.c_int, C.c_float, C.c_int,
                                 vp, vp, vp]
    L.vr_get_minmax.argtypes = [vp, fp, fp, vp]
    L.vr_get_stats.argtypes = [vp, C.POINTER(vr_stats)]
    L.vr_get_brick_flags.argtypes = [vp, ip]
    L.vr_brick_order.argtypes = [C.POINTER(vr_volume_desc), C.c_int, C.POINTER(vr_camera), ip, ip]
    L.vr_beam_plan.argtypes = [C.POINTER(vr_volume_desc), C.POINTER(vr_camera), C.c_int, C.c_int, C.c_int, C.c_int,
                               C.c_int, C.c_int, C.c_int, ip, ip]
    L.vr_host_alloc.argtypes = [C.c_size_t, C.POINTER(vp)]
    L.vr_host_free.argtypes = [vp]
    L.vr_host_free.restype = None
    L.vr_last_error.restype = C.c_char_p
    L.vr_version.restype = C.c_char_p
    return L


def _check(status):
    if status != VR_OK:
        raise VrError(status, lib().vr_last_error().decode())


def make_camera(cam):
    """dict (vr_inputs.cameras) or vr_camera -> vr_camera."""
    if isinstance(cam, vr_camera):
        return cam
    c = vr_camera()
    for k in ("eye", "right", "up", "forward"):
        getattr(c, k)[:] = [float(x) for x in np.asarray(cam[k], dtype=np.float32)]
    c.projection = int(cam["projection"])
    c.tan_half_fovy = float(np.float32(cam.get("tan_half_fovy", 0.0)))
    c.ortho_half_height = float(np.float32(cam.get("ortho_half_height", 0.0)))
    return c


def _desc(dims, host_brick=0, mm_brick=0, device=0, d_storage=0, d_storage_bytes=0,
          layout=VR_LAYOUT_LINEAR, n_slots=0):
    d = vr_volume_desc()
    d.nx, d.ny, d.nz = (int(v) for v in dims)
    d.host_brick, d.mm_brick, d.device = int(host_brick), int(mm_brick), int(device)
    d.d_storage, d.d_storage_bytes = d_storage, d_storage_bytes
    d.layout, d.n_slots = int(layout), int(n_slots)
    return d


# ---- the C calls, same names --------------------------------------------------
def vr_version():
    return lib().vr_version().decode()


def vr_volume_storage_bytes(dims, host_brick=0):
    return int(lib().vr_volume_storage_bytes(C.byref(_desc(dims, host_brick))))


def vr_volume_slot_bytes(dims, host_brick):
    return int(lib().vr_volume_slot_bytes(C.byref(_desc(dims, host_brick))))


def vr_volume_create(desc):
    h = C.c_void_p()
    _check(lib().vr_volume_create(C.byref(desc), C.byref(h)))
    return h


def vr_volume_create_part(desc, origin, dims):
    h = C.c_void_p()
    o = (C.c_int * 3)(*[int(x) for x in origin])
    d = (C.c_int * 3)(*[int(x) for x in dims])
    _check(lib().vr_volume_create_part(C.byref(desc), C.byref(o), C.byref(d), C.byref(h)))
    return h


def vr_composite(running_ptr, partial_ptr, width, height, mode, stream=0):
    _check(lib().vr_composite(C.c_void_p(running_ptr), C.c_void_p(partial_ptr), width, height, mode, C.c_void_p(stream)))


def vr_mip_finish(handle, running_ptr, width, height, stream=0):
    _check(lib().vr_mip_finish(handle, C.c_void_p(running_ptr), width, height, C.c_void_p(stream)))


def vr_volume_destroy(handle):
    lib().vr_volume_destroy(handle)


def vr_volume_upload_bricks(handle, origins, dims, ptrs, ptrs_are_device, stream=0):
    n = len(ptrs)
    o = (C.c_int * 3 * n)(*[(C.c_int * 3)(*map(int, q)) for q in origins])
    d = (C.c_int * 3 * n)(*[(C.c_int * 3)(*map(int, q)) for q in dims])
    p = (C.c_void_p * n)(*[int(q) for q in ptrs])
    _check(lib().vr_volume_upload_bricks(handle, n, o, d, p, int(ptrs_are_device), C.c_void_p(stream)))


def vr_set_transfer_function(handle, lut, vmin, vmax):
    lut = np.ascontiguousarray(lut, dtype=np.float32)
    if lut.ndim != 2 or lut.shape[1] != 4:
        raise ValueError("lut must be [n, 4] float32 RGBA")
    _check(lib().vr_set_transfer_function(handle, lut.ctypes.data_as(C.POINTER(C.c_float)),
                                          lut.shape[0], vmin, vmax))


def vr_set_option(handle, key, value):
    _check(lib().vr_set_option(handle, int(key), float(value)))


def vr_set_aux_output(handle, d_aux_ptr):
    _check(lib().vr_set_aux_output(handle, C.c_void_p(d_aux_ptr)))


def vr_render(handle, cam, width, height, step, mode, out_ptr, stream=0):
    c = make_camera(cam)
    _check(lib().vr_render(handle, C.byref(c), width, height, step, mode, C.c_void_p(out_ptr),
                           C.c_void_p(stream)))


def vr_render_wall(handle, cam, width, height, K, L, step, mode, out_ptrs, stream=0):
    c = make_camera(cam)
    p = (C.c_void_p * (K * L))(*[int(q) for q in out_ptrs])
    _check(lib().vr_render_wall(handle, C.byref(c), width, height, K, L, step, mode, p, C.c_void_p(stream)))


def vr_autotune(handle, cam, width, height, step, mode, out_ptr, stream=0):
    """-> (pipeline depth, tile order, cell reuse) now set on the handle."""
    c = make_camera(cam)
    p, t, r = C.c_int(0), C.c_int(0), C.c_int(0)
    _check(lib().vr_autotune(handle, C.byref(c), width, height, step, mode, C.c_void_p(out_ptr), C.c_void_p(stream),
                             C.byref(p), C.byref(t), C.byref(r)))
    return p.value, t.value, r.value


def vr_render_host(handle, cam, width, height, step, mode, d_staging_ptr, h_out_ptr, stream=0):
    c = make_camera(cam)
    _check(lib().vr_render_host(handle, C.byref(c), width, height, step, mode,
                                C.c_void_p(d_staging_ptr), C.c_void_p(h_out_ptr), C.c_void_p(stream)))


def vr_get_minmax(handle, n_bricks, stream=0):
    mn = np.empty(n_bricks, dtype=np.float32)
    mx = np.empty(n_bricks, dtype=np.float32)
    fp = C.POINTER(C.c_float)
    _check(lib().vr_get_minmax(handle, mn.ctypes.data_as(fp), mx.ctypes.data_as(fp), C.c_void_p(stream)))
    return mn, mx


def vr_get_stats(handle):
    s = vr_stats()
    _check(lib().vr_get_stats(handle, C.byref(s)))
    return {k: getattr(s, k) for k, _ in vr_stats._fields_}


def vr_get_brick_flags(handle, n_bricks):
    flags = np.zeros(n_bricks, dtype=np.int32)
    _check(lib().vr_get_brick_flags(handle, flags.ctypes.data_as(C.POINTER(C.c_int))))
    return flags


def vr_brick_order(dims, brick_edge, cam):
    n = 1
    for v in dims:
        n *= (int(v) - 1 + brick_edge - 1) // brick_edge
    order = np.empty(n, dtype=np.int32)
    keys = np.empty(n, dtype=np.int32)
    c = make_camera(cam)
    ip = C.POINTER(C.c_int)
    _check(lib().vr_brick_order(C.byref(_desc(dims)), int(brick_edge), C.byref(c),
                                order.ctypes.data_as(ip), keys.ctypes.data_as(ip)))
    return order, keys


def vr_beam_plan(dims, cam, W, H, tile_i, tile_j, stage_bytes=0, pad_mode=-1, max_slabs=4096):
    """Host-only diagnostic of the beam kernel: (info dict, slabs int array [n, 16])."""
    slabs = np.zeros((max_slabs, 16), dtype=np.int32)
    info = np.zeros(10, dtype=np.int32)
    c = make_camera(cam)
    ip = C.POINTER(C.c_int)
    _check(lib().vr_beam_plan(C.byref(_desc(dims)), C.byref(c), int(W), int(H), int(tile_i), int(tile_j),
                              int(stage_bytes), int(pad_mode), int(max_slabs),
                              slabs.ctypes.data_as(ip), info.ctypes.data_as(ip)))
    keys = ["axis", "pos", "cmin", "cmax", "n_slabs", "all_direct", "rays_hit", "stage_bytes", "fast", "pad_mode"]
    d = {k: int(v) for k, v in zip(keys, info)}
    return d, slabs[: min(d["n_slabs"], max_slabs)]


def vr_host_alloc(nbytes):
    p = C.c_void_p()
    _check(lib().vr_host_alloc(int(nbytes), C.byref(p)))
    return p.value


def vr_host_free(ptr):
    lib().vr_host_free(C.c_void_p(ptr))


class PinnedBrick:
    """A float32 [sz, sy, sx] array in pinned host memory from vr_host_alloc (exact size, no
    rounding); .array is a numpy view, .data_ptr() the address.  Freed on close() / garbage collection."""

    def __init__(self, shape):
        self.shape = tuple(int(v) for v in shape)
        n = int(np.prod(self.shape))
        self.ptr = vr_host_alloc(4 * n)
        self.array = np.ctypeslib.as_array((C.c_float * n).from_address(self.ptr)).reshape(self.shape)

    def data_ptr(self):
        return self.ptr

    def close(self):
        if getattr(self, "ptr", None):
            self.array = None
            vr_host_free(self.ptr)
            self.ptr = None

    __del__ = close


# ---- convenience wrapper ---------------------------------------------------------
class Volume:
    """A cube on one GPU.  Owns the torch tensor behind d_storage and the handle.

    resident:  Volume((nx, ny, nz))
    streamed:  Volume((nx, ny, nz), host_brick=512, n_slots=3)   (out-of-core)
    layout:    VR_LAYOUT_LINEAR (voxels in a torch tensor) or VR_LAYOUT_TEX (library-owned
               2D-layered CUDA arrays read with 4-texel gathers; same pixels, faster)
    """

    handle = None

    def __init__(self, dims, host_brick=0, mm_brick=0, device=0, n_slots=2, layout=VR_LAYOUT_LINEAR, part=None):
        """part = (origin, dims): a handle for that part of the cube `dims` (vr_volume_create_part, sort-last rendering)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1001_2049_b200 needs a CUDA device; there is no CPU fallback")
        self._torch = torch
        self.dims = tuple(int(v) for v in dims)
        self.host_brick = int(host_brick)
        self.device = int(device)
        self.layout = int(layout)
        n_slots = max(2, int(n_slots))
        if self.layout == VR_LAYOUT_TEX:
            self.storage = None
            self.desc = _desc(self.dims, host_brick, mm_brick, device, 0, 0, layout, n_slots)
        else:
            if host_brick:
                nbytes = vr_volume_slot_bytes(self.dims, host_brick) * n_slots
            elif part is not None:
                nbytes = vr_volume_storage_bytes(part[1])
            else:
                nbytes = vr_volume_storage_bytes(self.dims)
            if nbytes == 0:
                raise VrError(1, "every extent must be >= 2")
            self.storage = torch.empty(nbytes, dtype=torch.uint8, device=f"cuda:{device}")
            self.desc = _desc(self.dims, host_brick, mm_brick, device, self.storage.data_ptr(), nbytes,
                              layout, n_slots)
        self.part = None if part is None else (tuple(int(v) for v in part[0]), tuple(int(v) for v in part[1]))
        if self.part is not None:
            if host_brick:
                raise ValueError("a part of a cube is resident")
            self.handle = vr_volume_create_part(self.desc, self.part[0], self.part[1])
        else:
            self.handle = vr_volume_create(self.desc)
        self._keep = []          # host bricks / aux buffers that must outlive the handle
        self._aux = None
        mmB = mm_brick or 64
        self.mm_shape = tuple((n - 1 + mmB - 1) // mmB for n in reversed(self.dims))  # (nbz, nby, nbx)

    def close(self):
        if self.handle is not None:
            vr_volume_destroy(self.handle)
            self.handle = None
            self.storage = None
            self._keep = []

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def _stream(self, stream):
        if stream is None:
            stream = self._torch.cuda.current_stream(self.device)
        return stream.cuda_stream

    def as_tensor(self):
        """Resident VR_LAYOUT_LINEAR volumes: a float32 [nz, ny, nx] view of d_storage."""
        if self.storage is None:
            raise ValueError("VR_LAYOUT_TEX volumes live in a CUDA array, not in a tensor")
        nx, ny, nz = self.dims
        return self.storage[: nx * ny * nz * 4].view(self._torch.float32).view(nz, ny, nx)

    def vr_volume_upload_bricks(self, boxes, stream=None):
        """boxes: list of (origin(x,y,z), tensor[sz,sy,sx]) -- torch tensors (CPU, ideally
        pinned, or CUDA) or numpy arrays; all on the same side."""
        torch = self._torch
        origins, dims, ptrs, on_dev = [], [], [], None
        for origin, t in boxes:
            if isinstance(t, PinnedBrick):
                if on_dev:
                    raise ValueError("all boxes must be on the same side (host or device)")
                on_dev = False
                origins.append(origin)
                dims.append((t.shape[2], t.shape[1], t.shape[0]))
                ptrs.append(t.data_ptr())
                self._keep.append(t)
                continue
            if isinstance(t, np.ndarray):
                t = torch.from_numpy(np.ascontiguousarray(t, dtype=np.float32))
            if t.dtype != torch.float32 or not t.is_contiguous() or t.dim() != 3:
                raise ValueError("each box must be a contiguous float32 [sz, sy, sx] array")
            dev = t.is_cuda
            if on_dev is None:
                on_dev = dev
            elif on_dev != dev:
                raise ValueError("all boxes must be on the same side (host or device)")
            origins.append(origin)
            dims.append((t.shape[2], t.shape[1], t.shape[0]))
            ptrs.append(t.data_ptr())
            self._keep.append(t)
        vr_volume_upload_bricks(self.handle, origins, dims, ptrs, on_dev, self._stream(stream))
        if not self.host_brick:
            # resident copies are ordered on the stream they were given: the sources are released only once THAT
            # stream has run them
            (self._torch.cuda.current_stream(self.device) if stream is None else stream).synchronize()
            self._keep = []

    def upload(self, V, stream=None):
        """The whole cube (or the whole part) as one box."""
        self.vr_volume_upload_bricks([((0, 0, 0) if self.part is None else self.part[0], V)], stream)

    def vr_set_transfer_function(self, lut, vmin, vmax):
        vr_set_transfer_function(self.handle, lut, vmin, vmax)

    def vr_set_option(self, key, value):
        vr_set_option(self.handle, key, value)
        if key == VR_OPT_MM_BRICK:
            self.mm_shape = tuple((n - 1 + int(value) - 1) // int(value) for n in reversed(self.dims))

    def enable_aux(self, W, H):
        self._aux = self._torch.empty((H, W), dtype=self._torch.float32, device=f"cuda:{self.device}")
        vr_set_aux_output(self.handle, self._aux.data_ptr())
        return self._aux

    def disable_aux(self):
        self._aux = None
        vr_set_aux_output(self.handle, 0)

    def vr_render(self, cam, W, H, step, mode, out=None, stream=None):
        if out is None:
            out = self._torch.empty((H, W, 4), dtype=self._torch.float32, device=f"cuda:{self.device}")
        if self._aux is not None and tuple(self._aux.shape) != (H, W):
            raise ValueError("aux buffer has a different size; call enable_aux(W, H)")
        vr_render(self.handle, cam, W, H, step, mode, out.data_ptr(), self._stream(stream))
        return out

    def vr_render_wall(self, cam, W, H, K, L, step, mode, stream=None):
        """The frame as K x L tiles (row-major list of [h, w, 4] tensors, tile (a, b) at index b*K + a)."""
        w, h = W // K, H // L
        outs = [self._torch.empty((h, w, 4), dtype=self._torch.float32, device=f"cuda:{self.device}") for _ in range(K * L)]
        vr_render_wall(self.handle, cam, W, H, K, L, step, mode, [t.data_ptr() for t in outs], self._stream(stream))
        return outs

    def vr_autotune(self, cam, W, H, step, mode, out=None, stream=None):
        if out is None:
            out = self._torch.empty((H, W, 4), dtype=self._torch.float32, device=f"cuda:{self.device}")
        return vr_autotune(self.handle, cam, W, H, step, mode, out.data_ptr(), self._stream(stream))

    def vr_render_host(self, cam, W, H, step, mode, d_staging, h_out, stream=None):
        vr_render_host(self.handle, cam, W, H, step, mode, d_staging.data_ptr(), h_out.data_ptr(),
                       self._stream(stream))
        return h_out

    def vr_get_minmax(self, stream=None):
        n = int(np.prod(self.mm_shape))
        mn, mx = vr_get_minmax(self.handle, n, self._stream(stream))
        return mn.reshape(self.mm_shape), mx.reshape(self.mm_shape)

    def vr_get_stats(self):
        return vr_get_stats(self.handle)

    def vr_get_brick_flags(self):
        """Streamed volumes: VR_BRICK_* of every brick in the last frame, as an int array [nbz, nby, nbx]."""
        B = self.host_brick
        shape = tuple((n - 1 + B - 1) // B for n in reversed(self.dims))
        return vr_get_brick_flags(self.handle, int(np.prod(shape))).reshape(shape)

    # short aliases
    set_transfer_function = vr_set_transfer_function
    set_option = vr_set_option
    render = vr_render
    render_wall = vr_render_wall
    autotune = vr_autotune
    render_host = vr_render_host
    minmax = vr_get_minmax
    stats = vr_get_stats
    brick_flags = vr_get_brick_flags
