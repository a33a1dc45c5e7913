"""Two ways for the parity cases (tests/parity_cases.py) to reach the C ABI of include/vr.h:

  GpuBackend  libvr.so on a CUDA device through the package's own binding (the `-m gpu` tests);
  EmuBackend  tests/hostemu/libvr_hostemu.so -- the product's sources compiled against a host emulation of the CUDA
              subset they use (TEST INFRASTRUCTURE, see tests/hostemu/cuda_runtime.h) -- so that the library's host
              logic and the kernels' C++ are held against the oracle where there is no GPU.  The package never loads it.

Both hand the cases numpy arrays; the cases never see torch.
"""
import ctypes as C
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


class GpuBackend:
    name = "gpu"
    scheds = (None,)                        # the hardware schedules its streams itself

    def set_sched(self, name):
        pass

    def __init__(self):
        import torch
        import paper_1001_2049_b200 as vr
        if not torch.cuda.is_available():
            raise RuntimeError("needs a CUDA device")
        vr.lib()
        self.vr, self.torch = vr, torch

    def Volume(self, dims, **kw):
        return self.vr.Volume(dims, **kw)

    def dev(self, a):                       # numpy -> device array
        return self.torch.from_numpy(np.ascontiguousarray(a)).cuda()

    def pin(self, a):                       # numpy -> pinned host array the library may stream from
        return self.torch.from_numpy(np.ascontiguousarray(a)).pin_memory()

    def to_np(self, t):
        return t.cpu().numpy() if hasattr(t, "cpu") else np.asarray(t)

    def sync(self):
        self.torch.cuda.synchronize()


def _aligned(nbytes, align=256):
    raw = np.empty(nbytes + align, dtype=np.uint8)
    off = (-raw.ctypes.data) % align
    return raw[off:off + nbytes]


class EmuVolume:
    """The package's Volume wrapper over numpy memory instead of torch CUDA tensors (same method names)."""

    def __init__(self, be, dims, host_brick=0, mm_brick=0, device=0, n_slots=2, layout=0, part=None):
        vr = be.vr
        self.be, self.vr = be, vr
        self.dims = tuple(int(v) for v in dims)
        self.host_brick, self.layout = int(host_brick), int(layout)
        n_slots = max(2, int(n_slots))
        if self.layout == vr.VR_LAYOUT_TEX:
            self.storage = None
            self.desc = vr._desc(self.dims, host_brick, mm_brick, device, 0, 0, layout, n_slots)
        else:
            nbytes = (vr.vr_volume_slot_bytes(self.dims, host_brick) * n_slots if host_brick
                      else vr.vr_volume_storage_bytes(self.dims if part is None else part[1]))
            if nbytes == 0:
                raise vr.VrError(1, "every extent must be >= 2")
            self.storage = _aligned(nbytes)
            self.desc = vr._desc(self.dims, host_brick, mm_brick, device, self.storage.ctypes.data, nbytes, layout, n_slots)
        self.part = part
        self.handle = vr.vr_volume_create(self.desc) if part is None else vr.vr_volume_create_part(self.desc, part[0], part[1])
        self._keep, self._aux = [], None
        mmB = mm_brick or 64
        self.mm_shape = tuple((n - 1 + mmB - 1) // mmB for n in reversed(self.dims))

    def close(self):
        if self.handle is not None:
            self.vr.vr_volume_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def as_tensor(self):
        nx, ny, nz = self.dims
        return self.storage[: nx * ny * nz * 4].view(np.float32).reshape(nz, ny, nx)

    def vr_volume_upload_bricks(self, boxes, stream=None):
        origins, dims, ptrs, on_dev = [], [], [], False
        for origin, t in boxes:
            if hasattr(t, "data_ptr"):
                shape, ptr = t.shape, t.data_ptr()
            else:
                on_dev = on_dev or getattr(t, "_emu_device", False)
                t = np.ascontiguousarray(t, dtype=np.float32)
                shape, ptr = t.shape, t.ctypes.data
            origins.append(origin)
            dims.append((shape[2], shape[1], shape[0]))
            ptrs.append(ptr)
            self._keep.append(t)
        self.vr.vr_volume_upload_bricks(self.handle, origins, dims, ptrs, int(on_dev), 0)
        if not self.host_brick:
            self.be.sync()
            self._keep = []

    def upload(self, V, stream=None):
        self.vr_volume_upload_bricks([((0, 0, 0) if self.part is None else self.part[0], V)])

    def set_transfer_function(self, lut, vmin, vmax):
        self.vr.vr_set_transfer_function(self.handle, lut, vmin, vmax)

    def set_option(self, key, value):
        self.vr.vr_set_option(self.handle, key, value)
        if key == self.vr.VR_OPT_MM_BRICK:
            self.mm_shape = tuple((n - 1 + int(value) - 1) // int(value) for n in reversed(self.dims))

    def enable_aux(self, W, H):
        self._aux = np.full((H, W), np.nan, dtype=np.float32)
        self.vr.vr_set_aux_output(self.handle, self._aux.ctypes.data)
        return self._aux

    def disable_aux(self):
        self._aux = None
        self.vr.vr_set_aux_output(self.handle, 0)

    def render(self, cam, W, H, step, mode, out=None, stream=None):
        if out is None:
            out = np.full((H, W, 4), np.nan, dtype=np.float32)
        self.vr.vr_render(self.handle, cam, W, H, step, mode, out.ctypes.data, 0)
        self.be.sync()
        return out

    def autotune(self, cam, W, H, step, mode, out=None, stream=None):
        if out is None:
            out = np.full((H, W, 4), np.nan, dtype=np.float32)
        self._tune_out = out
        return self.vr.vr_autotune(self.handle, cam, W, H, step, mode, out.ctypes.data, 0)

    def render_wall(self, cam, W, H, K, L, step, mode, stream=None):
        w, h = W // K, H // L
        outs = [np.full((h, w, 4), np.nan, dtype=np.float32) for _ in range(K * L)]
        self.vr.vr_render_wall(self.handle, cam, W, H, K, L, step, mode, [t.ctypes.data for t in outs], 0)
        self.be.sync()
        return outs

    def minmax(self, stream=None):
        n = int(np.prod(self.mm_shape))
        mn, mx = self.vr.vr_get_minmax(self.handle, n, 0)
        return mn.reshape(self.mm_shape), mx.reshape(self.mm_shape)

    def stats(self):
        return self.vr.vr_get_stats(self.handle)

    def brick_flags(self):
        B = self.host_brick
        shape = tuple((n - 1 + B - 1) // B for n in reversed(self.dims))
        return self.vr.vr_get_brick_flags(self.handle, int(np.prod(shape))).reshape(shape)


class EmuPinned:
    """float32 [sz, sy, sx] in memory the emulated runtime knows as pinned (its cudaHostAlloc)."""

    def __init__(self, cdll, a):
        self.cdll = cdll
        self.shape = tuple(int(v) for v in a.shape)
        p = C.c_void_p()
        assert cdll.vr_host_alloc(C.c_size_t(4 * a.size), C.byref(p)) == 0
        self.ptr = p.value
        self.array = np.ctypeslib.as_array((C.c_float * a.size).from_address(self.ptr)).reshape(self.shape)
        self.array[...] = a

    def data_ptr(self):
        return self.ptr

    def close(self):
        if getattr(self, "ptr", None):
            self.array = None
            self.cdll.vr_host_free(C.c_void_p(self.ptr))
            self.ptr = None

    __del__ = close


class _DevArray(np.ndarray):
    """A numpy array the emulated library is told is device memory."""
    _emu_device = True


class EmuBackend:
    name = "emu"
    SCHED = {"sync": 0, "lazy": 1, "eager": 2}
    # stream scheduling policies a case with two streams should pass under (tests/hostemu/cuda_runtime.h)
    scheds = ("lazy", "eager")

    def __init__(self):
        sys.path.insert(0, os.path.join(HERE, "hostemu"))
        try:
            import build as emu_build
        finally:
            sys.path.pop(0)
        path = emu_build.build(asan=os.environ.get("VR_EMU_ASAN", "0") == "1")
        import paper_1001_2049_b200 as vr
        self.vr = vr
        self._saved = vr._lib
        self.cdll = C.CDLL(path)
        vr._bind(self.cdll)
        vr._lib = self.cdll                 # the module-level C wrappers now reach the emulated library
        self.cdll.vr_emu_pending.restype = C.c_ulonglong

    def restore(self):
        self.vr._lib = self._saved

    def set_sched(self, name):
        self.cdll.vr_emu_set_sched(self.SCHED[name or "lazy"])

    def Volume(self, dims, **kw):
        return EmuVolume(self, dims, **kw)

    def dev(self, a):
        return np.ascontiguousarray(a).view(_DevArray)

    def pin(self, a):
        return EmuPinned(self.cdll, np.ascontiguousarray(a, dtype=np.float32))

    def to_np(self, t):
        return np.asarray(t)

    def sync(self):
        self.cdll.vr_emu_sync()
