"""TEST INFRASTRUCTURE: lets bench.py's Python run end to end on a box without a GPU, against the host emulation of
tests/hostemu, so that its control flow, key names and arithmetic are exercised before the driver runs it on a B200
(tests/test_bench_dryrun.py).  `install()` patches, inside the calling process only, the handful of torch.cuda entry
points bench.py and the package's Volume wrapper touch: "cuda" devices become the CPU, streams and events become
host-clock stand-ins that synchronise the emulated runtime, pinned allocations become ordinary ones, and the package's
library handle is the emulated one.  Nothing here is imported by the product or by bench.py."""
import time
import types

import torch


class _Stream:
    cuda_stream = 0

    def __init__(self, be):
        self.be = be

    def synchronize(self):
        self.be.sync()


class _Event:
    be = None

    def __init__(self, enable_timing=False):
        self.t = None

    def record(self, stream=None):
        _Event.be.sync()
        self.t = time.perf_counter()

    def elapsed_time(self, other):
        return (other.t - self.t) * 1e3

    def synchronize(self):
        pass


def _cpu_device(d):
    if isinstance(d, str) and d.startswith("cuda"):
        return "cpu"
    if isinstance(d, _Dev):
        return "cpu"
    return d


class _Dev:
    """stands in for torch.device("cuda:N")"""
    type = "cuda"

    def __init__(self, spec):
        self.spec = spec
        self.index = int(str(spec).split(":")[1]) if ":" in str(spec) else 0

    def __str__(self):
        return str(self.spec)


def install():
    from tests.backends import EmuBackend
    be = EmuBackend()
    be.set_sched("lazy")
    _Event.be = be
    stream = _Stream(be)
    real_device = torch.device

    def device(spec):
        return _Dev(spec) if str(spec).startswith("cuda") else real_device(spec)

    def wrap_factory(fn):
        def inner(*a, **kw):
            kw.pop("pin_memory", None)
            if "device" in kw:
                kw["device"] = _cpu_device(kw["device"])
            return fn(*a, **kw)
        return inner

    real_empty = torch.empty

    def aligned_empty(*a, **kw):
        """"device" allocations are 256-byte aligned, like cudaMalloc's"""
        was_cuda = str(kw.get("device", "")).startswith("cuda")
        kw.pop("pin_memory", None)
        if "device" in kw:
            kw["device"] = _cpu_device(kw["device"])
        t = real_empty(*a, **kw)
        if not was_cuda or t.data_ptr() % 256 == 0 or t.numel() == 0:
            return t
        nbytes = t.numel() * t.element_size()
        raw = real_empty(nbytes + 256, dtype=torch.uint8)
        off = (-raw.data_ptr()) % 256
        return raw[off:off + nbytes].view(t.dtype).view(t.shape)

    torch.device = device
    torch.empty = aligned_empty
    for name in ("zeros", "ones", "full", "arange", "tensor", "rand", "randn", "linspace", "as_tensor", "empty_like", "zeros_like"):
        setattr(torch, name, wrap_factory(getattr(torch, name)))
    real_to = torch.Tensor.to
    torch.Tensor.to = lambda self, *a, **kw: real_to(self, *[_cpu_device(x) for x in a], **{k: _cpu_device(v) for k, v in kw.items()})
    torch.Tensor.cuda = lambda self, *a, **kw: self
    real_cpu = torch.Tensor.cpu
    torch.Tensor.cpu = lambda self, *a, **kw: (be.sync(), real_cpu(self, *a, **kw))[1]    # a device-to-host copy synchronises
    torch.Tensor.pin_memory = lambda self, *a, **kw: self
    cuda = torch.cuda
    cuda.is_available = lambda: True
    cuda.set_device = lambda d: None
    cuda.current_stream = lambda d=None: stream
    cuda.synchronize = lambda d=None: be.sync()
    cuda.Event = _Event
    cuda.empty_cache = lambda: None
    cuda.mem_get_info = lambda d=None: (150 << 30, 180 << 30)
    cuda.get_device_properties = lambda d=None: types.SimpleNamespace(multi_processor_count=148, total_memory=180 << 30)
    return be
