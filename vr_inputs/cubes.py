"""Synthetic spectral cubes: i.i.d. N(0,1) noise plus faint sources.

Stand-ins for ASKAP cubes; shapes, sizes and value
distributions are BASELINE.json `configs`; details are SURVEY.md Sec. 8(d).1.
Layout: V[z = frequency][y = Dec][x = RA], x fastest ("a stack of
images").  Everything is keyed by the global voxel index, so any sub-box (a
brick with its ghost layer) can be generated on its own and equals the same
region of the whole cube generated with the same device type.

Noise: Philox4x32-10, key (seed, 0), counter (g_lo, g_hi, 0, 0) with
g = (linear voxel index) >> 2; the four outputs give two Box-Muller pairs for
voxels 4g .. 4g+3 (needs nx % 4 == 0).  Source s draws its parameters from
counters (s, 0, 1, 0) and (s, 1, 1, 0).

CPU and CUDA transcendental functions differ in the last ulps, so a cube is
generated ONCE per test / bench run and the same bytes are handed to the
oracle and to the CUDA path.
"""
import math
from dataclasses import dataclass

import numpy as np
import torch

from .philox import philox4x32_10, uniform01


@dataclass(frozen=True)
class CubeSpec:
    name: str
    dims: tuple            # (nx, ny, nz) = (RA, Dec, freq)
    seed: int
    n_sources: int
    snr: tuple             # peak SNR range (lo, hi); sigma_noise = 1
    kind: str = "horn"     # "horn": 2-D Gaussian x double-horn profile; "blob": 3-D Gaussian
    inner: float = 0.8     # centres uniform in this inner fraction of each axis
    noise: bool = True


CONFIGS = {
    0: CubeSpec("tiny-64", (64, 64, 64), 0, 3, (3.0, 3.0), kind="blob", inner=0.5),
    1: CubeSpec("mid-512x512x1024", (512, 512, 1024), 1, 200, (0.5, 5.0)),
    2: CubeSpec("large-2048", (2048, 2048, 2048), 2, 5000, (0.3, 3.0)),
    3: CubeSpec("ooc-4096", (4096, 4096, 4096), 3, 20000, (0.3, 3.0)),
    4: CubeSpec("wide-1024x1024x8192", (1024, 1024, 8192), 4, 50000, (0.2, 1.5)),
}

_CHUNK_GROUPS = 1 << 22      # Philox counters per chunk (bounds temporaries)


def noise_box(seed, dims, origin=(0, 0, 0), size=None, device="cpu"):
    """N(0,1) noise for voxels origin .. origin+size of a cube of `dims`.
    Returns float32 [sz, sy, sx]."""
    nx, ny, nz = dims
    if nx % 4:
        raise ValueError("noise generator needs nx % 4 == 0")
    if size is None:
        size = (nx - origin[0], ny - origin[1], nz - origin[2])
    x0, y0, z0 = origin
    sx, sy, sz = size
    xa0 = x0 & ~3
    xa1 = (x0 + sx + 3) & ~3
    ngx = (xa1 - xa0) // 4
    out = torch.empty((sz, sy, xa1 - xa0), dtype=torch.float32, device=device)
    rows_per_chunk = max(1, _CHUNK_GROUPS // max(1, ngx * sy))
    gx = torch.arange(xa0 // 4, xa1 // 4, dtype=torch.int64, device=device)
    yy = torch.arange(y0, y0 + sy, dtype=torch.int64, device=device)
    zero = torch.zeros((), dtype=torch.int64, device=device)
    two_pi = 2.0 * math.pi
    for za in range(0, sz, rows_per_chunk):
        zb = min(sz, za + rows_per_chunk)
        zz = torch.arange(z0 + za, z0 + zb, dtype=torch.int64, device=device)
        g = ((zz[:, None, None] * ny + yy[None, :, None]) * (nx // 4) + gx[None, None, :])
        r0, r1, r2, r3 = philox4x32_10(g & 0xFFFFFFFF, g >> 32, zero, zero, seed, 0)
        del g
        rad_a = torch.sqrt(-2.0 * torch.log(uniform01(r0)))
        ang_a = two_pi * uniform01(r1)
        rad_b = torch.sqrt(-2.0 * torch.log(uniform01(r2)))
        ang_b = two_pi * uniform01(r3)
        del r0, r1, r2, r3
        blk = out[za:zb].view(zb - za, sy, ngx, 4)
        blk[..., 0] = rad_a * torch.cos(ang_a)
        blk[..., 1] = rad_a * torch.sin(ang_a)
        blk[..., 2] = rad_b * torch.cos(ang_b)
        blk[..., 3] = rad_b * torch.sin(ang_b)
    if xa0 != x0 or xa1 != x0 + sx:
        out = out[:, :, x0 - xa0: x0 - xa0 + sx].contiguous()
    return out


def source_params(spec):
    """float64 numpy table [n_sources, 6]: cx, cy, cz, sigma_xy, width, peak."""
    n = spec.n_sources
    if n == 0:
        return np.zeros((0, 6))
    s = torch.arange(n, dtype=torch.int64)
    z = torch.zeros_like(s)
    o = torch.ones_like(s)
    a = philox4x32_10(s, z, o, z, spec.seed, 0)
    b = philox4x32_10(s, o, o, z, spec.seed, 0)
    u = [(r.to(torch.float64) + 0.5) / 4294967296.0 for r in (*a, *b)]
    u = torch.stack(u, dim=1).numpy()
    dims = np.asarray(spec.dims, dtype=np.float64)
    lo = (0.5 - spec.inner / 2.0) * (dims - 1.0)
    hi = (0.5 + spec.inner / 2.0) * (dims - 1.0)
    p = np.empty((n, 6))
    p[:, 0:3] = lo[None, :] + u[:, 0:3] * (hi - lo)[None, :]
    p[:, 3] = 2.0 + 4.0 * u[:, 3]
    p[:, 4] = 20.0 + 180.0 * u[:, 4]
    p[:, 5] = spec.snr[0] + (spec.snr[1] - spec.snr[0]) * u[:, 5]
    if spec.kind == "blob":
        p[:, 3] = 4.0
    return p


def _add_source(box, origin, spec, prm):
    cx, cy, cz, sig, wid, peak = (float(v) for v in prm)
    sz, sy, sx = box.shape
    rxy = 4.0 * sig
    rz = 4.0 * sig if spec.kind == "blob" else wid / 2.0 + 8.0
    lo = [max(origin[0], int(math.ceil(cx - rxy))), max(origin[1], int(math.ceil(cy - rxy))),
          max(origin[2], int(math.ceil(cz - rz)))]
    hi = [min(origin[0] + sx - 1, int(math.floor(cx + rxy))),
          min(origin[1] + sy - 1, int(math.floor(cy + rxy))),
          min(origin[2] + sz - 1, int(math.floor(cz + rz)))]
    if lo[0] > hi[0] or lo[1] > hi[1] or lo[2] > hi[2]:
        return
    dev = box.device
    ar = lambda a, b: torch.arange(a, b + 1, dtype=torch.float32, device=dev)
    dx, dy, dz = ar(lo[0], hi[0]) - cx, ar(lo[1], hi[1]) - cy, ar(lo[2], hi[2]) - cz
    inv2s2 = 1.0 / (2.0 * sig * sig)
    r2 = dy[:, None] ** 2 + dx[None, :] ** 2
    if spec.kind == "blob":
        r3 = dz[:, None, None] ** 2 + r2[None]
        val = peak * torch.exp(-r3 * inv2s2) * (r3 <= rxy * rxy)
    else:
        spatial = torch.exp(-r2 * inv2s2) * (r2 <= rxy * rxy)
        u = dz.abs() / (wid / 2.0)
        horn = (1.0 + 1.5 * u * u) / 2.5
        roll = torch.exp(-(((u - 1.0) * (wid / 2.0)) ** 2) / (2.0 * 2.0 * 2.0))
        prof = torch.where(u <= 1.0, horn, roll)
        val = peak * prof[:, None, None] * spatial[None]
    box[lo[2] - origin[2]: hi[2] - origin[2] + 1,
        lo[1] - origin[1]: hi[1] - origin[1] + 1,
        lo[0] - origin[0]: hi[0] - origin[0] + 1] += val


def make_box(spec, origin=(0, 0, 0), size=None, device="cpu", params=None):
    """Voxels origin .. origin+size of the cube `spec` as float32 [sz, sy, sx]."""
    if size is None:
        size = tuple(spec.dims[c] - origin[c] for c in range(3))
    if spec.noise:
        box = noise_box(spec.seed, spec.dims, origin, size, device)
    else:
        box = torch.zeros((size[2], size[1], size[0]), dtype=torch.float32, device=device)
    if params is None:
        params = source_params(spec)
    for prm in params:                      # ascending source index
        _add_source(box, origin, spec, prm)
    return box


def make_cube(spec, device="cpu"):
    """The whole cube, float32 [nz, ny, nx]."""
    if isinstance(spec, int):
        spec = CONFIGS[spec]
    return make_box(spec, (0, 0, 0), None, device)


# ---- out-of-core cubes: brick-by-brick generation (BASELINE.json configs[3]) ----------
def brick_boxes(dims, brick):
    """(origin, size) of every host brick of `brick`^3 cells, in linear brick order
    bx + nbx*(by + nby*bz).  Brick b stores the voxels [B*b, min(B*b+B, n-1)] per axis: its own
    cells plus one ghost layer on the high side (S10)."""
    nx, ny, nz = dims
    out = []
    for z0 in range(0, nz - 1, brick):
        for y0 in range(0, ny - 1, brick):
            for x0 in range(0, nx - 1, brick):
                size = (min(x0 + brick, nx - 1) - x0 + 1, min(y0 + brick, ny - 1) - y0 + 1,
                        min(z0 + brick, nz - 1) - z0 + 1)
                out.append(((x0, y0, z0), size))
    return out


def sources_in_box(spec, params, origin, size):
    """Rows of `params` whose support can touch the box (a superset; make_box clips exactly)."""
    if len(params) == 0:
        return params
    rxy = 4.0 * params[:, 3]
    rz = rxy if spec.kind == "blob" else params[:, 4] / 2.0 + 8.0
    keep = np.ones(len(params), dtype=bool)
    for c, r in ((0, rxy), (1, rxy), (2, rz)):
        keep &= (params[:, c] + r >= origin[c]) & (params[:, c] - r <= origin[c] + size[c] - 1)
    return params[keep]


def ooc_spec(host_bytes, brick=512, max_per_axis=8):
    """configs[3] scaled to the host: the 4096^3 cube (256 GiB) needs more pinned memory than
    the box has, so keep its 512^3 bricks, seed, generator and source density and take the
    largest a x a x c brick grid (a/2 <= c <= a <= 8) whose brick store fits in `host_bytes`."""
    per_brick = (brick + 1) ** 3 * 4
    best = None
    for a in range(max_per_axis, 0, -1):
        c = min(a, int(host_bytes // (a * a * per_brick)))
        if c >= 1 and 2 * c >= a and (best is None or a * a * c > best[0] * best[0] * best[1]):
            best = (a, c)
    if best is None:
        raise ValueError("not even one brick fits")
    a, c = best
    dims = (brick * a, brick * a, brick * c)
    n_src = max(1, int(round(20000 * (dims[0] * dims[1] * dims[2]) / 4096.0 ** 3)))
    return CubeSpec(f"ooc-{dims[0]}x{dims[1]}x{dims[2]}", dims, 3, n_src, (0.3, 3.0))
