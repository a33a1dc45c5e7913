"""Definitional float64 brute force of the emission-absorption / MIP ray caster,
vectorised NumPy with scipy.ndimage.map_coordinates(order=1) as the trilinear
step.  Used only to pin the oracle on tiny cubes (pin C6).
Written from the prose definition (pixel centres -> rays -> slab clipping ->
midpoint samples -> trilinear -> piecewise-linear LUT -> front-to-back over),
with its own variable layout; shares nothing with oracle/ or the CUDA path."""
import numpy as np
from scipy.ndimage import map_coordinates


def rays(cam, W, H, window=None, spacing=None):
    """window = (l, r, t, b): an off-axis sub-frustum -- the part of the image plane between the fractions l..r of its
    width (from the left) and t..b of its height (from the top), sampled at W x H pixel centres of its own."""
    i = np.arange(W, dtype=np.float64)
    j = np.arange(H, dtype=np.float64)
    if window is None:
        sx = ((2 * i + 1) / W - 1.0) * (W / H)
        sy = 1.0 - (2 * j + 1) / H
    else:
        l, r, t, b, aspect = window
        x_left, x_right = (2.0 * l - 1.0) * aspect, (2.0 * r - 1.0) * aspect     # the whole plane spans [-aspect, aspect]
        y_top, y_bottom = 1.0 - 2.0 * t, 1.0 - 2.0 * b                           # and [1, -1] from top to bottom
        sx = x_left + (x_right - x_left) * (i + 0.5) / W
        sy = y_top + (y_bottom - y_top) * (j + 0.5) / H
    SX, SY = np.meshgrid(sx, sy)                     # [H, W]
    e, r, u, f = (np.asarray(cam[k], dtype=np.float64) for k in ("eye", "right", "up", "forward"))
    if cam["projection"] == 0:
        th = float(cam["tan_half_fovy"])
        D = f[None, None, :] + (SX * th)[..., None] * r + (SY * th)[..., None] * u
        D = D / np.linalg.norm(D, axis=-1, keepdims=True)
        O = np.broadcast_to(e, D.shape).copy()
    else:
        hh = float(cam["ortho_half_height"])
        O = e[None, None, :] + (SX * hh)[..., None] * r + (SY * hh)[..., None] * u
        D = np.broadcast_to(f, O.shape).copy()
    if spacing is not None:
        # the cube's voxels are `spacing` world units apart: the world-space ray in voxel-index coordinates (the
        # parameter along it keeps measuring world-space distance)
        sp = np.asarray(spacing, dtype=np.float64)
        O, D = O / sp, D / sp
    return O, D


def clip(O, D, dims):
    hi = np.asarray(dims, dtype=np.float64) - 1.0
    tn = np.zeros(O.shape[:-1])
    tf = np.full(O.shape[:-1], np.inf)
    ok = np.ones(O.shape[:-1], dtype=bool)
    for c in range(3):
        par = D[..., c] == 0.0
        with np.errstate(divide="ignore", invalid="ignore"):
            a = (0.0 - O[..., c]) / D[..., c]
            b = (hi[c] - O[..., c]) / D[..., c]
        lo_, hi_ = np.minimum(a, b), np.maximum(a, b)
        tn = np.where(par, tn, np.maximum(tn, lo_))
        tf = np.where(par, tf, np.minimum(tf, hi_))
        ok &= ~(par & ((O[..., c] < 0.0) | (O[..., c] > hi[c])))
    return tn, tf, ok & (tn < tf)


def lut_eval(table, vmin, vmax, v):
    n = table.shape[0]
    x = np.clip((v - vmin) * ((n - 1) / (vmax - vmin)), 0.0, n - 1.0)
    return np.interp(x, np.arange(n, dtype=np.float64), table.astype(np.float64))


def render(V, lut, vmin, vmax, cam, W, H, step, mode, tau, window=None, spacing=None):
    V64 = np.asarray(V, dtype=np.float64)
    nz, ny, nx = V64.shape
    O, D = rays(cam, W, H, window, spacing)
    tn, tf, hit = clip(O, D, (nx, ny, nz))
    kmax = int(np.ceil(np.max(np.where(hit, tf - tn, 0.0)) / step)) + 2
    hi = np.array([nx - 1.0, ny - 1.0, nz - 1.0])
    C = np.zeros((H, W, 3))
    A = np.zeros((H, W))
    M = np.full((H, W), -np.inf)
    alive = hit.copy()
    alpha_tab = 1.0 - (1.0 - np.clip(lut[:, 3].astype(np.float64), 0, 1)) ** step
    nsamp = 0
    for k in range(kmax):
        t = tn + (k + 0.5) * step
        act = alive & (t < tf)
        if not act.any():
            break
        P = np.clip(O + t[..., None] * D, 0.0, hi)
        v = map_coordinates(V64, [P[..., 2], P[..., 1], P[..., 0]], order=1, mode="nearest")
        nsamp += int(act.sum())
        if mode == 0:
            a = lut_eval(alpha_tab, vmin, vmax, v)
            w = np.where(act, (1.0 - A) * a, 0.0)
            for ch in range(3):
                C[..., ch] += w * lut_eval(lut[:, ch], vmin, vmax, v)
            A = A + w
            alive &= ~(A >= tau)
        else:
            M = np.where(act, np.maximum(M, v), M)
    if mode == 0:
        out = np.concatenate([C, A[..., None]], axis=-1)
    else:
        has = np.isfinite(M)
        Ms = np.where(has, M, 0.0)
        out = np.stack([np.where(has, lut_eval(lut[:, ch], vmin, vmax, Ms), 0.0) for ch in range(3)]
                       + [has.astype(np.float64)], axis=-1)
    return out, M, nsamp
