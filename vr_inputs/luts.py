"""Transfer-function tables (N x 4 float32 RGBA, straight colours).

LUT-A: BASELINE.json configs[0] ("256-entry RGBA LUT: linear grey ramp,
alpha = 0.05*ramp over [-3, 5]"); also used for configs[1]-[3].
LUT-S: configs[4] ("steep LUT (alpha 0 below 1.5 sigma)").
LUT-5sigma: mechanism demo for empty-space skipping only.
Each returns (lut, vmin, vmax).
"""
import numpy as np


def lut_a(n=256):
    ramp = (np.arange(n, dtype=np.float64) / (n - 1))
    lut = np.stack([ramp, ramp, ramp, 0.05 * ramp], axis=1).astype(np.float32)
    return lut, -3.0, 5.0


def lut_s(n=256):
    vmin, vmax = -3.0, 5.0
    ramp = (np.arange(n, dtype=np.float64) / (n - 1))
    v = vmin + ramp * (vmax - vmin)
    i0 = int(np.max(np.nonzero(v <= 1.5)[0]))          # 143 for n = 256
    a = np.zeros(n)
    idx = np.arange(n)
    up = idx > i0
    a[up] = 0.8 * ((idx[up] - i0) / float(n - 1 - i0)) ** 2
    lut = np.stack([ramp, ramp, ramp, a], axis=1).astype(np.float32)
    return lut, vmin, vmax


def lut_5sigma(n=256):
    vmin, vmax = -3.0, 13.0
    ramp = (np.arange(n, dtype=np.float64) / (n - 1))
    v = vmin + ramp * (vmax - vmin)
    a = np.where(v > 5.0, 0.3 * (v - 5.0) / (vmax - 5.0), 0.0)
    # the entry just below the threshold must be 0 too so that alpha(v) = 0 for v <= 5
    lut = np.stack([ramp, ramp, ramp, a], axis=1).astype(np.float32)
    return lut, vmin, vmax
