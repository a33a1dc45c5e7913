"""Seeded pixel subsets for full-size parity checks and the bounded CPU baseline."""
import numpy as np


def tile_subset(W, H, n_tiles=16, tile=64, seed=0):
    """n_tiles tile x tile pixel blocks at seeded, stratified positions.
    Returns int32 [n, 2] of (i, j)."""
    rng = np.random.RandomState(seed)
    g = int(np.ceil(np.sqrt(n_tiles)))
    out = []
    k = 0
    for gy in range(g):
        for gx in range(g):
            if k >= n_tiles:
                break
            x_lo, x_hi = gx * W // g, max((gx + 1) * W // g - tile, gx * W // g)
            y_lo, y_hi = gy * H // g, max((gy + 1) * H // g - tile, gy * H // g)
            x0 = int(rng.randint(x_lo, x_hi + 1))
            y0 = int(rng.randint(y_lo, y_hi + 1))
            jj, ii = np.meshgrid(np.arange(y0, min(y0 + tile, H)), np.arange(x0, min(x0 + tile, W)),
                                 indexing="ij")
            out.append(np.stack([ii.ravel(), jj.ravel()], axis=1))
            k += 1
    return np.concatenate(out, axis=0).astype(np.int32)
