"""Philox4x32-10 counter-based generator (Salmon, Moraes, Dror & Shaw, SC'11),
restated from the published algorithm with torch int64 tensor ops so the same
integer stream is produced on CPU and on CUDA.

State words are kept as non-negative int64 values < 2**32.
"""
import torch

_M0 = 0xD2511F53
_M1 = 0xCD9E8D57
_W0 = 0x9E3779B9
_W1 = 0xBB67AE85
_MASK = 0xFFFFFFFF


def _mulhilo(m, x):
    # x < 2**32 and m < 2**32: the int64 product wraps modulo 2**64, which keeps
    # all 64 low bits; the masks undo the sign extension of the arithmetic shift.
    p = x * m
    return (p >> 32) & _MASK, p & _MASK


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """c0..c3: int64 tensors (values < 2**32); k0, k1: python ints.  Returns 4 tensors."""
    k0 &= _MASK
    k1 &= _MASK
    for _ in range(10):
        hi0, lo0 = _mulhilo(_M0, c0)
        hi1, lo1 = _mulhilo(_M1, c2)
        c0, c1, c2, c3 = (hi1 ^ c1 ^ k0), lo1, (hi0 ^ c3 ^ k1), lo0
        k0 = (k0 + _W0) & _MASK
        k1 = (k1 + _W1) & _MASK
    return c0, c1, c2, c3


def uniform01(r):
    """u32 (int64 tensor) -> float32 in (0, 1]."""
    return (r.to(torch.float32) + 0.5) * (1.0 / 4294967296.0)
