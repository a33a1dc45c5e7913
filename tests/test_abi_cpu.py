"""CPU-side checks of the C-ABI library: it loads, exports every symbol
include/vr.h declares, validates arguments, and its host-only logic (brick view
order) agrees with the oracle.  No kernel is launched here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
import paper_1001_2049_b200 as vr
import vr_inputs as vi
from paper_1001_2049_b200.build import build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "vr.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vr_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = declared_symbols()
    assert len(names) >= 15
    L = C.CDLL(vr.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"libvr.so does not export {n}"
    assert sorted(vr.ABI_SYMBOLS) == names        # the binding covers the whole header
    assert "sm_100a" in vr.vr_version()


def test_storage_sizes():
    assert vr.vr_volume_storage_bytes((64, 64, 64)) == 64 ** 3 * 4
    assert vr.vr_volume_storage_bytes((512, 512, 1024)) == 1 << 30
    assert vr.vr_volume_storage_bytes((1, 64, 64)) == 0
    # a 512^3-cell brick carries one ghost layer on the high side: 513^3 voxels
    sb = vr.vr_volume_slot_bytes((4096, 4096, 4096), 512)
    assert 513 ** 3 * 4 <= sb < 513 ** 3 * 4 + 256 and sb % 256 == 0
    assert vr.vr_volume_slot_bytes((40, 33, 27), 16) >= 17 ** 3 * 4
    assert vr.vr_volume_slot_bytes((40, 33, 27), 0) == 0


def test_create_fails_loudly_without_valid_arguments_or_device():
    import torch
    d = vr._desc((64, 64, 64), 0, 0, 0, 0, 0)
    with pytest.raises(vr.VrError) as e:
        vr.vr_volume_create(d)
    assert e.value.status == 1 and "d_storage" in str(e.value)
    d = vr._desc((64, 64, 64), 0, 48, 0, 4096, 1 << 30)       # mm_brick not a power of two
    with pytest.raises(vr.VrError) as e:
        vr.vr_volume_create(d)
    assert e.value.status == 1
    d = vr._desc((64, 64, 64), 0, 0, 0, 4096, 100)            # storage too small
    with pytest.raises(vr.VrError) as e:
        vr.vr_volume_create(d)
    assert e.value.status == 5
    if not torch.cuda.is_available():
        d = vr._desc((64, 64, 64), 0, 0, 0, 4096, 1 << 30)
        with pytest.raises(vr.VrError) as e:                   # no device: error, not a fallback
            vr.vr_volume_create(d)
        assert e.value.status == 6
        with pytest.raises(RuntimeError):
            vr.Volume((64, 64, 64))


@pytest.mark.parametrize("dims,B", [((40, 33, 27), 6), ((4096, 4096, 4096), 512), ((64, 64, 64), 32)])
def test_brick_order_matches_oracle(dims, B):
    cams = vi.orbit_views(dims, 8) + [vi.ortho_axis_camera(dims, axis=a) for a in range(3)]
    inside = dict(cams[0])
    inside["eye"] = np.float32([dims[0] * 0.3, dims[1] * 0.6, dims[2] * 0.5])
    cams.append(inside)
    for cam in cams:
        o_ref, k_ref = oracle.brick_order(dims, B, cam)
        o, k = vr.vr_brick_order(dims, B, cam)
        assert np.array_equal(k, k_ref)
        assert np.array_equal(o, o_ref)
