"""CPU tests of the library's host side: the C-ABI library loads and exports every symbol of
include/mm.h, and its own demag-tensor set-up (long double near field + multipole far field +
symmetric host FFT; csrc/demag_host.cpp) agrees with the oracle's independent __float128 tensor."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import mm_oracle as orc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def mm():
    from paper_1102_3069_b200 import build
    build.build()
    import paper_1102_3069_b200 as mm
    return mm


def test_library_exports_every_declared_symbol(mm):
    hdr = open(os.path.join(ROOT, "include", "mm.h")).read()
    names = set(re.findall(r"\b(mm_[a-z0-9_]+)\s*\(", hdr))
    assert {"mm_create", "mm_set_material", "mm_demag_init", "mm_heff", "mm_torque", "mm_step"} <= names
    L = mm.lib()
    for n in sorted(names):
        assert hasattr(L, n), n


def test_create_without_device_fails_loudly(mm):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    with pytest.raises(mm.MMError) as e:
        mm.Sim((4, 4, 1), (1e-9, 1e-9, 1e-9))
    assert e.value.status == 3 and "no CPU fallback" in str(e.value)


def test_unsupported_size_is_reported(mm):
    L = mm.lib()
    ctx = ctypes.c_void_p()
    st = L.mm_create(ctypes.byref(ctx), (ctypes.c_int * 3)(11, 4, 1), (ctypes.c_double * 3)(1, 1, 1),
                     (ctypes.c_int * 3)(0, 0, 0), None)
    assert st == 5 and b"prime factor" in L.mm_last_error(None)


@pytest.mark.parametrize("cell", [(1.0, 1.0, 1.0), (4e-9, 4e-9, 2e-9), (1.0, 2.0, 0.5)])
def test_library_tensor_matches_oracle_near_and_far(mm, cell):
    rng = np.random.default_rng(3)
    near = rng.integers(-6, 7, size=(60, 3))
    mid = rng.integers(-60, 61, size=(60, 3))
    far = rng.integers(-1100, 1101, size=(60, 3))
    far[:, 2] = rng.integers(-63, 64, size=60)
    off = np.concatenate([[[0, 0, 0], [1, 0, 0], [0, 0, 1], [40, 25, -13], [1000, 700, 63]], near, mid, far])
    a = mm.demag_tensor_host(cell, (2048, 2048, 128), (0, 0, 0), off)
    b = orc.tensor_at(off, cell)
    # absolute agreement 1e-12 and relative 3e-7 of the tensor's own magnitude at that offset
    scale = np.abs(b).max(axis=1, keepdims=True)
    assert np.abs(a - b).max() <= 1e-12
    assert np.all(np.abs(a - b) <= 3e-7 * scale + 1e-16)


def test_library_tensor_with_periodic_images(mm):
    cell, grid, pbc = (4e-9, 4e-9, 2e-9), (16, 12, 1), (3, 2, 0)
    off = np.array([[0, 0, 0], [1, 0, 0], [5, -4, 0], [8, 6, 0], [-7, 3, 0]])
    a = mm.demag_tensor_host(cell, grid, pbc, off)
    b = orc.tensor_at(off, cell, nimg=pbc, period=grid)
    assert np.abs(a - b).max() <= 1e-12


@pytest.mark.parametrize("grid,cell,pbc", [
    ((32, 32, 1), (4e-9, 4e-9, 4e-9), (0, 0, 0)),
    ((12, 10, 6), (3e-9, 4e-9, 5e-9), (0, 0, 0)),
    ((15, 9, 5), (3e-9, 3e-9, 3e-9), (0, 0, 0)),
    ((16, 12, 1), (4e-9, 4e-9, 2e-9), (2, 2, 0)),
    ((8, 6, 4), (4e-9, 3e-9, 2e-9), (0, 1, 2)),
    ((16, 1, 1), (2e-9, 3e-9, 4e-9), (0, 0, 0)),
    ((1, 1, 1), (5e-9, 5e-9, 5e-9), (0, 0, 0)),
])
def test_library_khat_matches_oracle_kernel_transform(mm, grid, cell, pbc):
    """K-hat octant (float32, -1/(PxPyPz) folded in) == real part of the oracle's FFT'd kernel."""
    kh = mm.demag_khat_host(cell, grid, pbc).astype(np.float64)
    K = orc.demag_kernel(grid, cell, pbc)
    Kh = orc.demag_kernel_fft(K)                       # (6, Pz, Py, Cx)
    P = orc.padded_size(grid, pbc)
    ref = -Kh.real[:, :P[2] // 2 + 1, :P[1] // 2 + 1, :] / (P[0] * P[1] * P[2])
    assert kh.shape == ref.shape
    assert np.abs(kh - ref).max() <= 2e-7 * np.abs(ref).max()
