"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol include/cgtp.h
declares; host-side argument validation returns the documented codes without touching a GPU."""
import ctypes
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    from paper_2605_15073_b200 import build
    return ctypes.CDLL(build.build())


def test_every_declared_symbol_is_exported():
    hdr = open(os.path.join(ROOT, "include", "cgtp.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = sorted(set(re.findall(r"\b(cgtp_[a-z_0-9]+)\s*\(", hdr)))
    assert len(names) >= 15
    L = _lib()
    for n in names:
        assert hasattr(L, n), n


def test_validation_codes_without_gpu():
    L = _lib()
    L.cgtp_last_error.restype = ctypes.c_char_p
    assert L.cgtp_version() >= 100
    assert L.cgtp_max_lmax() >= 20
    U, V = ctypes.c_int(), ctypes.c_int()
    assert L.cgtp_grid_shape(6, 6, ctypes.byref(U), ctypes.byref(V)) == 0
    assert (U.value, V.value) == (10, 19)  # U >= (3 lmax+1)/2, V >= 3 lmax+1
    assert L.cgtp_grid_shape(3, 3, ctypes.byref(U), ctypes.byref(V)) == 0 and (U.value, V.value) == (5, 10)
    assert L.cgtp_grid_shape(2, 5, ctypes.byref(U), ctypes.byref(V)) == 1
    mask = np.array([0, 1, 2, 0], np.uint8)
    i64, sz = ctypes.c_int64, ctypes.c_size_t
    rc = L.cgtp_onsite(None, None, None, None, None, 2, 2, 4, 4, mask.ctypes.data_as(ctypes.c_void_p), None, i64(1),
                       None, sz(0), None)
    assert rc == 1 and b"parity_mask" in L.cgtp_last_error()
    mask[2] = 1
    rc = L.cgtp_onsite(None, None, None, None, None, 30, 30, 4, 4, mask.ctypes.data_as(ctypes.c_void_p), None, i64(1),
                       None, sz(0), None)
    assert rc == 2
    rc = L.cgtp_onsite(None, None, None, None, None, 2, 2, 4, 4, mask.ctypes.data_as(ctypes.c_void_p), None, i64(1),
                       None, sz(0), None)
    assert rc == 1 and b"null" in L.cgtp_last_error()
    rc = L.cgtp_onsite(None, None, None, None, None, 2, 2, 4, 4, mask.ctypes.data_as(ctypes.c_void_p), None, i64(0),
                       None, sz(0), None)
    assert rc == 0  # empty batch is a no-op
    rc = L.cgtp_onsite_parity(None, None, None, None, None, 2, 2, 4, 300, None, i64(1), None, sz(0), None)
    assert rc == 2  # 4*C internal channels above the compiled limit
    rc = L.cgtp_message_parity(None, None, None, None, None, None, 2, 5, 4, 4, None, i64(1), i64(0), None, sz(0), None)
    assert rc == 1 and b"band" in L.cgtp_last_error()
    L.cgtp_onsite_workspace_bytes.restype = sz
    L.cgtp_onsite_workspace_bytes.argtypes = [ctypes.c_int] * 4 + [i64]
    assert L.cgtp_onsite_workspace_bytes(6, 6, 64, 64, 4096) >= 4096 * 64 * (2 * 52 + 52) * 4


def test_binding_refuses_cpu_tensors():
    import pytest
    import torch
    from paper_2605_15073_b200 import binding as cg
    z = torch.zeros((1, 4, 9))
    w = torch.zeros((4, 4))
    with pytest.raises(TypeError):
        cg.cgtp_onsite(z, z, w, w, w, 2, 2, 4, 4, [0, 0, 1, 1])


def test_kernel_path_switch_bounds_without_gpu():
    """cgtp_set_kernel_path only stores a process-wide word: every documented CGTP_PATH_* bit is accepted, anything above is
    CGTP_ERR_INVALID, and the previous value stays in force after a refused call."""
    L = _lib()
    try:
        for bit in (1, 2, 4, 8, 16, 32, 64, 128, 256):
            assert L.cgtp_set_kernel_path(bit) == 0
            assert L.cgtp_get_kernel_path() == bit
        assert L.cgtp_set_kernel_path(511) == 0
        assert L.cgtp_set_kernel_path(512) != 0
        assert L.cgtp_set_kernel_path(-1) != 0
        assert L.cgtp_get_kernel_path() == 511
    finally:
        assert L.cgtp_set_kernel_path(0) == 0

