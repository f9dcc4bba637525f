"""Binding of libvmat_probe.so (include/vmat_probe.h): measurement aids for bench.py, kept out of the product library.
Built beside libvmat.so by `python -m paper_1503_01721_b200.build`."""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvmat_probe.so")
_lib = None


def load_library():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_1503_01721_b200.build`")
        lib = ctypes.CDLL(LIB_PATH)
        lib.vmat_hbm_read_probe.argtypes = [ctypes.c_int64, ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.vmat_hbm_read_probe.restype = ctypes.c_int
        lib.vmat_probe_last_error.restype = ctypes.c_char_p
        _lib = lib
    return _lib


def hbm_read_probe(n_bytes: int, reps: int = 20):
    """(GB/s, kernels launched) of a read-only stream over a scratch buffer of n_bytes on the current CUDA device, with
    the 256-bit streaming loads of the dose and price kernels (vmat_hbm_read_probe)."""
    lib = load_library()
    gbs, n = ctypes.c_double(0.0), ctypes.c_int32(0)
    rc = lib.vmat_hbm_read_probe(int(n_bytes), int(reps), ctypes.byref(gbs), ctypes.byref(n),
                                 torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise RuntimeError(f"vmat_hbm_read_probe failed ({rc}): {lib.vmat_probe_last_error().decode()}")
    return float(gbs.value), int(n.value)
