"""CPU FP64 oracle for the VMAT beamlet-price path - TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin numpy/ctypes wrapper around `vmat_oracle.c` (plain C loops over COO triplets; see the
header of that file for the passages of PAPER.md each function follows and for how it is
pinned).  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this package.  It imports nothing from
`paper_1503_01721_b200` and the CUDA library imports nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vmat_oracle.c")
_SO = os.path.join(_HERE, "libvmat_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile vmat_oracle.c with gcc (strict IEEE: no -ffast-math, no FMA contraction)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i32, i64, vp, f64 = ctypes.c_int32, ctypes.c_int64, ctypes.c_void_p, ctypes.c_double
        lib.oracle_dose.argtypes = [i64, vp, vp, vp, i32, vp, vp]
        lib.oracle_dose.restype = None
        lib.oracle_objective_grad.argtypes = [i32, vp, vp, vp, vp, vp, vp]
        lib.oracle_objective_grad.restype = f64
        lib.oracle_price.argtypes = [i64, vp, vp, vp, i32, vp, vp]
        lib.oracle_price.restype = None
        lib.oracle_select_rows.argtypes = [i32, vp, vp, vp, vp, vp, vp]
        lib.oracle_select_rows.restype = None
        lib.oracle_angle_price.argtypes = [i32, vp, vp, vp, vp]
        lib.oracle_angle_price.restype = i32
        lib.oracle_select_constrained.argtypes = [i32, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp, vp]
        lib.oracle_select_constrained.restype = i32
        _lib = lib
    return _lib


def _c(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data


def dose(coo_voxel, coo_beamlet, coo_val, n_voxels: int, x) -> np.ndarray:
    """O1: d = D x (FP64)."""
    v, pv = _c(coo_voxel, np.int32)
    b, pb = _c(coo_beamlet, np.int32)
    a, pa = _c(coo_val, np.float32)
    xx, px = _c(x, np.float32)
    d = np.empty(n_voxels, dtype=np.float64)
    _load().oracle_dose(v.size, pv, pb, pa, n_voxels, px, d.ctypes.data)
    return d


def objective_grad(d, voxel_struct, T, w_over, w_under):
    """O2: (F, g) of Eq. (1) L45 with g = +dF/dd (reading C1)."""
    dd, pd = _c(d, np.float64)
    s, ps = _c(voxel_struct, np.uint8)
    t, pt = _c(T, np.float32)
    wo, pwo = _c(w_over, np.float32)
    wu, pwu = _c(w_under, np.float32)
    g = np.empty(dd.size, dtype=np.float64)
    F = _load().oracle_objective_grad(dd.size, pd, ps, pt, pwo, pwu, g.ctypes.data)
    return float(F), g


def price(coo_voxel, coo_beamlet, coo_val, n_beamlets: int, g) -> np.ndarray:
    """O3: p = D^T g (FP64), Eq. (3) L60."""
    v, pv = _c(coo_voxel, np.int32)
    b, pb = _c(coo_beamlet, np.int32)
    a, pa = _c(coo_val, np.float32)
    gg, pg = _c(g, np.float64)
    p = np.empty(n_beamlets, dtype=np.float64)
    _load().oracle_price(v.size, pv, pb, pa, n_beamlets, pg, p.ctypes.data)
    return p


def select_rows(p_f32, leafrow_col_offset):
    """O4: per leaf row the minimum-price contiguous opening [L,R) of an FP32 price vector (L133)."""
    p, pp = _c(p_f32, np.float32)
    off, po = _c(leafrow_col_offset, np.int32)
    n_rows = off.size - 1
    L = np.zeros(n_rows, dtype=np.int32)
    R = np.zeros(n_rows, dtype=np.int32)
    rp = np.zeros(n_rows, dtype=np.float64)
    max_n = int(np.max(np.diff(off))) if n_rows > 0 else 0
    S = np.zeros(max_n + 1, dtype=np.float64)
    _load().oracle_select_rows(n_rows, po, pp, L.ctypes.data, R.ctypes.data, rp.ctypes.data, S.ctypes.data)
    return L, R, rp


def angle_price(row_price, angle_row_offset, angle_mask=None):
    """O5: aperture price per control point and the best control point (L133, L56)."""
    rp, prp = _c(row_price, np.float64)
    off, po = _c(angle_row_offset, np.int32)
    n_a = off.size - 1
    ap = np.zeros(n_a, dtype=np.float64)
    if angle_mask is not None:
        m, pm = _c(angle_mask, np.uint8)
    else:
        m, pm = None, None
    best = _load().oracle_angle_price(n_a, po, prp, pm, ap.ctypes.data)
    return ap, int(best)


def select_constrained(p_f32, angle_row_offset, leafrow_col_offset, leafrow_pos0, interdigitation: bool,
                       angle_mask=None, L_lo=None, L_hi=None, R_lo=None, R_hi=None):
    """O6: aperture selection with the interdigitation constraint of L135 and / or per-row leaf windows (L66):
    (L, R, row_price, angle_price, best_angle).  See vmat_oracle.c for the readings."""
    p, pp = _c(p_f32, np.float32)
    aro, pa = _c(angle_row_offset, np.int32)
    lco, pl = _c(leafrow_col_offset, np.int32)
    u0, pu = _c(leafrow_pos0, np.int32)
    n_a, n_rows = aro.size - 1, lco.size - 1
    keep = [p, aro, lco, u0]

    def opt(a, dt):
        if a is None:
            return None
        arr, ptr = _c(a, dt)
        keep.append(arr)
        return ptr

    pm = opt(angle_mask, np.uint8)
    w = [opt(a, np.int32) for a in (L_lo, L_hi, R_lo, R_hi)]
    L = np.zeros(n_rows, dtype=np.int32)
    R = np.zeros(n_rows, dtype=np.int32)
    rp = np.zeros(n_rows, dtype=np.float64)
    ap = np.zeros(n_a, dtype=np.float64)
    best = _load().oracle_select_constrained(n_a, pa, pl, pu, pp, pm, 1 if interdigitation else 0, w[0], w[1], w[2],
                                             w[3], L.ctypes.data, R.ctypes.data, rp.ctypes.data, ap.ctypes.data)
    return L, R, rp, ap, int(best)


@dataclass
class PriceEval:
    d: np.ndarray
    F: float
    g: np.ndarray
    p: np.ndarray
    p_f32: np.ndarray
    L: np.ndarray
    R: np.ndarray
    row_price: np.ndarray
    angle_price: np.ndarray
    best_angle: int


def price_eval(coo_voxel, coo_beamlet, coo_val, n_voxels, n_beamlets, x, voxel_struct, T, w_over,
               w_under, leafrow_col_offset, angle_row_offset, angle_mask=None) -> PriceEval:
    """One whole price evaluation O1 -> O5 (the `step` bench.py times)."""
    d = dose(coo_voxel, coo_beamlet, coo_val, n_voxels, x)
    F, g = objective_grad(d, voxel_struct, T, w_over, w_under)
    p = price(coo_voxel, coo_beamlet, coo_val, n_beamlets, g)
    p32 = p.astype(np.float32)                      # C6: the selection is a function of an FP32 p
    L, R, rp = select_rows(p32, leafrow_col_offset)
    if angle_mask is not None:                      # C7: occupied control points stay closed
        aro = np.asarray(angle_row_offset)
        for a in np.nonzero(np.asarray(angle_mask))[0]:
            L[aro[a]:aro[a + 1]] = 0
            R[aro[a]:aro[a + 1]] = 0
            rp[aro[a]:aro[a + 1]] = 0.0
    ap, best = angle_price(rp, angle_row_offset, angle_mask)
    return PriceEval(d, F, g, p, p32, L, R, rp, ap, best)


# ----------------------------------------------------------------------------------------------------------------
# All-cores variant for the TIMED baseline only (vmat_oracle_mt.c: the same C functions, each thread on its share of
# the triplets / voxels / leaf rows).  Pinned against the functions above in tests/test_oracle_mt.py.
_SRC_MT = os.path.join(_HERE, "vmat_oracle_mt.c")
_SO_MT = os.path.join(_HERE, "libvmat_oracle_mt.so")
_lib_mt = None


def build_mt(force: bool = False) -> str:
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_MT))
    if force or not os.path.exists(_SO_MT) or os.path.getmtime(_SO_MT) < newest:
        tmp = _SO_MT + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
                               "-o", tmp, _SRC, _SRC_MT, "-lm"])
        os.replace(tmp, _SO_MT)
    return _SO_MT


def _load_mt():
    global _lib_mt
    if _lib_mt is None:
        lib = ctypes.CDLL(build_mt())
        i32, i64, vp, f64, ci = ctypes.c_int32, ctypes.c_int64, ctypes.c_void_p, ctypes.c_double, ctypes.c_int
        lib.oracle_mt_dose.argtypes = [ci, i64, vp, vp, vp, i32, vp, vp, vp]
        lib.oracle_mt_dose.restype = None
        lib.oracle_mt_price.argtypes = [ci, i64, vp, vp, vp, i32, vp, vp, vp]
        lib.oracle_mt_price.restype = None
        lib.oracle_mt_objective_grad.argtypes = [ci, i32, vp, vp, vp, vp, vp, vp]
        lib.oracle_mt_objective_grad.restype = f64
        lib.oracle_mt_select_rows.argtypes = [ci, i32, vp, vp, vp, vp, vp, i32]
        lib.oracle_mt_select_rows.restype = None
        _lib_mt = lib
    return _lib_mt


def available_cores() -> int:
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def price_eval_mt(coo_voxel, coo_beamlet, coo_val, n_voxels, n_beamlets, x, voxel_struct, T, w_over, w_under,
                  leafrow_col_offset, angle_row_offset, n_threads: Optional[int] = None) -> PriceEval:
    """One whole price evaluation O1 -> O5 with the work of O1-O4 spread over `n_threads` (default: every core
    this process may run on)."""
    lib = _load_mt()
    nt = int(n_threads or available_cores())
    v, pv = _c(coo_voxel, np.int32)
    b, pb = _c(coo_beamlet, np.int32)
    a, pa = _c(coo_val, np.float32)
    xx, px = _c(x, np.float32)
    s, ps = _c(voxel_struct, np.uint8)
    t, pt = _c(T, np.float32)
    wo, pwo = _c(w_over, np.float32)
    wu, pwu = _c(w_under, np.float32)
    off, po = _c(leafrow_col_offset, np.int32)
    priv = np.empty(nt * max(n_voxels, n_beamlets, 1), dtype=np.float64)
    d = np.empty(n_voxels, dtype=np.float64)
    lib.oracle_mt_dose(nt, v.size, pv, pb, pa, n_voxels, px, d.ctypes.data, priv.ctypes.data)
    g = np.empty(n_voxels, dtype=np.float64)
    F = float(lib.oracle_mt_objective_grad(nt, n_voxels, d.ctypes.data, ps, pt, pwo, pwu, g.ctypes.data))
    p = np.empty(n_beamlets, dtype=np.float64)
    lib.oracle_mt_price(nt, v.size, pv, pb, pa, n_beamlets, g.ctypes.data, p.ctypes.data, priv.ctypes.data)
    p32 = p.astype(np.float32)
    n_rows = off.size - 1
    L = np.zeros(n_rows, dtype=np.int32)
    R = np.zeros(n_rows, dtype=np.int32)
    rp = np.zeros(n_rows, dtype=np.float64)
    max_n = int(np.max(np.diff(off))) if n_rows > 0 else 0
    lib.oracle_mt_select_rows(nt, n_rows, po, p32.ctypes.data, L.ctypes.data, R.ctypes.data, rp.ctypes.data, max_n)
    ap, best = angle_price(rp, angle_row_offset)
    return PriceEval(d, F, g, p, p32, L, R, rp, ap, best)
