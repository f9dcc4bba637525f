"""paper_1503_01721_b200 - thin Python binding of libvmat (include/vmat.h).

The beamlet-price step of the column-generation VMAT optimiser of arXiv 1503.01721 on one
B200: d = D x -> (F, g) -> p = D^T g -> per-leaf-row minimum-price opening -> best control
point.  Every step runs in the CUDA kernels of `csrc/`; this module only marshals arguments
(torch tensors provide device memory and the stream).  There is no CPU fallback: if
`libvmat.so` is missing or cannot be loaded, the first call raises.

Function names mirror the C ABI: vmat_ddc_create, vmat_dose, vmat_objective_grad,
vmat_price, vmat_select_apertures, vmat_price_eval, vmat_price_eval_host, vmat_aperture_dose.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvmat.so")
_lib = None

VMAT_OK = 0
STATUS_NAMES = {0: "VMAT_OK", -1: "VMAT_ERR_INVALID_ARG", -2: "VMAT_ERR_INDEX_RANGE", -3: "VMAT_ERR_DUPLICATE",
                -4: "VMAT_ERR_OOM", -5: "VMAT_ERR_CUDA", -6: "VMAT_ERR_NONFINITE"}

EXPORTS = [
    "vmat_ddc_create", "vmat_ddc_create_ex", "vmat_ddc_destroy", "vmat_ddc_info_get", "vmat_ddc_export_csr", "vmat_dose",
    "vmat_objective_grad", "vmat_price", "vmat_select_apertures", "vmat_price_eval", "vmat_price_eval_host",
    "vmat_aperture_dose", "vmat_ddc_set_profile_events", "vmat_last_error", "vmat_last_launch_count",
    "vmat_mp_create", "vmat_mp_destroy", "vmat_mp_reset", "vmat_mp_add_aperture", "vmat_mp_set_fluence", "vmat_mp_size",
    "vmat_mp_solve", "vmat_mp_history", "vmat_column_generation",
    "vmat_ddc_set_leaf_geometry", "vmat_select_apertures_constrained", "vmat_leaf_windows",
    "vmat_column_generation_ex", "vmat_price_select", "vmat_mp_reached_voxels", "vmat_mp_pass_geometry", "vmat_check_structure_ids", "vmat_best_pair", "vmat_merge_best",
    "vmat_price_eval_host_submit", "vmat_price_eval_host_wait", "vmat_ddc_set_schedule",
    "vmat_objective_grad_static",
]


class VmatError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


class _Info(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int64) for n in (
        "n_voxels", "n_beamlets", "nnz", "n_angles", "n_leaf_rows", "bytes_csr_d", "bytes_csr_dt",
        "bytes_device_total", "n_dose_blocks", "max_leaf_row_len", "max_voxel_row_nnz", "max_beamlet_row_nnz",
        "index_bits_d", "index_bits_dt", "padded_d", "padded_dt", "bytes_stream_d", "bytes_stream_dt",
        "tiles_d", "tiles_uniform_d", "tiles_dt", "tiles_uniform_dt", "grid_dose", "grid_price",
        "sm_affine_dose", "sm_affine_price")]


def load_library(path: Optional[str] = None):
    """Load libvmat.so (built in-tree by `python -m paper_1503_01721_b200.build`).  Raises if absent.
    path: another build of the library (e.g. one made with tuning -D flags); only honoured by the first call of the
    process, a later call with a different path raises."""
    global _lib, LIB_PATH
    if _lib is not None:
        if path is not None and os.path.abspath(path) != os.path.abspath(LIB_PATH):
            raise RuntimeError(f"libvmat is already loaded from {LIB_PATH}")
        return _lib
    if path is not None:
        LIB_PATH = path
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_1503_01721_b200.build` "
                           "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
    lib.vmat_ddc_create.argtypes = [ctypes.POINTER(vp), i32, i32, i64, vp, vp, vp, i32, vp, vp, vp, vp]
    lib.vmat_ddc_destroy.argtypes = [vp]
    lib.vmat_ddc_info_get.argtypes = [vp, ctypes.POINTER(_Info)]
    lib.vmat_ddc_export_csr.argtypes = [vp, ctypes.c_int, vp, vp, vp]
    lib.vmat_ddc_create_ex.argtypes = [ctypes.POINTER(vp), i32, i32, i64, vp, vp, vp, i32, vp, vp, vp, i32, vp]
    lib.vmat_dose.argtypes = [vp, vp, vp, vp]
    lib.vmat_objective_grad.argtypes = [vp, vp, vp, i32, vp, vp, vp, vp, vp, vp]
    lib.vmat_objective_grad_static.argtypes = [i32, vp, vp, i32, vp, vp, vp, vp, vp, vp]
    lib.vmat_price.argtypes = [vp, vp, vp, vp]
    lib.vmat_check_structure_ids.argtypes = [vp, i32, i32, vp]
    lib.vmat_select_apertures.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vmat_price_eval.argtypes = [vp, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vmat_price_eval_host.argtypes = [vp, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vmat_aperture_dose.argtypes = [vp, i32, vp, vp, vp, vp, vp]
    lib.vmat_price_eval_host_submit.argtypes = [vp, i32, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vmat_price_eval_host_wait.argtypes = [vp, i32]
    lib.vmat_ddc_set_profile_events.argtypes = [vp, vp]
    lib.vmat_ddc_set_schedule.argtypes = [vp, i32]
    f64 = ctypes.c_double
    lib.vmat_mp_create.argtypes = [ctypes.POINTER(vp), i32, i32, vp]
    lib.vmat_mp_destroy.argtypes = [vp]
    lib.vmat_mp_reset.argtypes = [vp, vp]
    lib.vmat_mp_add_aperture.argtypes = [vp, vp, f64, f64, f64, vp]
    lib.vmat_mp_set_fluence.argtypes = [vp, vp, vp]
    lib.vmat_mp_size.argtypes = [vp, vp, vp]
    lib.vmat_mp_reached_voxels.argtypes = [vp, vp]
    lib.vmat_mp_pass_geometry.argtypes = [vp, i32, vp, vp]
    lib.vmat_mp_solve.argtypes = [vp, vp, i32, vp, vp, vp, i32, f64, f64, vp, vp, vp, vp, vp, vp]
    lib.vmat_mp_history.argtypes = [vp, vp, vp]
    lib.vmat_column_generation.argtypes = [vp, vp, vp, i32, vp, vp, vp, i32, f64, f64, i32, f64, f64, vp, vp, vp,
                                           vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vmat_ddc_set_leaf_geometry.argtypes = [vp, vp]
    lib.vmat_select_apertures_constrained.argtypes = [vp, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vmat_leaf_windows.argtypes = [vp, vp, vp, vp, i32, vp, i32, vp, vp, vp, vp, vp]
    lib.vmat_column_generation_ex.argtypes = [vp, vp, vp, i32, vp, vp, vp, i32, f64, f64, i32, f64, f64, i32, i32, i32, vp,
                                              vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vmat_price_select.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vmat_best_pair.argtypes = [vp, vp, vp, i32, vp, vp]
    lib.vmat_merge_best.argtypes = [vp, i32, vp, vp]
    lib.vmat_last_error.restype = ctypes.c_char_p
    lib.vmat_last_launch_count.restype = ctypes.c_int
    for name in EXPORTS:
        if name not in ("vmat_last_error",):
            getattr(lib, name).restype = ctypes.c_int
    _lib = lib
    return lib


def _check(rc: int):
    if rc != VMAT_OK:
        raise VmatError(rc, load_library().vmat_last_error().decode())


def _ptr(t: Optional[torch.Tensor], dtype=None, device_type=None, n=None):
    if t is None:
        return None
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected {dtype}, got {t.dtype}")
    if device_type is not None and t.device.type != device_type:
        raise ValueError(f"expected a {device_type} tensor, got {t.device}")
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    if n is not None and t.numel() < n:
        raise ValueError(f"tensor too small: {t.numel()} < {n}")
    return t.data_ptr()


def _stream():
    return torch.cuda.current_stream().cuda_stream


@dataclass
class Objective:
    """Per-voxel structure ids and per-structure {T, w_over, w_under} on the device (Eq. (1))."""
    voxel_struct: torch.Tensor   # uint8 [n_voxels]
    T: torch.Tensor              # float32 [n_struct]
    w_over: torch.Tensor
    w_under: torch.Tensor

    @property
    def n_struct(self) -> int:
        return int(self.T.numel())

    def validate(self):
        """vmat_check_structure_ids: every id indexes the per-structure tables (raises VmatError otherwise)."""
        with torch.cuda.device(self.voxel_struct.device):
            _check(load_library().vmat_check_structure_ids(_ptr(self.voxel_struct, torch.uint8, "cuda"),
                                                           int(self.voxel_struct.numel()), self.n_struct, _stream()))


@dataclass
class PriceEvalOut:
    d: torch.Tensor
    g: torch.Tensor
    F: torch.Tensor            # float64 [1]
    p: torch.Tensor
    L: torch.Tensor            # int32 [n_leaf_rows]
    R: torch.Tensor
    row_price: torch.Tensor    # float64 [n_leaf_rows]
    angle_price: torch.Tensor  # float64 [n_angles]
    best_angle: torch.Tensor   # int32 [1]


class DDC:
    """Owns a vmat_ddc handle (both CSR layouts on the device)."""

    def __init__(self, handle: int, device: torch.device):
        self._h = ctypes.c_void_p(handle)
        self.device = device
        self._read_info()
        self.n_voxels, self.n_beamlets = self.info["n_voxels"], self.info["n_beamlets"]
        self.n_angles, self.n_leaf_rows, self.nnz = self.info["n_angles"], self.info["n_leaf_rows"], self.info["nnz"]

    def close(self):
        if self._h is not None and self._h.value:
            load_library().vmat_ddc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def alloc_outputs(self) -> PriceEvalOut:
        dev, f32, f64, i32 = self.device, torch.float32, torch.float64, torch.int32
        return PriceEvalOut(
            d=torch.empty(self.n_voxels, dtype=f32, device=dev), g=torch.empty(self.n_voxels, dtype=f32, device=dev),
            F=torch.empty(1, dtype=f64, device=dev), p=torch.empty(self.n_beamlets, dtype=f32, device=dev),
            L=torch.empty(self.n_leaf_rows, dtype=i32, device=dev), R=torch.empty(self.n_leaf_rows, dtype=i32, device=dev),
            row_price=torch.empty(self.n_leaf_rows, dtype=f64, device=dev),
            angle_price=torch.empty(self.n_angles, dtype=f64, device=dev),
            best_angle=torch.empty(1, dtype=i32, device=dev))

    def set_profile_events(self, events=None):
        """events: four torch.cuda.Event(enable_timing=True) (already recorded once, so their handles exist)
        or None to clear; see vmat_ddc_set_profile_events."""
        if events is None:
            _check(load_library().vmat_ddc_set_profile_events(self._h, None))
            return
        arr = (ctypes.c_void_p * 4)(*[e.cuda_event for e in events])
        _check(load_library().vmat_ddc_set_profile_events(self._h, arr))

    def _read_info(self):
        info = _Info()
        _check(load_library().vmat_ddc_info_get(self._h, ctypes.byref(info)))
        self.info = {n: int(getattr(info, n)) for n, _ in _Info._fields_}

    def set_schedule(self, sm_affine):
        """vmat_ddc_set_schedule: True / 1 = SM-affine persistent kernels, False / 0 = one CTA per item,
        None / -1 = the automatic per-kernel choice (what create sets)."""
        mode = -1 if sm_affine is None else int(sm_affine)
        _check(load_library().vmat_ddc_set_schedule(self._h, mode))
        self._read_info()

    def export_ptr(self, which: int) -> torch.Tensor:
        """Row pointers (int64 [rows+1], host) of CSR(D) (0) or CSR(D^T) (1)."""
        rows = self.n_voxels if which == 0 else self.n_beamlets
        ptr = torch.empty(rows + 1, dtype=torch.int64)
        _check(load_library().vmat_ddc_export_csr(self._h, which, ptr.data_ptr(), None, None))
        return ptr

    def export_csr(self, which: int):
        """(ptr int64 [rows+1], idx int32 [nnz], val float32 [nnz]) of CSR(D) (0) or CSR(D^T) (1), on the host."""
        rows = self.n_voxels if which == 0 else self.n_beamlets
        ptr = torch.empty(rows + 1, dtype=torch.int64)
        idx = torch.empty(self.nnz, dtype=torch.int32)
        val = torch.empty(self.nnz, dtype=torch.float32)
        _check(load_library().vmat_ddc_export_csr(self._h, which, ptr.data_ptr(), idx.data_ptr(), val.data_ptr()))
        return ptr, idx, val


def vmat_ddc_create(n_voxels: int, n_beamlets: int, coo_voxel: torch.Tensor, coo_beamlet: torch.Tensor,
                    coo_val: torch.Tensor, angle_col_offset: torch.Tensor, angle_row_offset: torch.Tensor,
                    leafrow_col_offset: torch.Tensor, device=None, index_bits: int = 0) -> DDC:
    """A0: build both layouts from COO triplets (host or device tensors).
    index_bits = 0 calls vmat_ddc_create (encoding chosen per layout); 16 or 32 call vmat_ddc_create_ex."""
    lib = load_library()
    if not torch.cuda.is_available():
        raise RuntimeError("vmat_ddc_create needs a CUDA device (there is no CPU fallback)")
    dev = torch.device(device if device is not None else (coo_val.device if coo_val.is_cuda else "cuda:0"))
    nnz = int(coo_val.numel())
    if coo_voxel.numel() != nnz or coo_beamlet.numel() != nnz:
        raise ValueError("the three COO vectors must have equal length (PAPER.md L115)")
    offs = [t.to(torch.int32).cpu().contiguous() for t in (angle_col_offset, angle_row_offset, leafrow_col_offset)]
    n_angles = offs[0].numel() - 1
    if offs[1].numel() != n_angles + 1:
        raise ValueError("angle_row_offset must have n_angles+1 entries")
    if offs[2].numel() != int(offs[1][-1]) + 1:
        raise ValueError("leafrow_col_offset must have n_leaf_rows+1 entries")
    out = ctypes.c_void_p()
    with torch.cuda.device(dev):
        args = (ctypes.byref(out), n_voxels, n_beamlets, nnz,
                _ptr(coo_voxel, torch.int32), _ptr(coo_beamlet, torch.int32), _ptr(coo_val, torch.float32),
                n_angles, offs[0].data_ptr(), offs[1].data_ptr(), offs[2].data_ptr())
        if index_bits == 0:
            rc = lib.vmat_ddc_create(*args, _stream())
        else:
            rc = lib.vmat_ddc_create_ex(*args, int(index_bits), _stream())
    _check(rc)
    return DDC(out.value, dev)


def vmat_dose(h: DDC, x: torch.Tensor, d: torch.Tensor):
    """A1: d = D x."""
    _check(load_library().vmat_dose(h._h, _ptr(x, torch.float32, "cuda", h.n_beamlets),
                                    _ptr(d, torch.float32, "cuda", h.n_voxels), _stream()))


def vmat_objective_grad(h: DDC, d: torch.Tensor, obj: Objective, g: torch.Tensor, F: torch.Tensor):
    """A2: F and g = dF/dd (Eq. (1), Eq. (4))."""
    _check(load_library().vmat_objective_grad(
        h._h, _ptr(d, torch.float32, "cuda", h.n_voxels), _ptr(obj.voxel_struct, torch.uint8, "cuda", h.n_voxels),
        obj.n_struct, _ptr(obj.T, torch.float32, "cuda"), _ptr(obj.w_over, torch.float32, "cuda"),
        _ptr(obj.w_under, torch.float32, "cuda"), _ptr(g, torch.float32, "cuda", h.n_voxels),
        _ptr(F, torch.float64, "cuda", 1), _stream()))


OBJECTIVE_STATIC_MAX_VOXELS = 1 << 23      # VMAT_OBJECTIVE_STATIC_MAX_VOXELS of include/vmat.h


def vmat_objective_grad_static(d: torch.Tensor, obj: Objective, g: torch.Tensor, F: torch.Tensor):
    """A2 for callers that may not allocate device memory (a host that pooled the whole GPU at start-up, a real-time
    loop, a plug-in whose host forbids allocations after start-up): same F and g as vmat_objective_grad, bit for bit, but no
    handle and no cudaMalloc anywhere on the path - the partial sums of F go to a 256 KiB array built into libvmat.so.
    At most OBJECTIVE_STATIC_MAX_VOXELS voxels (VmatError beyond).  Runs on d's device; the first call on a device
    looks up the array's address and should not happen inside a stream capture.  All calls share the array: keep them
    on one stream or order them with events, overlapping calls corrupt F."""
    n = int(d.numel())
    with torch.cuda.device(d.device):
        _check(load_library().vmat_objective_grad_static(
            n, _ptr(d, torch.float32, "cuda"), _ptr(obj.voxel_struct, torch.uint8, "cuda", n), obj.n_struct,
            _ptr(obj.T, torch.float32, "cuda"), _ptr(obj.w_over, torch.float32, "cuda"),
            _ptr(obj.w_under, torch.float32, "cuda"), _ptr(g, torch.float32, "cuda", n),
            _ptr(F, torch.float64, "cuda", 1), _stream()))


def vmat_price(h: DDC, g: torch.Tensor, p: torch.Tensor):
    """A3: p = D^T g (Eq. (3))."""
    _check(load_library().vmat_price(h._h, _ptr(g, torch.float32, "cuda", h.n_voxels),
                                     _ptr(p, torch.float32, "cuda", h.n_beamlets), _stream()))


def vmat_select_apertures(h: DDC, p: torch.Tensor, angle_mask: Optional[torch.Tensor], L, R, row_price,
                          angle_price, best_angle):
    """A4 + A5: best opening per leaf row, aperture price per control point, best control point (L133)."""
    _check(load_library().vmat_select_apertures(
        h._h, _ptr(p, torch.float32, "cuda", h.n_beamlets), _ptr(angle_mask, torch.uint8, "cuda", h.n_angles),
        _ptr(L, torch.int32, "cuda", h.n_leaf_rows), _ptr(R, torch.int32, "cuda", h.n_leaf_rows),
        _ptr(row_price, torch.float64, "cuda", h.n_leaf_rows), _ptr(angle_price, torch.float64, "cuda", h.n_angles),
        _ptr(best_angle, torch.int32, "cuda", 1), _stream()))


def vmat_price_select(h: DDC, g: torch.Tensor, out: PriceEvalOut, angle_mask: Optional[torch.Tensor] = None):
    """A3 -> A5 fused, from a gradient g: writes out.p, out.L, out.R, out.row_price, out.angle_price, out.best_angle."""
    _check(load_library().vmat_price_select(
        h._h, _ptr(g, torch.float32, "cuda", h.n_voxels), _ptr(angle_mask, torch.uint8, "cuda", h.n_angles),
        _ptr(out.p, torch.float32, "cuda", h.n_beamlets), _ptr(out.L, torch.int32, "cuda", h.n_leaf_rows),
        _ptr(out.R, torch.int32, "cuda", h.n_leaf_rows), _ptr(out.row_price, torch.float64, "cuda", h.n_leaf_rows),
        _ptr(out.angle_price, torch.float64, "cuda", h.n_angles), _ptr(out.best_angle, torch.int32, "cuda", 1),
        _stream()))


def vmat_best_pair(h: DDC, out: PriceEvalOut, angle_lo: int, pair: torch.Tensor):
    """NEXT-4: this block's candidate {aperture price, GLOBAL control point} (or {0, -1}) into pair (float64 [2], device)."""
    _check(load_library().vmat_best_pair(h._h, _ptr(out.angle_price, torch.float64, "cuda", h.n_angles),
                                         _ptr(out.best_angle, torch.int32, "cuda", 1), int(angle_lo),
                                         _ptr(pair, torch.float64, "cuda", 2), _stream()))


def vmat_merge_best(pairs: torch.Tensor, best: torch.Tensor):
    """NEXT-4: the A5 rule over n candidate pairs (float64 [n, 2], device) into best (float64 [2], device)."""
    n = int(pairs.numel() // 2)
    with torch.cuda.device(pairs.device):
        _check(load_library().vmat_merge_best(_ptr(pairs, torch.float64, "cuda", 2 * n), n,
                                              _ptr(best, torch.float64, "cuda", 2), _stream()))


def vmat_ddc_set_leaf_geometry(h: DDC, leafrow_pos0: torch.Tensor):
    """NEXT-3: physical column of the first beamlet of every leaf row (host int32 [n_leaf_rows])."""
    pos0 = leafrow_pos0.to(torch.int32).cpu().contiguous()
    if pos0.numel() != h.n_leaf_rows:
        raise ValueError("leafrow_pos0 must have n_leaf_rows entries")
    with torch.cuda.device(h.device):
        _check(load_library().vmat_ddc_set_leaf_geometry(h._h, pos0.data_ptr() if pos0.numel() else None))


def vmat_select_apertures_constrained(h: DDC, p: torch.Tensor, angle_mask: Optional[torch.Tensor],
                                      interdigitation: bool, L, R, row_price, angle_price, best_angle,
                                      L_lo=None, L_hi=None, R_lo=None, R_hi=None):
    """NEXT-3: A4 + A5 under the interdigitation constraint (L135) and / or per-row leaf windows (L66)."""
    n = h.n_leaf_rows
    _check(load_library().vmat_select_apertures_constrained(
        h._h, _ptr(p, torch.float32, "cuda", h.n_beamlets), _ptr(angle_mask, torch.uint8, "cuda", h.n_angles),
        1 if interdigitation else 0, _ptr(L_lo, torch.int32, "cuda", n), _ptr(L_hi, torch.int32, "cuda", n),
        _ptr(R_lo, torch.int32, "cuda", n), _ptr(R_hi, torch.int32, "cuda", n),
        _ptr(L, torch.int32, "cuda", n), _ptr(R, torch.int32, "cuda", n), _ptr(row_price, torch.float64, "cuda", n),
        _ptr(angle_price, torch.float64, "cuda", h.n_angles), _ptr(best_angle, torch.int32, "cuda", 1), _stream()))


def vmat_leaf_windows(h: DDC, angle_mask: torch.Tensor, L: torch.Tensor, R: torch.Tensor, arc_angle_offset: torch.Tensor,
                      max_leaf_travel: int, L_lo, L_hi, R_lo, R_hi):
    """NEXT-3: per-row leaf windows of the unoccupied control points from their occupied neighbours (reading C25)."""
    n = h.n_leaf_rows
    arcs = arc_angle_offset.to(torch.int32).cpu().contiguous()
    _check(load_library().vmat_leaf_windows(
        h._h, _ptr(angle_mask, torch.uint8, "cuda", h.n_angles), _ptr(L, torch.int32, "cuda", n),
        _ptr(R, torch.int32, "cuda", n), arcs.numel() - 1, arcs.data_ptr(), int(max_leaf_travel),
        _ptr(L_lo, torch.int32, "cuda", n), _ptr(L_hi, torch.int32, "cuda", n), _ptr(R_lo, torch.int32, "cuda", n),
        _ptr(R_hi, torch.int32, "cuda", n), _stream()))


def vmat_price_eval(h: DDC, x: torch.Tensor, obj: Objective, out: PriceEvalOut,
                    angle_mask: Optional[torch.Tensor] = None):
    """One whole price evaluation A1 -> A5 with the fused kernels; outputs are written into `out`."""
    _check(load_library().vmat_price_eval(
        h._h, _ptr(x, torch.float32, "cuda", h.n_beamlets), _ptr(obj.voxel_struct, torch.uint8, "cuda", h.n_voxels),
        obj.n_struct, _ptr(obj.T, torch.float32, "cuda"), _ptr(obj.w_over, torch.float32, "cuda"),
        _ptr(obj.w_under, torch.float32, "cuda"), _ptr(angle_mask, torch.uint8, "cuda", h.n_angles),
        _ptr(out.d, torch.float32, "cuda", h.n_voxels), _ptr(out.g, torch.float32, "cuda", h.n_voxels),
        _ptr(out.F, torch.float64, "cuda", 1), _ptr(out.p, torch.float32, "cuda", h.n_beamlets),
        _ptr(out.L, torch.int32, "cuda", h.n_leaf_rows), _ptr(out.R, torch.int32, "cuda", h.n_leaf_rows),
        _ptr(out.row_price, torch.float64, "cuda", h.n_leaf_rows),
        _ptr(out.angle_price, torch.float64, "cuda", h.n_angles), _ptr(out.best_angle, torch.int32, "cuda", 1),
        _stream()))


def vmat_price_eval_host(h: DDC, x_host: torch.Tensor, obj: Objective, F_host, L_host, R_host, row_price_host,
                         angle_price_host, best_angle_host, angle_mask: Optional[torch.Tensor] = None):
    """End-to-end call with HOST buffers (x in, F/L/R/prices/best out); synchronises before returning."""
    _check(load_library().vmat_price_eval_host(
        h._h, _ptr(x_host, torch.float32, "cpu", h.n_beamlets), _ptr(obj.voxel_struct, torch.uint8, "cuda", h.n_voxels),
        obj.n_struct, _ptr(obj.T, torch.float32, "cuda"), _ptr(obj.w_over, torch.float32, "cuda"),
        _ptr(obj.w_under, torch.float32, "cuda"), _ptr(angle_mask, torch.uint8, "cuda", h.n_angles),
        _ptr(F_host, torch.float64, "cpu", 1), _ptr(L_host, torch.int32, "cpu", h.n_leaf_rows),
        _ptr(R_host, torch.int32, "cpu", h.n_leaf_rows), _ptr(row_price_host, torch.float64, "cpu", h.n_leaf_rows),
        _ptr(angle_price_host, torch.float64, "cpu", h.n_angles), _ptr(best_angle_host, torch.int32, "cpu", 1),
        _stream()))


def vmat_price_eval_host_submit(h: DDC, slot: int, x_host: torch.Tensor, obj: Objective, F_host, L_host, R_host,
                                row_price_host, angle_price_host, best_angle_host, angle_mask: Optional[torch.Tensor] = None):
    """Pipelined end-to-end call, slot 0 or 1: enqueues copy-in, evaluation and copy-out and returns at once; the host
    tensors (pinned) belong to the library until vmat_price_eval_host_wait(h, slot) returns."""
    _check(load_library().vmat_price_eval_host_submit(
        h._h, int(slot), _ptr(x_host, torch.float32, "cpu", h.n_beamlets),
        _ptr(obj.voxel_struct, torch.uint8, "cuda", h.n_voxels), obj.n_struct, _ptr(obj.T, torch.float32, "cuda"),
        _ptr(obj.w_over, torch.float32, "cuda"), _ptr(obj.w_under, torch.float32, "cuda"),
        _ptr(angle_mask, torch.uint8, "cuda", h.n_angles), _ptr(F_host, torch.float64, "cpu", 1),
        _ptr(L_host, torch.int32, "cpu", h.n_leaf_rows), _ptr(R_host, torch.int32, "cpu", h.n_leaf_rows),
        _ptr(row_price_host, torch.float64, "cpu", h.n_leaf_rows), _ptr(angle_price_host, torch.float64, "cpu", h.n_angles),
        _ptr(best_angle_host, torch.int32, "cpu", 1), _stream()))


def vmat_price_eval_host_wait(h: DDC, slot: int):
    _check(load_library().vmat_price_eval_host_wait(h._h, int(slot)))


def vmat_aperture_dose(h: DDC, angle: int, L: torch.Tensor, R: torch.Tensor, x_scratch: torch.Tensor,
                       DA: torch.Tensor):
    """NEXT-1: DA(A_k) = sum_{j in A_k} D_:j (Eq. (5)) for the openings [L,R) of control point `angle`."""
    _check(load_library().vmat_aperture_dose(
        h._h, int(angle), _ptr(L, torch.int32, "cuda", h.n_leaf_rows), _ptr(R, torch.int32, "cuda", h.n_leaf_rows),
        _ptr(x_scratch, torch.float32, "cuda", h.n_beamlets), _ptr(DA, torch.float32, "cuda", h.n_voxels), _stream()))


MP_STOP_REASONS = {1: "stationary", 2: "objective", 3: "step", 4: "max_iter"}


@dataclass
class MPSolution:
    y: torch.Tensor            # float64 [n_apertures], host
    F: float
    n_iter: int
    reason: int                # 1 stationary, 2 objective, 3 step, 4 max_iter


class MasterProblem:
    """Owns a vmat_mp handle: the aperture dose vectors chosen so far and the BB iteration state (NEXT-2;
    PAPER.md Eq. (6)-(10))."""

    def __init__(self, n_voxels: int, max_apertures: int, device="cuda:0"):
        if not torch.cuda.is_available():
            raise RuntimeError("vmat_mp_create needs a CUDA device (there is no CPU fallback)")
        self.device = torch.device(device)
        self.n_voxels = int(n_voxels)
        out = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            _check(load_library().vmat_mp_create(ctypes.byref(out), self.n_voxels, int(max_apertures), _stream()))
        self._h = out

    def close(self):
        if self._h is not None and self._h.value:
            load_library().vmat_mp_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def n_apertures(self) -> int:
        n = ctypes.c_int32()
        _check(load_library().vmat_mp_size(self._h, ctypes.byref(n), None))
        return int(n.value)

    @property
    def n_reached_voxels(self) -> int:
        """Voxels reached by at least one aperture as of the last solve (the rows the BB passes read)."""
        n = ctypes.c_int32()
        _check(load_library().vmat_mp_reached_voxels(self._h, ctypes.byref(n)))
        return int(n.value)

    def pass_geometry(self, m: int) -> dict:
        """CTAs and voxel rows per grid step of the pass kernel for m apertures (vmat_mp_pass_geometry)."""
        c, r = ctypes.c_int32(), ctypes.c_int32()
        _check(load_library().vmat_mp_pass_geometry(self._h, int(m), ctypes.byref(c), ctypes.byref(r)))
        return {"n_cta": int(c.value), "rows_per_grid_step": int(r.value)}

    def reset(self):
        _check(load_library().vmat_mp_reset(self._h, _stream()))

    def add_aperture(self, DA: torch.Tensor, y0: float, y_lo: float, y_hi: float):
        _check(load_library().vmat_mp_add_aperture(self._h, _ptr(DA, torch.float32, "cuda", self.n_voxels),
                                                   float(y0), float(y_lo), float(y_hi), _stream()))

    def set_fluence(self, y: torch.Tensor):
        _check(load_library().vmat_mp_set_fluence(self._h, _ptr(y, torch.float64, "cpu", self.n_apertures), _stream()))

    def solve(self, obj: Objective, max_iter: int = 200, eps_F: float = 1e-6, eps_y: float = 1e-9,
              z: Optional[torch.Tensor] = None) -> MPSolution:
        y = torch.empty(self.n_apertures, dtype=torch.float64)
        F, n_iter, reason = ctypes.c_double(), ctypes.c_int32(), ctypes.c_int32()
        _check(load_library().vmat_mp_solve(
            self._h, _ptr(obj.voxel_struct, torch.uint8, "cuda", self.n_voxels), obj.n_struct,
            _ptr(obj.T, torch.float32, "cuda"), _ptr(obj.w_over, torch.float32, "cuda"),
            _ptr(obj.w_under, torch.float32, "cuda"), int(max_iter), float(eps_F), float(eps_y),
            _ptr(z, torch.float32, "cuda", self.n_voxels), y.data_ptr(), ctypes.addressof(F),
            ctypes.addressof(n_iter), ctypes.addressof(reason), _stream()))
        self._last_n_iter = int(n_iter.value)
        return MPSolution(y, float(F.value), int(n_iter.value), int(reason.value))

    def history(self):
        """(F_hist float64 [n_iter+1], delta_hist float64 [n_iter]) of the last solve, on the host."""
        Fh = torch.empty(self._last_n_iter + 1, dtype=torch.float64)
        dh = torch.empty(self._last_n_iter, dtype=torch.float64)
        _check(load_library().vmat_mp_history(self._h, Fh.data_ptr(), dh.data_ptr() if dh.numel() else None))
        return Fh, dh


@dataclass
class CGPlan:
    angles: torch.Tensor           # int32 [n_apertures], host: control point of aperture k in the order chosen
    y: torch.Tensor                # float64 [n_apertures], host
    F_hist: torch.Tensor           # float64 [n_apertures + 1], host
    aperture_price: torch.Tensor   # float64 [n_apertures], host
    mp_iters: torch.Tensor         # int32 [n_apertures], host
    stop: str                      # "no improving aperture" | "max_apertures"
    z: torch.Tensor                # float32 [n_voxels], device
    L: torch.Tensor                # int32 [n_leaf_rows], device
    R: torch.Tensor


def vmat_column_generation(h: DDC, mp: MasterProblem, obj: Objective, max_apertures: int, y_lo: float, y_hi: float,
                           mp_max_iter: int = 300, eps_F: float = 1e-10, eps_y: float = 1e-12,
                           interdigitation: bool = False, max_leaf_travel: int = -1,
                           arc_angle_offset: Optional[torch.Tensor] = None) -> CGPlan:
    """The column-generation loop on the device; see vmat_column_generation and (with
    interdigitation / max_leaf_travel, NEXT-3) vmat_column_generation_ex in include/vmat.h."""
    dev = h.device
    z = torch.empty(h.n_voxels, dtype=torch.float32, device=dev)
    L = torch.empty(h.n_leaf_rows, dtype=torch.int32, device=dev)
    R = torch.empty(h.n_leaf_rows, dtype=torch.int32, device=dev)
    n = ctypes.c_int32()
    stop = ctypes.c_int32()
    cap = max(int(max_apertures), 1)
    angles = torch.zeros(cap, dtype=torch.int32)
    y = torch.zeros(cap, dtype=torch.float64)
    Fh = torch.zeros(cap + 1, dtype=torch.float64)
    ap = torch.zeros(cap, dtype=torch.float64)
    its = torch.zeros(cap, dtype=torch.int32)
    head = (h._h, mp._h, _ptr(obj.voxel_struct, torch.uint8, "cuda", h.n_voxels), obj.n_struct,
            _ptr(obj.T, torch.float32, "cuda"), _ptr(obj.w_over, torch.float32, "cuda"),
            _ptr(obj.w_under, torch.float32, "cuda"), int(max_apertures), float(y_lo), float(y_hi), int(mp_max_iter),
            float(eps_F), float(eps_y))
    tail = (z.data_ptr(), L.data_ptr(), R.data_ptr(), ctypes.addressof(n), angles.data_ptr(), y.data_ptr(),
            Fh.data_ptr(), ap.data_ptr(), its.data_ptr(), ctypes.addressof(stop), _stream())
    if interdigitation or max_leaf_travel >= 0:
        arcs = None if arc_angle_offset is None else arc_angle_offset.to(torch.int32).cpu().contiguous()
        _check(load_library().vmat_column_generation_ex(
            *head, 1 if interdigitation else 0, int(max_leaf_travel), 0 if arcs is None else arcs.numel() - 1,
            None if arcs is None else arcs.data_ptr(), *tail))
    else:
        _check(load_library().vmat_column_generation(*head, *tail))
    k = int(n.value)
    return CGPlan(angles[:k], y[:k], Fh[:k + 1], ap[:k], its[:k],
                  "max_apertures" if stop.value == 1 else "no improving aperture", z, L, R)


def mp_pass_geometry(m: int, device="cuda:0") -> dict:
    """vmat_mp_pass_geometry on a throw-away one-voxel handle of capacity m."""
    mp = MasterProblem(1, m, device)
    try:
        return mp.pass_geometry(m)
    finally:
        mp.close()


def last_launch_count() -> int:
    return int(load_library().vmat_last_launch_count())
