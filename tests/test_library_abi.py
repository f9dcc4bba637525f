"""CPU-only: libvmat.so builds, loads and exports every symbol include/vmat.h declares; the Python
binding refuses to compute without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1503_01721_b200 import build
    return build.build()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "vmat.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vmat_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_calls_of_the_north_star():
    syms = _declared_symbols()
    for name in ["vmat_ddc_create", "vmat_ddc_destroy", "vmat_dose", "vmat_objective_grad", "vmat_price",
                 "vmat_select_apertures", "vmat_price_eval", "vmat_last_error"]:
        assert name in syms


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in _declared_symbols():
        assert hasattr(lib, name), name
    lib.vmat_last_error.restype = ctypes.c_char_p
    assert lib.vmat_last_error() is not None


def test_probe_library_is_separate(lib_path):
    """The measurement aid of bench.py lives in its own library: libvmat exports nothing of it."""
    from paper_1503_01721_b200 import build
    assert os.path.exists(build.PROBE_LIB)
    probe, lib = ctypes.CDLL(build.PROBE_LIB), ctypes.CDLL(lib_path)
    assert hasattr(probe, "vmat_hbm_read_probe") and hasattr(probe, "vmat_probe_last_error")
    assert not hasattr(lib, "vmat_hbm_read_probe")
    assert probe.vmat_hbm_read_probe(ctypes.c_int64(10), 1, None, None, None) == -1     # rejected before any CUDA call


def test_binding_lists_the_same_symbols(lib_path):
    import paper_1503_01721_b200 as vm
    assert sorted(vm.EXPORTS) == _declared_symbols()
    vm.load_library()


def test_argument_errors_need_no_gpu(lib_path):
    """NULL / negative arguments are rejected before any CUDA call."""
    lib = ctypes.CDLL(lib_path)
    lib.vmat_last_error.restype = ctypes.c_char_p
    assert lib.vmat_ddc_create(None, 1, 1, 0, None, None, None, 0, None, None, None, None) == -1
    assert b"out is NULL" in lib.vmat_last_error()
    assert lib.vmat_ddc_destroy(None) == 0
    assert lib.vmat_dose(None, None, None, None) == -1


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback(lib_path, cfg0):
    import paper_1503_01721_b200 as vm
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        vm.vmat_ddc_create(cfg0.n_voxels, cfg0.n_beamlets, cfg0.coo_voxel, cfg0.coo_beamlet, cfg0.coo_val,
                           cfg0.angle_col_offset, cfg0.angle_row_offset, cfg0.leafrow_col_offset)


def test_product_does_not_import_the_oracle():
    """The CUDA path and the oracle share no code: neither imports, includes or loads the other."""
    pkg = os.path.join(ROOT, "paper_1503_01721_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import oracle|from oracle|oracle/|libvmat_oracle", src), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"(import|from) paper_1503_01721_b200|libvmat\.so|#include.*csrc", src), f
