"""vmat_objective_grad_static: the objective / gradient call (A2) for callers that cannot allocate device memory.

Some users of libvmat may not call cudaMalloc when they need F and g: a planning host that handed the whole GPU to its
own pool at start-up, a real-time loop that must not wait on the driver's allocation lock, a plug-in whose host forbids
driver allocations after start-up.  For them the library has one entry point whose scratch (the per-block partial sums of F) is an
array compiled into libvmat.so, 256 KiB, good for up to 2^23 voxels.  This file checks that it returns what the
handle-based vmat_objective_grad returns, on calls that follow one another and therefore find the array dirty.

Named test_zz_* so that pytest collects it after every other file: with `-x` a failure here hides nothing.  It needs no
state from the other tests and leaves none behind (run it alone: `pytest tests/test_zz_no_alloc.py -m gpu`)."""
import ctypes

import numpy as np
import pytest
import torch

from helpers import REL_L2, assert_vec_close

DEV = "cuda:0"


def _objective(n, seed, dev):
    """Seeded dose and objective tables with both hinges of Eq. (1) active."""
    from paper_1503_01721_b200 import Objective
    rng = np.random.default_rng(seed)
    n_struct = 5
    d = (rng.random(n, dtype=np.float32) * 80.0).astype(np.float32)
    sid = rng.integers(0, n_struct, n, dtype=np.uint8)
    T = np.array([70.0, 60.0, 20.0, 45.0, 0.0], np.float32)
    wo = np.array([1.0, 0.5, 2.0, 0.0, 0.25], np.float32)
    wu = np.array([3.0, 1.0, 0.0, 0.0, 0.0], np.float32)
    t = lambda a: torch.from_numpy(a).to(dev)
    return t(d), Objective(t(sid), t(T), t(wo), t(wu))


def _handle(vm, n_voxels):
    """The existing path needs a handle, which owns its scratch: a matrix without entries over n_voxels voxels."""
    e = torch.empty(0, dtype=torch.int32)
    one = torch.tensor([0, 1], dtype=torch.int32)
    return vm.vmat_ddc_create(n_voxels, 1, e, e.clone(), torch.empty(0, dtype=torch.float32), one, one.clone(),
                              one.clone(), device=DEV)


@pytest.mark.gpu
def test_static_scratch_matches_handle_path_on_consecutive_calls():
    """Calls in a row on one stream, sizes chosen so that each later call finds the shared array holding the partial
    sums of a LARGER problem: the limit itself (2^23 voxels), then a small ragged size, then a size whose partials
    exceed one pass of the summing kernel's 1024 threads, then the small one again with another dose.  F and g must be
    the bits of vmat_objective_grad (same kernels, same order of summation), which also puts them inside the
    tolerance of the parity tests.  Device memory in use must not grow from one call to the next."""
    import paper_1503_01721_b200 as vm
    vm.load_library()
    sizes = [vm.OBJECTIVE_STATIC_MAX_VOXELS, 5003, 700001, 5003]
    free_after = []
    for k, n in enumerate(sizes):
        d, obj = _objective(n, 100 + k, DEV)
        g_ref, g_new = torch.full((n,), 7.0, device=DEV), torch.full((n,), -7.0, device=DEV)
        F_ref = torch.full((1,), -1.0, dtype=torch.float64, device=DEV)
        F_new = torch.full((1,), -2.0, dtype=torch.float64, device=DEV)
        h = _handle(vm, n)
        vm.vmat_objective_grad(h, d, obj, g_ref, F_ref)
        torch.cuda.synchronize()
        before = torch.cuda.mem_get_info()[0]
        vm.vmat_objective_grad_static(d, obj, g_new, F_new)
        torch.cuda.synchronize()
        free_after.append((before, torch.cuda.mem_get_info()[0]))
        assert vm.last_launch_count() == 2
        assert_vec_close(f"g[{k}]", g_new.cpu().numpy(), g_ref.cpu().numpy())
        assert abs(F_new.item() - F_ref.item()) <= REL_L2 * abs(F_ref.item())
        assert torch.equal(g_new, g_ref), f"call {k} (n = {n}): g differs from vmat_objective_grad"
        assert F_new.item() == F_ref.item(), f"call {k} (n = {n}): F differs from vmat_objective_grad"
        assert F_ref.item() > 0.0
        h.close()
    # the first call may load the kernels' module; from the second on the call must leave free memory where it was
    for before, after in free_after[1:]:
        assert after >= before, "vmat_objective_grad_static changed the device memory in use"


@pytest.mark.gpu
def test_static_scratch_empty_input_gives_zero():
    import paper_1503_01721_b200 as vm
    d, obj = _objective(0, 1, DEV)
    F = torch.full((1,), 3.0, dtype=torch.float64, device=DEV)
    vm.vmat_objective_grad_static(d, obj, torch.empty(0, device=DEV), F)
    torch.cuda.synchronize()
    assert F.item() == 0.0


def test_static_scratch_rejects_sizes_beyond_its_limit():
    """One voxel more than the built-in array serves: refused with a message that names the limit, before any CUDA
    call (so this runs without a GPU; the pointers are never dereferenced)."""
    from paper_1503_01721_b200 import build
    lib = ctypes.CDLL(build.build())
    lib.vmat_last_error.restype = ctypes.c_char_p
    fake = ctypes.c_void_p(256)
    limit = 1 << 23
    rc = lib.vmat_objective_grad_static(ctypes.c_int32(limit + 1), fake, fake, ctypes.c_int32(1), fake, fake, fake, fake,
                                        fake, None)
    assert rc == -1
    msg = lib.vmat_last_error().decode()
    assert "VMAT_OBJECTIVE_STATIC_MAX_VOXELS" in msg and str(limit) in msg
    assert lib.vmat_objective_grad_static(ctypes.c_int32(4), None, fake, ctypes.c_int32(1), fake, fake, fake, fake, fake,
                                          None) == -1
