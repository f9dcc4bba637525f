"""Shared helpers for the GPU parity tests: tolerances of BASELINE.json `north_star` and the
selection parity protocol (reading C6)."""
import numpy as np
import torch

import oracle

REL_L2 = 1e-5          # relative L2 error of FP32 vectors and of F
ABS_MAX = 1e-4         # per-element |delta| <= ABS_MAX * max|ref|


def assert_vec_close(name, got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape, name
    assert np.isfinite(got).all(), name
    nref = np.linalg.norm(ref)
    err = np.linalg.norm(got - ref)
    mx = np.abs(ref).max() if ref.size else 0.0
    if nref > 0:
        assert err <= REL_L2 * nref, f"{name}: rel L2 {err / nref:.3e} > {REL_L2}"
    else:
        assert err == 0.0, name
    if ref.size:
        worst = np.abs(got - ref).max()
        assert worst <= ABS_MAX * mx + 0.0, f"{name}: max |delta| {worst:.3e} > {ABS_MAX}*{mx:.3e}"


def oracle_eval(A, x, angle_mask=None):
    return oracle.price_eval(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], x, A["sid"], A["T"], A["wo"],
                             A["wu"], A["lco"], A["aro"], angle_mask)


def check_selection_protocol(A, out, ev, angle_mask=None):
    """(ii) the oracle's O4/O5 applied to the GPU's own FP32 p must reproduce the GPU's leaf positions,
    row prices, aperture prices and best control point bit for bit;
    (iii) against the oracle's pure FP64 path: rows may differ only on a margin below rounding."""
    p_gpu = out.p.cpu().numpy()
    L, R, rp = oracle.select_rows(p_gpu, A["lco"])
    if angle_mask is not None:
        for a in np.nonzero(np.asarray(angle_mask))[0]:
            sl = slice(A["aro"][a], A["aro"][a + 1])
            L[sl] = 0; R[sl] = 0; rp[sl] = 0.0
    ap, best = oracle.angle_price(rp, A["aro"], angle_mask)
    assert np.array_equal(out.L.cpu().numpy(), L)
    assert np.array_equal(out.R.cpu().numpy(), R)
    assert np.array_equal(out.row_price.cpu().numpy(), rp)          # FP64, same operations in the same order
    assert np.array_equal(out.angle_price.cpu().numpy(), ap)
    assert int(out.best_angle.item()) == best
    # (iii)
    diff = np.nonzero((L != ev.L) | (R != ev.R))[0]
    pmax = np.abs(ev.p).max() if ev.p.size else 0.0
    for r in diff:
        j0, n = A["lco"][r], A["lco"][r + 1] - A["lco"][r]
        S = np.concatenate([[0.0], np.cumsum(ev.p[j0:j0 + n])])
        v_gpu_choice = S[R[r]] - S[L[r]]
        assert v_gpu_choice - ev.row_price[r] <= 2 * ABS_MAX * pmax * max(n, 1), r
    return len(diff)


def obj_to_device(A, dev):
    from paper_1503_01721_b200 import Objective
    return Objective(torch.from_numpy(A["sid"]).to(dev), torch.from_numpy(A["T"]).to(dev),
                     torch.from_numpy(A["wo"]).to(dev), torch.from_numpy(A["wu"]).to(dev))


def ddc_from_arrays(A, dev, coo_on_device=True, index_bits=0):
    import paper_1503_01721_b200 as vm
    conv = (lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)) if coo_on_device else \
        (lambda a: torch.from_numpy(np.ascontiguousarray(a)))
    return vm.vmat_ddc_create(A["n_v"], A["n_b"], conv(A["vox"]), conv(A["beam"]), conv(A["val"]),
                              torch.from_numpy(A["aco"]), torch.from_numpy(A["aro"]), torch.from_numpy(A["lco"]),
                              device=dev, index_bits=index_bits)
