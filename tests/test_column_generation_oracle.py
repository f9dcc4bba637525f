"""Pins of the column-generation oracle (oracle/column_generation.py; Figure 1(a)) on config 0.

The loop only strings together functions pinned elsewhere; these tests pin the stringing: the first iteration
against the closed form of the paper's start z = 0 (L56), every later one against invariants of the method and
against scipy.sparse products of the same triplets.
"""
import numpy as np
import pytest
import scipy.sparse as sp

from conftest import as_np
from oracle import column_generation as cg
from oracle import master_problem as mp


@pytest.fixture(scope="module")
def run0(cfg0):
    A = as_np(cfg0)
    res = cg.run(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], A["sid"], A["T"], A["wo"], A["wu"], A["lco"],
                 A["aro"], max_apertures=len(A["aro"]) - 1, y_lo=0.0, y_hi=50.0)
    D = sp.csr_matrix((A["val"].astype(np.float64), (A["vox"], A["beam"])), shape=(A["n_v"], A["n_b"]))
    return A, res, D


def test_first_iteration_is_the_papers_start(run0):
    """z = 0 (L56): g_i = -2 w_under T on under-dosed voxels, so p_j = -2 sum_i w_under_i T_i D_ij <= 0; every
    leaf row opens over all its beamlets that reach a target, and the first control point is the one with the
    most negative total."""
    A, res, D = run0
    Tv, wu = A["T"][A["sid"]].astype(np.float64), A["wu"][A["sid"]].astype(np.float64)
    p = -2.0 * (D.T @ (wu * Tv))
    assert (p <= 0).all() and (p < 0).any()
    n_a = len(A["aro"]) - 1
    totals = np.array([p[A["aco"][a]:A["aco"][a + 1]].sum() for a in range(n_a)])
    assert res.angles[0] == int(np.argmin(totals))
    assert res.aperture_price[0] == pytest.approx(totals.min(), rel=1e-6)      # prices are rounded to FP32 (C6)
    a = res.angles[0]
    for r in range(A["aro"][a], A["aro"][a + 1]):
        pr = p[A["lco"][r]:A["lco"][r + 1]]
        neg = np.nonzero(pr < 0)[0]
        if neg.size:                                                          # all-non-positive row: from first to last negative
            assert (res.L[r], res.R[r]) == (neg[0], neg[-1] + 1) or pr[res.L[r]] == 0.0
        else:
            assert (res.L[r], res.R[r]) == (0, 0)
    assert res.F_hist[0] == pytest.approx(float(np.sum(wu * Tv * Tv)))


def test_invariants_of_the_loop(run0):
    A, res, D = run0
    n_a = len(A["aro"]) - 1
    assert len(res.angles) >= 3 and len(set(res.angles)) == len(res.angles)
    assert all(pr < 0 for pr in res.aperture_price)                           # only improving apertures are added
    assert all(b < a for a, b in zip(res.F_hist, res.F_hist[1:]))             # F decreases with every aperture
    assert len(res.F_hist) == len(res.angles) + 1 == len(res.mp_iters) + 1
    assert np.all(res.y >= 0.0) and np.all(res.y <= 50.0)
    # rows of control points never chosen stay closed
    chosen = np.zeros(n_a, bool)
    chosen[res.angles] = True
    for a in range(n_a):
        rows = slice(A["aro"][a], A["aro"][a + 1])
        if not chosen[a]:
            assert not res.L[rows].any() and not res.R[rows].any()
        else:
            assert (res.R[rows] > res.L[rows]).any()


def test_final_dose_is_the_weighted_sum_of_the_aperture_dose_vectors(run0):
    """z = sum_k y_k DA(A_k), DA(A_k) = D 1_{A_k} (Eq. (5), (6)) recomputed with scipy.sparse from the returned
    openings: equivalently z = D x with the fluence map x = sum_k y_k 1_{A_k}."""
    A, res, D = run0
    x = np.zeros(A["n_b"])
    for k, a in enumerate(res.angles):
        for r in range(A["aro"][a], A["aro"][a + 1]):
            x[A["lco"][r] + res.L[r]: A["lco"][r] + res.R[r]] = res.y[k]
    assert np.allclose(D @ x, res.z, rtol=1e-12, atol=1e-12)
    Tv, wo, wu = (A[k][A["sid"]].astype(np.float64) for k in ("T", "wo", "wu"))
    assert mp.objective(res.z, Tv, wo, wu)[0] == pytest.approx(res.F_hist[-1], rel=1e-12)


def test_stop_condition(run0):
    """Either every control point is occupied, or no beamlet of an unoccupied control point has a negative price
    at the final dose (then no opening can have one, L56)."""
    A, res, D = run0
    n_a = len(A["aro"]) - 1
    Tv, wo, wu = (A[k][A["sid"]].astype(np.float64) for k in ("T", "wo", "wu"))
    if res.stop == "max_apertures":
        assert len(res.angles) == n_a
    else:
        assert res.stop == "no improving aperture"
        p = D.T @ mp.objective(res.z, Tv, wo, wu)[1]
        for a in range(n_a):
            if a not in res.angles:
                rows = range(A["aro"][a], A["aro"][a + 1])
                best = min(min((p[A["lco"][r] + l: A["lco"][r] + rr].sum() for l in range(9) for rr in range(l, 9)
                                if rr <= A["lco"][r + 1] - A["lco"][r]), default=0.0) for r in rows)
                assert best >= -1e-4 * np.abs(p).max()
    # the master problem left a KKT point: no single fluence rate can be changed to lower F
    x_cols = []
    for k, a in enumerate(res.angles):
        ind = np.zeros(A["n_b"])
        for r in range(A["aro"][a], A["aro"][a + 1]):
            ind[A["lco"][r] + res.L[r]: A["lco"][r] + res.R[r]] = 1.0
        x_cols.append(D @ ind)
    g = np.stack(x_cols, 1).T @ mp.objective(res.z, Tv, wo, wu)[1]
    scale = np.abs(np.stack(x_cols, 1).T @ (2 * wu * Tv)).max()
    inside = (res.y > 0.0) & (res.y < 50.0)
    assert np.all(np.abs(g[inside]) <= 1e-5 * scale)
    assert np.all(g[res.y <= 0.0] >= -1e-5 * scale) and np.all(g[res.y >= 50.0] <= 1e-5 * scale)


def test_max_apertures_caps_the_loop(cfg0):
    A = as_np(cfg0)
    res = cg.run(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], A["sid"], A["T"], A["wo"], A["wu"], A["lco"],
                 A["aro"], max_apertures=2, y_lo=0.0, y_hi=50.0)
    assert res.stop == "max_apertures" and len(res.angles) == 2 and len(res.F_hist) == 3


# ---------------------------------------------------------------- NEXT-3: the loop under hardware constraints
def test_leaf_windows_hand_worked():
    """Reading C25 on one arc of five control points with two leaf rows each (3 beamlets per row; row 1 starts one
    beamlet to the right: pos0 = 0, 1).  Occupied: k = 1 with rows (0,2), (1,3) and k = 4 with rows (1,1), (0,1);
    leaf travel 1 per step.  Physical positions: k = 1: (0,2), (2,4); k = 4: (1,1), (1,2).
      k = 0: only k = 1 (one step away): row 0: a in [-1,1], b in [1,3]; row 1: a in [1,3], b in [3,5]
             -> row-local (pos0 = 0, 1): row 0: L [-1,1], R [1,3]; row 1: L [0,2], R [2,4]
      k = 2: k = 1 one step, k = 4 two steps: row 0: a in [-1,1] & [-1,3] = [-1,1], b in [1,3] & [-1,3] = [1,3];
             row 1: a in [1,3] & [-1,3] = [1,3], b in [3,5] & [0,4] = [3,4] -> row-local L [0,2], R [2,3]
      k = 3: k = 1 two steps, k = 4 one step: row 0: a in [-2,2] & [0,2] = [0,2], b in [0,4] & [0,2] = [0,2];
             row 1: a in [0,4] & [0,2] = [0,2], b in [2,6] & [1,3] = [2,3] -> row-local L [-1,1], R [1,2]"""
    aro = np.arange(0, 11, 2)
    lco = np.arange(0, 31, 3)
    pos0 = np.tile([0, 1], 5)
    mask = np.array([0, 1, 0, 0, 1], np.uint8)
    L = np.zeros(10, np.int32); R = np.zeros(10, np.int32)
    L[2:4], R[2:4] = [0, 1], [2, 3]
    L[8:10], R[8:10] = [1, 0], [1, 1]
    W = cg.leaf_windows(mask, L, R, lco, aro, pos0, [0, 5], 1)
    got = np.stack(W, 1)
    B = cg.BIG
    assert got[0].tolist() == [-1, 1, 1, 3] and got[1].tolist() == [0, 2, 2, 4]
    assert got[4].tolist() == [-1, 1, 1, 3] and got[5].tolist() == [0, 2, 2, 3]
    assert got[6].tolist() == [0, 2, 0, 2] and got[7].tolist() == [-1, 1, 1, 2]
    for r in (2, 3, 8, 9):                                          # occupied control points: no bound
        assert got[r].tolist() == [-B, B, -B, B]
    # two arcs: a control point sees only its own arc
    W2 = np.stack(cg.leaf_windows(mask, L, R, lco, aro, pos0, [0, 2, 5], 1), 1)
    assert W2[0].tolist() == [-1, 1, 1, 3]                          # k = 0 sees k = 1
    assert W2[4].tolist() == [-1, 3, -1, 3]                         # k = 2 (second arc) sees only k = 4, two steps away


@pytest.fixture(scope="module")
def run0_constrained(cfg0):
    A = as_np(cfg0)
    n_a = len(A["aro"]) - 1
    res = cg.run(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], A["sid"], A["T"], A["wo"], A["wu"], A["lco"],
                 A["aro"], max_apertures=n_a, y_lo=0.0, y_hi=50.0, interdigitation=True, max_leaf_travel=1,
                 leafrow_pos0=cfg0.leafrow_pos0.numpy(), arc_angle_offset=cfg0.arc_angle_offset.numpy())
    return A, res


def test_constrained_loop_invariants(run0_constrained, run0, cfg0):
    A, res = run0_constrained
    free = run0[1]
    u0 = cfg0.leafrow_pos0.numpy()
    assert len(res.angles) >= 2 and len(set(res.angles)) == len(res.angles)
    assert all(p < 0 for p in res.aperture_price)
    F = np.array(res.F_hist)
    assert (F[1:] <= F[:-1] * (1 + 1e-12)).all()                    # every master problem starts from the previous optimum
    a, b = res.L + u0, res.R + u0
    occ = sorted(res.angles)
    for k in occ:                                                   # L135 inside every chosen aperture
        for r in range(A["aro"][k], A["aro"][k + 1] - 1):
            assert a[r] <= b[r + 1] and a[r + 1] <= b[r]
    for k, kk in zip(occ[:-1], occ[1:]):                            # C25 between consecutive occupied control points
        ra, rb = slice(A["aro"][k], A["aro"][k + 1]), slice(A["aro"][kk], A["aro"][kk + 1])
        assert (np.abs(a[ra] - a[rb]) <= kk - k).all() and (np.abs(b[ra] - b[rb]) <= kk - k).all()
    assert res.angles[0] == free.angles[0]                          # z = 0: all prices <= 0, every row opens fully
    assert res.F_hist[-1] >= free.F_hist[-1] * (1 - 1e-9)           # constraints cannot help


def test_constrained_loop_reduces_to_the_free_one(run0, cfg0):
    """No interdigitation and a leaf travel nobody can exceed: the same control points, openings and objective."""
    A, free, _ = run0
    n_a = len(A["aro"]) - 1
    res = cg.run(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], A["sid"], A["T"], A["wo"], A["wu"], A["lco"],
                 A["aro"], max_apertures=n_a, y_lo=0.0, y_hi=50.0, interdigitation=False, max_leaf_travel=1000,
                 leafrow_pos0=cfg0.leafrow_pos0.numpy(), arc_angle_offset=cfg0.arc_angle_offset.numpy())
    assert res.angles == free.angles and res.F_hist == free.F_hist and res.stop == free.stop
    opened = free.R > free.L
    assert np.array_equal(res.L[opened], free.L[opened]) and np.array_equal(res.R[opened], free.R[opened])
