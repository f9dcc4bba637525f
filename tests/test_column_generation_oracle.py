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
