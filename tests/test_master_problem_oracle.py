"""Pins of the master-problem oracle (oracle/master_problem.py; Eq. (6)-(10), L70-L101).

None of these re-types the oracle's loop: they check its results against library solvers on the special
cases that have one, against closed forms, against the optimality (KKT) conditions of Eq. (6), and its
step sizes against the Hessian of a kink-free quadratic.  The paper prints no worked MP example.
"""
import numpy as np
import pytest
from scipy.optimize import lsq_linear, minimize_scalar

from oracle import master_problem as mp


def _problem(rng, n_v=400, m=6, sym=True):
    DA = rng.random((n_v, m)) * (rng.random((n_v, m)) < 0.6)          # dense-ish aperture dose vectors, Eq. (5)
    T = rng.uniform(20.0, 70.0, n_v)
    wo = rng.uniform(0.1, 1.0, n_v)
    wu = wo.copy() if sym else wo * (rng.random(n_v) < 0.5)           # OAR voxels: w_under = 0 (L48)
    return DA, T, wo, wu


def test_one_aperture_closed_form():
    """m = 1, w_over = w_under = w: F(y) = sum w (a y - T)^2, minimiser y* = sum(w a T) / sum(w a^2)."""
    rng = np.random.default_rng(0)
    a = rng.random(50) + 0.1
    T = np.full(50, 70.0)
    w = rng.uniform(0.5, 2.0, 50)
    r = mp.solve(a[:, None], [0.0], [0.0], [1e9], T, w, w, max_iter=50, eps_F=0.0, eps_y=0.0)
    y_star = np.sum(w * a * T) / np.sum(w * a * a)
    assert abs(r.y[0] - y_star) <= 1e-12 * y_star
    F_star = np.sum(w * (a * y_star - T) ** 2)
    assert abs(r.F - F_star) <= 1e-9 * r.F
    # a quadratic in one variable: the first step (C17) is already exact
    assert abs(r.F_hist[1] - F_star) <= 1e-12 * F_star


def test_weighted_least_squares_special_case_matches_lstsq():
    """w_over = w_under: Eq. (1) is a weighted least-squares problem; with inactive bounds the MP solution is
    numpy.linalg.lstsq's."""
    rng = np.random.default_rng(1)
    DA, T, w, _ = _problem(rng)
    sw = np.sqrt(w)
    y_ref = np.linalg.lstsq(DA * sw[:, None], T * sw, rcond=None)[0]
    m = DA.shape[1]
    r = mp.solve(DA, np.zeros(m), np.full(m, -1e9), np.full(m, 1e9), T, w, w, max_iter=2000, eps_F=0.0, eps_y=1e-13)
    assert r.reason in (1, 2, 3)          # with eps_F = 0 "objective" fires once F has stopped changing in FP64
    assert np.allclose(r.y, y_ref, rtol=1e-8, atol=1e-10)
    assert np.allclose(r.z, DA @ r.y)
    assert abs(r.F - np.sum(w * (DA @ y_ref - T) ** 2)) <= 1e-10 * r.F


@pytest.mark.parametrize("seed", [2, 3, 4])
def test_box_constrained_case_matches_lsq_linear_and_kkt(seed):
    """Bounds active (Eq. (6)): scipy.optimize.lsq_linear solves the same bounded weighted least squares."""
    rng = np.random.default_rng(seed)
    DA, T, w, _ = _problem(rng, m=8)
    sw = np.sqrt(w)
    y_free = np.linalg.lstsq(DA * sw[:, None], T * sw, rcond=None)[0]
    lo = np.minimum(y_free, 0.0) - 1.0
    hi = np.maximum(y_free, 0.0) + 1.0
    lo[:3] = y_free[:3] + 0.5                                 # these three bounds cut the free optimum off
    hi[:3] = lo[:3] + 5.0
    hi[3:5] = y_free[3:5] - 0.5
    lo[3:5] = hi[3:5] - 5.0
    ref = lsq_linear(DA * sw[:, None], T * sw, bounds=(lo, hi), tol=1e-14, method="bvls")
    r = mp.solve(DA, np.clip(np.zeros(8), lo, hi), lo, hi, T, w, w, max_iter=5000, eps_F=0.0, eps_y=1e-13)
    assert r.reason in (1, 2, 3)          # with eps_F = 0 "objective" fires once F has stopped changing in FP64
    assert abs(r.F - 2.0 * ref.cost) <= 1e-9 * r.F          # lsq_linear's cost is half the sum of squares
    assert np.allclose(r.y, ref.x, rtol=1e-6, atol=1e-8)
    assert np.all(r.y >= lo) and np.all(r.y <= hi)
    # KKT of Eq. (6) with the raw gradient: 0 inside, >= 0 at the lower bound, <= 0 at the upper bound
    _, gz = mp.objective(DA @ r.y, T, w, w)
    g = DA.T @ gz
    scale = np.abs(DA.T @ (2 * w * T)).max()
    inside = (r.y > lo) & (r.y < hi)
    assert np.all(np.abs(g[inside]) <= 1e-7 * scale)
    assert np.all(g[r.y <= lo] >= -1e-7 * scale) and np.all(g[r.y >= hi] <= 1e-7 * scale)
    assert (r.y <= lo).sum() + (r.y >= hi).sum() >= 3        # bounds really are active


def test_one_sided_penalties_reach_a_kkt_point_and_beat_a_generic_solver():
    """OAR voxels (w_under = 0): F is piecewise quadratic and convex; the result satisfies the KKT conditions
    and its objective is not above what scipy's L-BFGS-B finds from the same start."""
    from scipy.optimize import minimize
    rng = np.random.default_rng(7)
    DA, T, wo, wu = _problem(rng, n_v=600, m=7, sym=False)
    m = DA.shape[1]
    lo, hi = np.zeros(m), np.full(m, 60.0)

    def fun(y):
        F, gz = mp.objective(DA @ y, T, wo, wu)
        return F, DA.T @ gz

    ref = minimize(fun, np.zeros(m), jac=True, bounds=list(zip(lo, hi)), method="L-BFGS-B",
                   options=dict(ftol=1e-15, gtol=1e-12, maxiter=5000))
    r = mp.solve(DA, np.zeros(m), lo, hi, T, wo, wu, max_iter=5000, eps_F=0.0, eps_y=1e-12)
    assert r.F <= ref.fun * (1 + 1e-9)
    assert abs(r.F - ref.fun) <= 1e-7 * ref.fun
    F0, _ = mp.objective(np.zeros(DA.shape[0]), T, wo, wu)
    assert r.F < F0 and r.F_hist[0] == pytest.approx(F0)     # start: z = 0 (L56)
    _, g = fun(r.y)
    scale = np.abs(DA.T @ (2 * wu * T)).max()
    inside = (r.y > lo) & (r.y < hi)
    assert np.all(np.abs(g[inside]) <= 1e-6 * scale)
    assert np.all(g[r.y <= lo] >= -1e-6 * scale) and np.all(g[r.y >= hi] <= 1e-6 * scale)


def test_step_sizes_are_eq7_and_eq8_alternately():
    """Kink-free quadratic (all voxels stay under-dosed, w_over = w_under): g_A(y) = H y - b with
    H = 2 DA^T W DA, so t = H s and Eq. (7) = <s,s>/<s,Hs>, Eq. (8) = <s,Hs>/<Hs,Hs>; the first step (C17) is
    the exact line minimiser <g,g>/<g,Hg>.  Pins the formulas and the order of alternation (C18)."""
    rng = np.random.default_rng(11)
    DA, T, w, _ = _problem(rng, n_v=300, m=5)
    T = T + 1000.0                                            # nobody reaches the prescription: no kink is crossed
    H = 2.0 * DA.T @ (w[:, None] * DA)
    b = 2.0 * DA.T @ (w * T)
    m = DA.shape[1]
    r = mp.solve(DA, np.zeros(m), np.full(m, -1e12), np.full(m, 1e12), T, w, w, max_iter=6, eps_F=0.0, eps_y=0.0)
    assert len(r.delta_hist) == 6
    y = np.zeros(m)
    ys = [y]
    for d in r.delta_hist:                                    # replay the iterates from the recorded step sizes
        y = y - d * (H @ y - b)
        ys.append(y)
    assert np.allclose(ys[-1], r.y, rtol=1e-9)
    g0 = H @ ys[0] - b
    assert r.delta_hist[0] == pytest.approx(float(g0 @ g0) / float(g0 @ H @ g0), rel=1e-10)
    for it in range(1, 6):
        s = ys[it] - ys[it - 1]
        Hs = H @ s
        bb1, bb2 = float(s @ s) / float(s @ Hs), float(s @ Hs) / float(Hs @ Hs)
        assert abs(bb1 - bb2) > 1e-6 * bb1                    # the two formulas are distinguishable here
        assert r.delta_hist[it] == pytest.approx(bb1 if it % 2 == 1 else bb2, rel=1e-8)


def test_first_step_minimises_along_the_gradient():
    """C17 against a line search: with no kink crossed on the way, delta_0 minimises F(y - delta g)."""
    rng = np.random.default_rng(13)
    DA, T, w, _ = _problem(rng, n_v=200, m=4)
    T = T + 500.0
    m = DA.shape[1]
    r = mp.solve(DA, np.zeros(m), np.full(m, -1e12), np.full(m, 1e12), T, w, w, max_iter=1, eps_F=0.0, eps_y=0.0)
    _, gz = mp.objective(np.zeros(DA.shape[0]), T, w, w)
    g = DA.T @ gz
    ls = minimize_scalar(lambda d: mp.objective(DA @ (-d * g), T, w, w)[0], bracket=(0.0, r.delta_hist[0] * 2),
                         tol=1e-14)
    assert r.delta_hist[0] == pytest.approx(ls.x, rel=1e-6)


def test_subspace_rule_holds_variables_at_their_bounds():
    """Eq. (9)/(10) (C15, C16): a variable whose descent direction leaves the box stays on the bound and its
    gradient entry is zero; iterates never leave the box; F never ends above its start."""
    rng = np.random.default_rng(17)
    DA, T, wo, wu = _problem(rng, n_v=300, m=6, sym=False)
    lo, hi = np.full(6, 0.5), np.full(6, 3.0)                # far too little fluence allowed: upper bounds bind
    r = mp.solve(DA, np.full(6, 0.5), lo, hi, T, wo, wu, max_iter=500, eps_F=0.0, eps_y=1e-13)
    assert np.all(r.y >= lo) and np.all(r.y <= hi)
    assert (r.y >= hi).sum() >= 1
    assert np.all(r.g_A[r.y >= hi] == 0.0) and np.all(r.g_A[r.y <= lo] == 0.0)
    assert r.F <= r.F_hist[0]
    assert r.reason in (1, 2, 3)          # with eps_F = 0 "objective" fires once F has stopped changing in FP64


def test_stopping_rules():
    rng = np.random.default_rng(19)
    DA, T, wo, wu = _problem(rng, n_v=300, m=6, sym=False)
    lo, hi = np.zeros(6), np.full(6, 1e6)
    r = mp.solve(DA, np.zeros(6), lo, hi, T, wo, wu, max_iter=3, eps_F=0.0, eps_y=0.0)
    assert r.reason == 4 and r.n_iter == 3 and len(r.F_hist) == 4 and len(r.delta_hist) == 3
    r = mp.solve(DA, np.zeros(6), lo, hi, T, wo, wu, max_iter=10000, eps_F=1e-4, eps_y=0.0)
    assert r.reason == 2 and r.n_iter >= 5
    rel = [abs(r.F_hist[j] - r.F_hist[j - 1]) / r.F_hist[j - 1] for j in range(r.n_iter - 4, r.n_iter + 1)]
    assert max(rel) <= 1e-4
    r2 = mp.solve(DA, np.zeros(6), lo, hi, T, wo, wu, max_iter=10000, eps_F=0.0, eps_y=1e-3)
    assert r2.reason == 3
    # returned z and F belong to the returned y
    assert np.allclose(r2.z, DA @ r2.y) and r2.F == pytest.approx(mp.objective(r2.z, T, wo, wu)[0])
    # nothing to improve: every aperture at its lower bound and pushing down -> stationary at once
    r3 = mp.solve(DA, np.zeros(6), lo, hi, T * 0.0, wo, wu * 0.0, max_iter=10, eps_F=0.0, eps_y=0.0)
    assert r3.reason == 1 and r3.n_iter == 0
