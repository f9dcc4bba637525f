"""CPU FP64 oracle of the master problem (MP) - TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md L70-L101 (section 2.1, Eq. (6)-(10)) and L139 (the four BB steps): with the apertures
chosen so far and their dose vectors DA(A_k), k in C, find fluence rates y_k in [lo_k, hi_k]
(Eq. (6): lo_k = R^L/S^U_k, hi_k = R^U/S^L_k, given by the caller) that minimise F(z), z = DA y,
by the Barzilai-Borwein iteration with the subspace step rule.

This is an iteration, so the oracle follows it step by step in the paper's order (L139: 1 gradient
in the aperture domain, 2 step size by Eq. (7)/(8) alternately, 3 update within the subspace
Eq. (9)/(10), 4 dose update), in FP64 with numpy; nothing is blocked, fused or reordered.

Readings where PAPER.md is silent or at odds with itself (C15-C20):
  C15 sign: g_A here is +dF/dy ("the gradient of the objective function in the aperture fluence
      rate domain", L94) and the update is y <- y - delta g_A.  Eq. (9)/(10) are printed in the
      convention of Eq. (4) (g = -grad F); in the + convention a variable is held at its LOWER bound
      when g_A,k > 0 and at its UPPER bound when g_A,k < 0, and its gradient entry is set to 0.
  C16 y is projected onto [lo, hi] after every update (Eq. (9)/(10) "y_k = bound"); z, F and g_A are
      always evaluated at a feasible y; the zeroed entries take part in Eq. (7)/(8) as zeros.
  C17 first step (no previous iterate; paper silent): the exact minimiser along -g_A of the quadratic
      that F is on the current side of every voxel's kink,
      delta_0 = <g,g> / (2 sum_i w_i (DA g)_i^2),  w_i = w_over if z_i > T_i, w_under if z_i < T_i, else 0.
  C18 alternation: iteration 1, 3, 5, ... use Eq. (7) (<s,s>/<s,t>), iteration 2, 4, ... Eq. (8)
      (<s,t>/<t,t>), s = y(it) - y(it-1), t = g_A(it) - g_A(it-1).  If <s,t> <= 0 (or <t,t> = 0) the
      previous delta is kept.
  C19 stopping rules (L101), tested at the top of every iteration, in this order:
      "stationary": every entry of g_A is 0 after the subspace rule (KKT point);
      "objective":  it >= 5 and |F(j) - F(j-1)| <= eps_F |F(j-1)| for the five latest j = it-4 .. it;
      "step":       it >= 1 and max_k |y_k(it) - y_k(it-1)| <= eps_y;
      "max_iter":   it == max_iter.
      The iterate at which a rule fires is returned (z and F belong to it).
  C20 dose update (step 4): z = DA y is recomputed from y (Eq. (6)), not accumulated.

Pins (tests/test_master_problem_oracle.py; none re-types these loops): weighted least-squares special
case against numpy.linalg.lstsq; box-constrained case against scipy.optimize.lsq_linear and against
the KKT conditions; one-aperture closed form; Eq. (7)/(8) against the Hessian of a kink-free quadratic;
the first step against a line search.  The paper prints no worked MP example: parity unpinned by publication.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

STOP_REASONS = {0: "running", 1: "stationary", 2: "objective", 3: "step", 4: "max_iter"}


def objective(z, T, w_over, w_under):
    """Eq. (1) L45 with per-voxel parameters: F and dF/dz (+ gradient, reading C1)."""
    over = np.maximum(z - T, 0.0)
    under = np.maximum(T - z, 0.0)
    F = float(np.sum(w_over * over * over + w_under * under * under))
    return F, 2.0 * w_over * over - 2.0 * w_under * under


@dataclass
class MPResult:
    y: np.ndarray
    z: np.ndarray
    F: float
    n_iter: int
    reason: int
    F_hist: list = field(default_factory=list)       # F(it), it = 0 .. n_iter
    delta_hist: list = field(default_factory=list)   # delta used to leave iterate it, it = 0 .. n_iter-1
    g_A: np.ndarray = None                           # gradient at the returned iterate, after the subspace rule


def solve(DA, y0, lo, hi, T, w_over, w_under, max_iter=200, eps_F=1e-6, eps_y=1e-9) -> MPResult:
    """BB with the subspace step rule on min F(DA y), lo <= y <= hi.
    DA [n_voxels, m] (column k = DA(A_k), Eq. (5)); T, w_over, w_under per voxel [n_voxels]."""
    DA = np.asarray(DA, dtype=np.float64)
    T = np.asarray(T, dtype=np.float64)
    w_over = np.asarray(w_over, dtype=np.float64)
    w_under = np.asarray(w_under, dtype=np.float64)
    lo = np.asarray(lo, dtype=np.float64)
    hi = np.asarray(hi, dtype=np.float64)
    y = np.clip(np.asarray(y0, dtype=np.float64), lo, hi)                      # C16
    res = MPResult(y=y, z=None, F=0.0, n_iter=0, reason=0)
    y_prev = g_prev = None
    delta = 0.0
    it = 0
    while True:
        z = DA @ y                                                             # step 4 / Eq. (6), C20
        F, gz = objective(z, T, w_over, w_under)
        g = DA.T @ gz                                                          # step 1: gradient in the aperture domain
        held = ((y <= lo) & (g > 0.0)) | ((y >= hi) & (g < 0.0))               # Eq. (9), (10) with the sign of C15
        g = np.where(held, 0.0, g)
        res.F_hist.append(F)
        # ---- stopping rules (C19)
        reason = 0
        if not np.any(g != 0.0):
            reason = 1
        elif it >= 5 and all(abs(res.F_hist[j] - res.F_hist[j - 1]) <= eps_F * abs(res.F_hist[j - 1])
                             for j in range(it - 4, it + 1)):
            reason = 2
        elif it >= 1 and np.max(np.abs(y - y_prev)) <= eps_y:
            reason = 3
        elif it >= max_iter:
            reason = 4
        if reason:
            res.y, res.z, res.F, res.n_iter, res.reason, res.g_A = y, z, F, it, reason, g
            return res
        # ---- step 2: step size
        if it == 0:                                                            # C17
            q = DA @ g
            w = np.where(z > T, w_over, np.where(z < T, w_under, 0.0))
            den = 2.0 * float(np.sum(w * q * q))
            delta = float(g @ g) / den if den > 0.0 else 1.0
        else:                                                                  # Eq. (7) / (8), C18
            s = y - y_prev
            t = g - g_prev
            ss, st, tt = float(s @ s), float(s @ t), float(t @ t)
            if st > 0.0 and tt > 0.0:
                delta = ss / st if it % 2 == 1 else st / tt
        res.delta_hist.append(delta)
        # ---- step 3: update within the box
        y_prev, g_prev = y, g
        y = np.clip(y - delta * g, lo, hi)
        it += 1
