"""CPU FP64 oracle of the column-generation loop - TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md L56 (section 2.1) and Figure 1(a): "The algorithm starts with an initial dose distribution z = 0
and no apertures.  At each iteration step, it attempts to improve the current solution by choosing an
aperture among the control points that haven't been occupied yet, and then optimizing the fluence rates of
all currently generated apertures ... until no more apertures at unoccupied beam angles could be found such
that the objective function can be further decreased."

One outer iteration, in the paper's order (L58-L68, L127-L139):
  PP1  g = dF/dz at the current dose (Eq. (1), (4); sign C1), beamlet prices p = D^T g (Eq. (3))
  PP2  per leaf row of every unoccupied control point the best opening (L133; readings C4-C8), per control
       point the sum of its rows' prices, the control point with the smallest sum; stop if none is < 0
       aperture dose vector DA(A_k) = sum_{j in A_k} D_:j (Eq. (5))
  MP   fluence rates of all apertures so far by BB (oracle/master_problem.py), warm-started from the previous
       solution with the new aperture at y = 0 (clipped into its bounds); z = DA y
It only strings together oracle functions that are pinned on their own (tests/test_oracle_pins.py,
tests/test_master_problem_oracle.py); nothing here comes from the CUDA path.

Readings (C7, C21): all beamlets of unoccupied control points are priced; every aperture gets the
same caller-supplied bounds [y_lo, y_hi].  The selection works on the FP32-rounded price vector (C6).

Optional hardware constraints (NEXT-3; readings C22-C25): `interdigitation` (L135) and `max_leaf_travel`
(L66: "the candidate apertures need to be compatible with those chosen apertures" at neighbouring control
points, through s_k <= S^U_{k,k+1}(A_k, A_{k+1}); PAPER.md does not define S^U, so the caller gives the
largest distance, in beamlet widths, a leaf end may move per control-point step - reading C25).  Then PP2 is
`select_constrained` (O6) with the windows of `leaf_windows`, and the loop also stops when the best feasible
aperture has a price >= 0.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import angle_price, dose, objective_grad, price, select_constrained, select_rows
from . import master_problem as mp


@dataclass
class CGResult:
    angles: list = field(default_factory=list)      # control point of aperture k, in the order chosen
    L: np.ndarray = None                            # [n_leaf_rows] openings of the chosen apertures, 0 elsewhere
    R: np.ndarray = None
    y: np.ndarray = None                            # [n_apertures] fluence rates
    z: np.ndarray = None                            # [n_voxels] final dose
    F_hist: list = field(default_factory=list)      # F(z = 0), then F after every master problem
    aperture_price: list = field(default_factory=list)   # price of aperture k when it was chosen (< 0)
    mp_iters: list = field(default_factory=list)
    stop: str = ""                                  # "no improving aperture" | "max_apertures"


BIG = 1 << 30                                       # "no bound" of a leaf window


def leaf_windows(angle_mask, L, R, leafrow_col_offset, angle_row_offset, leafrow_pos0, arc_angle_offset,
                 max_leaf_travel):
    """Reading C25.  For every leaf row of every UNOCCUPIED control point k the interval each leaf end may take
    so that the row can be reached from / can reach the same leaf row of the nearest occupied control point on
    either side of k within k's arc: a leaf end moves at most max_leaf_travel beamlet widths per control-point
    step, so |a_k - a_k'| <= max_leaf_travel * |k - k'| and the same for b.  Positions are physical (row-local
    + pos0; rows without beamlets count from the left end Pmin of their control point's field range, as in O6);
    the windows are returned row-local: (L_lo, L_hi, R_lo, R_hi), -BIG / +BIG where nothing binds.  Rows of
    occupied control points get no bound (they are not priced)."""
    lco, aro = np.asarray(leafrow_col_offset), np.asarray(angle_row_offset)
    n_rows, n_a = lco.size - 1, aro.size - 1
    n = np.diff(lco)
    u0 = np.asarray(leafrow_pos0, dtype=np.int64).copy()
    for k in range(n_a):                                                        # empty rows count from Pmin
        sl = slice(aro[k], aro[k + 1])
        ne = n[sl] > 0
        u0[sl][~ne] = u0[sl][ne].min() if ne.any() else 0
    W = [np.full(n_rows, -BIG, np.int32), np.full(n_rows, BIG, np.int32),
         np.full(n_rows, -BIG, np.int32), np.full(n_rows, BIG, np.int32)]
    arcs = np.asarray(arc_angle_offset)
    for s in range(arcs.size - 1):
        for k in range(arcs[s], arcs[s + 1]):
            if angle_mask[k]:
                continue
            nbrs = []
            for step in (-1, 1):                                                # nearest occupied control point on each side
                kk = k + step
                while arcs[s] <= kk < arcs[s + 1] and not angle_mask[kk]:
                    kk += step
                if arcs[s] <= kk < arcs[s + 1]:
                    nbrs.append(kk)
            for kk in nbrs:
                assert aro[kk + 1] - aro[kk] == aro[k + 1] - aro[k], "control points of an arc share the MLC"
                reach = max_leaf_travel * abs(kk - k)
                for rho in range(aro[k + 1] - aro[k]):
                    r, rr = aro[k] + rho, aro[kk] + rho
                    a, b = L[rr] + u0[rr], R[rr] + u0[rr]                       # physical positions of the neighbour's row
                    W[0][r] = max(W[0][r], a - reach - u0[r]); W[1][r] = min(W[1][r], a + reach - u0[r])
                    W[2][r] = max(W[2][r], b - reach - u0[r]); W[3][r] = min(W[3][r], b + reach - u0[r])
    return W


def run(coo_voxel, coo_beamlet, coo_val, n_voxels, n_beamlets, voxel_struct, T, w_over, w_under,
        leafrow_col_offset, angle_row_offset, max_apertures, y_lo, y_hi, mp_max_iter=300, eps_F=1e-10,
        eps_y=1e-12, interdigitation=False, max_leaf_travel=-1, leafrow_pos0=None, arc_angle_offset=None) -> CGResult:
    lco = np.asarray(leafrow_col_offset)
    aro = np.asarray(angle_row_offset)
    constrained = bool(interdigitation) or max_leaf_travel >= 0
    n_a, n_rows = aro.size - 1, lco.size - 1
    sid = np.asarray(voxel_struct)
    Tv, wov, wuv = (np.asarray(a, dtype=np.float32)[sid].astype(np.float64) for a in (T, w_over, w_under))
    res = CGResult(L=np.zeros(n_rows, np.int32), R=np.zeros(n_rows, np.int32), y=np.zeros(0), z=np.zeros(n_voxels))
    mask = np.zeros(n_a, np.uint8)
    cols = []
    F0, _ = objective_grad(res.z, sid, T, w_over, w_under)
    res.F_hist.append(F0)
    while True:
        if len(cols) >= max_apertures:
            res.stop = "max_apertures"
            return res
        _, g = objective_grad(res.z, sid, T, w_over, w_under)                  # PP1
        p = price(coo_voxel, coo_beamlet, coo_val, n_beamlets, g)
        if constrained:                                                        # PP2 under hardware constraints (O6)
            W = [None] * 4
            if max_leaf_travel >= 0:
                W = leaf_windows(mask, res.L, res.R, lco, aro, leafrow_pos0, arc_angle_offset, max_leaf_travel)
            L, R, rp, ap, best = select_constrained(p.astype(np.float32), aro, lco, leafrow_pos0, interdigitation,
                                                    angle_mask=mask, L_lo=W[0], L_hi=W[1], R_lo=W[2], R_hi=W[3])
        else:
            L, R, rp = select_rows(p.astype(np.float32), lco)                  # PP2 (C6)
            for a in np.nonzero(mask)[0]:                                      # occupied control points stay closed (C7)
                L[aro[a]:aro[a + 1]] = 0
                R[aro[a]:aro[a + 1]] = 0
                rp[aro[a]:aro[a + 1]] = 0.0
            ap, best = angle_price(rp, aro, mask)
        if best < 0:                                                           # L56: nothing decreases F any more
            res.stop = "no improving aperture"
            return res
        rows = slice(aro[best], aro[best + 1])
        res.L[rows], res.R[rows] = L[rows], R[rows]
        ind = np.zeros(n_beamlets, np.float32)                                 # Eq. (5)
        for r in range(aro[best], aro[best + 1]):
            ind[lco[r] + L[r]: lco[r] + R[r]] = 1.0
        cols.append(dose(coo_voxel, coo_beamlet, coo_val, n_voxels, ind))
        mask[best] = 1
        res.angles.append(int(best))
        res.aperture_price.append(float(ap[best]))
        m = len(cols)
        sol = mp.solve(np.stack(cols, 1), np.concatenate([res.y, [0.0]]), np.full(m, y_lo), np.full(m, y_hi),
                       Tv, wov, wuv, max_iter=mp_max_iter, eps_F=eps_F, eps_y=eps_y)      # MP, warm start
        res.y, res.z = sol.y, sol.z
        res.F_hist.append(sol.F)
        res.mp_iters.append(sol.n_iter)
