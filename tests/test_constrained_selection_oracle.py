"""Pins of the oracle's constrained aperture selection O6 (oracle_select_constrained; PAPER.md L133-L135, L66;
DESIGN.md readings C22-C24).  None of them re-types the oracle's recursion:
  * hand-worked control points in tests/golden/interdigitation_cases.txt;
  * exhaustive enumeration of EVERY combination of row states of tiny control points (the paper's own definition,
    L135: "calculating the prices of all the combinations of openings at different MLC rows that can satisfy the
    interdigitation constraint"), constraint checked with the formula as printed, prices summed directly from p;
  * without constraints it must reduce to the pinned O4 / O5 routines;
  * invariants on config 0's real prices: feasibility of the result, constrained optimum >= unconstrained optimum,
    equality when the unconstrained apertures already satisfy the constraint.
"""
import itertools
import os

import numpy as np
import pytest

import oracle
import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "interdigitation_cases.txt")


def parse_cases():
    cases = []
    for ln in open(GOLDEN):
        ln = ln.strip()
        if not ln or ln.startswith("#"):
            continue
        mode, pos0, rows, wins, exp, price = [t.strip() for t in ln.split(";")]
        rows = [[float(v) for v in r.split()] for r in rows.split("|")]
        pos0 = [int(v) for v in pos0.split()]
        n_rows = len(rows)
        W = None
        if wins != "-":
            big = 1 << 20
            W = [np.full(n_rows, -big, np.int32), np.full(n_rows, big, np.int32),
                 np.full(n_rows, -big, np.int32), np.full(n_rows, big, np.int32)]
            for ent in wins.split(","):
                r, a, b, c, d = [int(v) for v in ent.split()]
                W[0][r], W[1][r], W[2][r], W[3][r] = a, b, c, d
        exp = [[int(v) for v in e.split()] for e in exp.split("|")]
        cases.append((mode == "I", pos0, rows, W, exp, float(price)))
    return cases


def run_oracle(rows, pos0, interdig, W=None, mask=None):
    p = np.array([v for r in rows for v in r], dtype=np.float32)
    lco = np.concatenate([[0], np.cumsum([len(r) for r in rows])]).astype(np.int32)
    aro = np.array([0, len(rows)], dtype=np.int32)
    kw = {} if W is None else dict(L_lo=W[0], L_hi=W[1], R_lo=W[2], R_hi=W[3])
    return oracle.select_constrained(p, aro, lco, np.array(pos0, np.int32), interdig, angle_mask=mask, **kw)


@pytest.mark.parametrize("case", parse_cases())
def test_hand_worked_control_points(case):
    interdig, pos0, rows, W, exp, price = case
    L, R, rp, ap, best = run_oracle(rows, pos0, interdig, W)
    assert [[int(l), int(r)] for l, r in zip(L, R)] == exp
    assert ap[0] == price
    assert best == (0 if price < 0 else -1)
    for r, row in enumerate(rows):                                  # row prices are the sums of the exposed beamlets
        assert rp[r] == sum(row[L[r]:R[r]]) if R[r] > L[r] else rp[r] == 0.0


def brute_force(rows, pos0, interdig, W):
    """Every combination of row states, straight from the definitions (L135 as printed)."""
    nonempty = [r for r in range(len(rows)) if len(rows[r]) > 0]
    Pmin = min((pos0[r] for r in nonempty), default=0)
    Pmax = max((pos0[r] + len(rows[r]) for r in nonempty), default=0)
    per_row = []
    for r, row in enumerate(rows):
        n = len(row)
        u0 = pos0[r] if n > 0 else Pmin
        st = []
        for a in range(Pmin, Pmax + 1):
            for b in range(a, Pmax + 1):
                L, R = a - u0, b - u0
                if a < b and not (n > 0 and 0 <= L and R <= n):
                    continue
                if W is not None and not (W[0][r] <= L <= W[1][r] and W[2][r] <= R <= W[3][r]):
                    continue
                st.append((a, b, sum(row[L:R]) if a < b else 0.0, L, R))
        per_row.append(st)
    best_key, best_combo = None, None
    for combo in itertools.product(*per_row):
        if interdig:
            ok = True
            for r in range(len(combo)):
                nb = [combo[q][1] for q in (r - 1, r + 1) if 0 <= q < len(combo)]
                if nb and combo[r][0] > min(nb):                      # L_{k,irow} <= min{R_{k,irow-1}, R_{k,irow+1}}
                    ok = False
                    break
            if not ok:
                continue
        total = sum(s[2] for s in combo)
        key = (total,) + tuple((s[0], s[1]) for s in reversed(combo))
        if best_key is None or key < best_key:
            best_key, best_combo = key, combo
    return best_combo, (best_key[0] if best_key else None)


def test_exhaustive_enumeration_of_all_combinations():
    rng = np.random.default_rng(1503)
    n_checked = n_infeasible = 0
    for trial in range(400):
        n_rows = int(rng.integers(1, 5))
        rows = [list(rng.integers(-3, 4, size=int(rng.integers(0, 4))).astype(float)) for _ in range(n_rows)]
        pos0 = [int(rng.integers(0, 3)) for _ in range(n_rows)]
        interdig = bool(trial % 2)
        W = None
        if trial % 3 == 0:
            lo = rng.integers(-1, 3, size=(2, n_rows))
            W = [lo[0].astype(np.int32), (lo[0] + rng.integers(0, 4, n_rows)).astype(np.int32),
                 lo[1].astype(np.int32), (lo[1] + rng.integers(0, 4, n_rows)).astype(np.int32)]
        combo, total = brute_force(rows, pos0, interdig, W)
        L, R, rp, ap, best = run_oracle(rows, pos0, interdig, W)
        if combo is None:
            assert np.isinf(ap[0]) and best == -1 and not L.any() and not R.any()
            n_infeasible += 1
            continue
        assert ap[0] == total, (trial, rows, pos0, W)
        assert [(int(l), int(r)) for l, r in zip(L, R)] == [(s[3], s[4]) for s in combo], (trial, rows, pos0, W)
        assert list(rp) == [s[2] for s in combo]
        assert best == (0 if total < 0 else -1)
        n_checked += 1
    assert n_checked > 300 and n_infeasible > 5                      # both outcomes were exercised


def config0_prices(scale):
    ph = synth.generate(synth.config_spec(0))
    x = synth.draw_x(ph.n_beamlets, 0, scale=scale).numpy()
    ev = oracle.price_eval(ph.coo_voxel.numpy(), ph.coo_beamlet.numpy(), ph.coo_val.numpy(), ph.n_voxels,
                           ph.n_beamlets, x, ph.voxel_struct.numpy(), ph.struct_T.numpy(), ph.struct_w_over.numpy(),
                           ph.struct_w_under.numpy(), ph.leafrow_col_offset.numpy(), ph.angle_row_offset.numpy())
    return ph, ev


def satisfies_interdigitation(L, R, pos0, aro, lco=None):
    """L135 for every adjacent pair of rows, in physical positions (rows without beamlets count from Pmin)."""
    u0 = np.array(pos0, dtype=np.int64)
    if lco is not None:
        n = np.diff(lco)
        for k in range(len(aro) - 1):
            sl = slice(aro[k], aro[k + 1])
            ne = n[sl] > 0
            u0[sl][~ne] = u0[sl][ne].min() if ne.any() else 0
    a, b = L + u0, R + u0
    for k in range(len(aro) - 1):
        for r in range(aro[k], aro[k + 1] - 1):
            if a[r] > b[r + 1] or a[r + 1] > b[r]:
                return False
    return True


@pytest.mark.parametrize("scale", [1.0, 14.0, 16.0])
def test_without_constraints_it_reduces_to_O4_O5(scale):
    ph, ev = config0_prices(scale)
    aro, lco, u0 = ph.angle_row_offset.numpy(), ph.leafrow_col_offset.numpy(), ph.leafrow_pos0.numpy()
    L, R, rp, ap, best = oracle.select_constrained(ev.p_f32, aro, lco, u0, False)
    open_rows = ev.R > ev.L
    assert np.array_equal(L[open_rows], ev.L[open_rows]) and np.array_equal(R[open_rows], ev.R[open_rows])
    assert np.array_equal(L[~open_rows], R[~open_rows])             # closed rows stay closed (parked at the left end)
    assert np.array_equal(rp, ev.row_price)
    assert np.array_equal(ap, ev.angle_price) and best == ev.best_angle


@pytest.mark.parametrize("scale", [1.0, 14.0, 16.0])
def test_invariants_on_config0(scale):
    ph, ev = config0_prices(scale)
    aro, lco, u0 = ph.angle_row_offset.numpy(), ph.leafrow_col_offset.numpy(), ph.leafrow_pos0.numpy()
    L, R, rp, ap, best = oracle.select_constrained(ev.p_f32, aro, lco, u0, True)
    assert satisfies_interdigitation(L, R, u0, aro)
    assert (ap >= ev.angle_price).all()                              # a constraint never improves the optimum
    for k in range(len(aro) - 1):
        sl = slice(aro[k], aro[k + 1])
        S = [np.concatenate([[0.0], np.cumsum(ev.p_f32[lco[r]:lco[r + 1]].astype(np.float64))]) for r in range(sl.start, sl.stop)]
        assert list(rp[sl]) == [s[R[sl][i]] - s[L[sl][i]] if R[sl][i] > L[sl][i] else 0.0 for i, s in enumerate(S)]
        if satisfies_interdigitation(ev.L[sl], ev.R[sl], u0[sl], np.array([0, sl.stop - sl.start])) and \
                (ev.R[sl] > ev.L[sl]).all():
            assert ap[k] == ev.angle_price[k]
            assert np.array_equal(L[sl], ev.L[sl]) and np.array_equal(R[sl], ev.R[sl])


def test_mask_windows_and_infeasible_control_points():
    rows = [[-1.0, -2.0, -1.0], [-1.0, -1.0, -1.0]]
    # an occupied control point is skipped
    L, R, rp, ap, best = run_oracle(rows, [0, 0], True, mask=np.array([1], np.uint8))
    assert np.isinf(ap[0]) and best == -1 and not L.any() and not R.any()
    # windows that pin both rows to one state each return exactly that state
    W = [np.array([1, 0], np.int32), np.array([1, 0], np.int32), np.array([2, 3], np.int32), np.array([2, 3], np.int32)]
    L, R, rp, ap, best = run_oracle(rows, [0, 0], True, W)
    assert list(L) == [1, 0] and list(R) == [2, 3] and ap[0] == -5.0 and best == 0
    # windows nobody can meet: no feasible aperture
    W = [np.array([2, 0], np.int32), np.array([2, 0], np.int32), np.array([1, 0], np.int32), np.array([1, 3], np.int32)]
    L, R, rp, ap, best = run_oracle(rows, [0, 0], False, W)
    assert np.isinf(ap[0]) and best == -1
    # pinned states that interdigitate: row 0 = (2,3), row 1 = (0,1): a_0 = 2 > b_1 = 1
    W = [np.array([2, 0], np.int32), np.array([2, 0], np.int32), np.array([3, 1], np.int32), np.array([3, 1], np.int32)]
    assert np.isinf(run_oracle(rows, [0, 0], True, W)[3][0])
    assert run_oracle(rows, [0, 0], False, W)[3][0] == -2.0


def test_several_control_points_and_best_angle():
    # three control points: the middle one has the best constrained aperture although its unconstrained one is not the best
    p = np.array([-1, 5, 5, 5, 5, -1,      # cp 0: rows collide, constrained price -1 (unconstrained -2)
                  -1, -0.5, 0, 0, 0, 0,    # cp 1: -1.5, compatible as it is
                  0, 0, 0, 0, 0, 0],       # cp 2: nothing to gain
                 dtype=np.float32)
    aro = np.array([0, 2, 4, 6], np.int32)
    lco = np.arange(0, 19, 3).astype(np.int32)
    u0 = np.zeros(6, np.int32)
    L, R, rp, ap, best = oracle.select_constrained(p, aro, lco, u0, True)
    assert list(ap) == [-1.0, -1.5, 0.0] and best == 1
    L2, R2, rp2, ap2, best2 = oracle.select_constrained(p, aro, lco, u0, False)
    assert list(ap2) == [-2.0, -1.5, 0.0] and best2 == 0
