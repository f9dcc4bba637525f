"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Each test names the pin (P1..P12 of DESIGN.md) and the mistake it would catch.  None of them
re-types the oracle's loops: they use closed forms, invariants, library routines
(scipy.sparse), brute force of a different shape, or hand-worked fixtures in tests/golden/.
"""
import itertools
import os

import numpy as np
import pytest
import scipy.sparse as sp
import torch

import oracle
import synth
from conftest import as_np

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _x(n_b, k=0, scale=1.0):
    return synth.draw_x(n_b, k, scale=scale).numpy()


# ---------------------------------------------------------------- P4: closed forms, Eq. (1)
def _golden_1x1():
    rows = []
    for line in open(os.path.join(GOLDEN, "closed_form_1x1.txt")):
        line = line.split("#")[0].strip()
        if line:
            rows.append([float(t) for t in line.split()])
    return rows


@pytest.mark.parametrize("row", _golden_1x1())
def test_P4_closed_form_1x1(row):
    a, x, T, wo, wu, d_exp, F_exp, g_exp, p_exp = row
    vox, beam, val = np.array([0], np.int32), np.array([0], np.int32), np.array([a], np.float32)
    d = oracle.dose(vox, beam, val, 1, np.array([x], np.float32))
    F, g = oracle.objective_grad(d, np.array([0], np.uint8), [T], [wo], [wu])
    p = oracle.price(vox, beam, val, 1, g)
    assert d[0] == d_exp and F == F_exp and g[0] == g_exp and p[0] == p_exp


# ---------------------------------------------------------------- P1: D e_j = column j
def test_P1_unit_vector_reproduces_column(cfg0):
    A = as_np(cfg0)
    for j in range(A["n_b"]):
        e = np.zeros(A["n_b"], np.float32)
        e[j] = 1.0
        d = oracle.dose(A["vox"], A["beam"], A["val"], A["n_v"], e)
        col = np.zeros(A["n_v"])
        m = A["beam"] == j
        col[A["vox"][m]] = A["val"][m].astype(np.float64)     # no duplicate (voxel, beamlet) pairs
        assert np.array_equal(d, col), j


def test_P1b_no_duplicate_pairs_in_generator(cfg0):
    A = as_np(cfg0)
    key = A["vox"].astype(np.int64) * A["n_b"] + A["beam"]
    assert np.unique(key).size == key.size


# ---------------------------------------------------------------- library special case: scipy.sparse
def test_dose_and_price_match_scipy_sparse(cfg0):
    A = as_np(cfg0)
    D = sp.coo_matrix((A["val"].astype(np.float64), (A["vox"], A["beam"])), shape=(A["n_v"], A["n_b"])).tocsr()
    x = _x(A["n_b"], 0, 8.0)
    d = oracle.dose(A["vox"], A["beam"], A["val"], A["n_v"], x)
    np.testing.assert_allclose(d, D @ x.astype(np.float64), rtol=1e-13, atol=0)
    g = np.random.default_rng(1).standard_normal(A["n_v"])
    p = oracle.price(A["vox"], A["beam"], A["val"], A["n_b"], g)
    np.testing.assert_allclose(p, D.T @ g, rtol=0, atol=1e-12 * np.abs(p).max())


# ---------------------------------------------------------------- P2: adjoint identity
def test_P2_adjoint_identity(cfg0):
    A = as_np(cfg0)
    rng = np.random.default_rng(2)
    for k in range(3):
        x = _x(A["n_b"], k)
        g = rng.standard_normal(A["n_v"])
        lhs = np.dot(oracle.dose(A["vox"], A["beam"], A["val"], A["n_v"], x), g)
        rhs = np.dot(x.astype(np.float64), oracle.price(A["vox"], A["beam"], A["val"], A["n_b"], g))
        assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs))


# ---------------------------------------------------------------- P3: p is dF/dx (sign, factor 2, weights)
def _F_of_x(A, x):
    d = oracle.dose(A["vox"], A["beam"], A["val"], A["n_v"], x)
    return oracle.objective_grad(d, A["sid"], A["T"], A["wo"], A["wu"])[0]


@pytest.mark.parametrize("scale", [1.0, 8.0, 14.0, 16.0])
def test_P3_finite_difference_gradient(cfg0, scale):
    """Central differences of F(D x) equal p.  F is piecewise quadratic, so the central
    difference is exact up to rounding unless a voxel crosses a kink inside [x-eps, x+eps]."""
    A = as_np(cfg0)
    x = _x(A["n_b"], 3, scale).astype(np.float64)
    # FD needs FP64 steps: run the oracle's dose on an FP64 x by splitting x = hi + lo (both FP32-exact)
    def F64(xv):
        hi = xv.astype(np.float32)
        lo = (xv - hi.astype(np.float64)).astype(np.float32)
        d = oracle.dose(A["vox"], A["beam"], A["val"], A["n_v"], hi) + \
            oracle.dose(A["vox"], A["beam"], A["val"], A["n_v"], lo)
        return oracle.objective_grad(d, A["sid"], A["T"], A["wo"], A["wu"])[0]
    ev = oracle.price_eval(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], x.astype(np.float32),
                           A["sid"], A["T"], A["wo"], A["wu"], A["lco"], A["aro"])
    # the branches the scale is meant to reach (C13)
    if scale >= 8.0:
        assert (ev.g > 0).any() and (ev.g < 0).any()
    x = x.astype(np.float32).astype(np.float64)
    eps = 1e-3
    pscale = np.abs(ev.p).max()
    rng = np.random.default_rng(4)
    for j in rng.choice(A["n_b"], 12, replace=False):
        e = np.zeros_like(x)
        e[j] = eps
        fd = (F64(x + e) - F64(x - e)) / (2 * eps)
        assert abs(fd - ev.p[j]) <= 2e-5 * pscale, (j, fd, ev.p[j])
    for _ in range(3):                                    # random directions: <p, v>
        v = rng.standard_normal(A["n_b"])
        fd = (F64(x + eps * v) - F64(x - eps * v)) / (2 * eps)
        ref = np.dot(ev.p, v)
        assert abs(fd - ref) <= 1e-4 * np.linalg.norm(ev.p) * np.linalg.norm(v) / np.sqrt(A["n_b"]) + 1e-6 * abs(ref)


# ---------------------------------------------------------------- P5: the paper's first iteration (z = 0, L56)
def test_P5_first_iteration_closed_form(cfg0):
    A = as_np(cfg0)
    ev = oracle.price_eval(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], np.zeros(A["n_b"], np.float32),
                           A["sid"], A["T"], A["wo"], A["wu"], A["lco"], A["aro"])
    tgt = (A["wu"][A["sid"]] > 0)                          # voxels with an under-dose weight = targets
    assert tgt.sum() > 0
    assert np.array_equal(ev.d, np.zeros(A["n_v"]))
    assert ev.F == pytest.approx(float(np.sum(A["wu"][A["sid"]][tgt].astype(np.float64) * A["T"][A["sid"]][tgt].astype(np.float64) ** 2)), rel=1e-14)
    # p_j = -2 sum_{i in targets} w-_i T_i D_ij : a masked column sum, via bincount
    wT = 2.0 * A["wu"][A["sid"]].astype(np.float64) * A["T"][A["sid"]].astype(np.float64)
    colsum = np.bincount(A["beam"], weights=A["val"].astype(np.float64) * wT[A["vox"]], minlength=A["n_b"])
    np.testing.assert_allclose(ev.p, -colsum, rtol=1e-12, atol=0)
    touching = np.bincount(A["beam"], weights=tgt[A["vox"]].astype(np.float64), minlength=A["n_b"]) > 0
    assert (ev.p[touching] < 0).all() and (ev.p[~touching] == 0).all()
    # P12: every p <= 0 -> every row opens over all its negative beamlets, the aperture price is the
    # plain sum of the angle's prices and the best control point sees the largest target column mass
    mass = np.add.reduceat(colsum, A["aco"][:-1])
    np.testing.assert_allclose(ev.angle_price, -mass, rtol=1e-6)       # p rounded to FP32 before O4 (C6)
    assert ev.best_angle == int(np.argmax(mass))


# ---------------------------------------------------------------- P6: linearity, angle-block additivity (L119, L155)
def test_P6_linearity_and_angle_blocks(cfg0):
    A = as_np(cfg0)
    # x with <= 10 fractional bits: sums and doublings are exact in FP32
    xa = (np.floor(_x(A["n_b"], 5) * 1024) / 1024).astype(np.float32)
    xb = (np.floor(_x(A["n_b"], 6) * 1024) / 1024).astype(np.float32)
    dose = lambda x: oracle.dose(A["vox"], A["beam"], A["val"], A["n_v"], x)
    np.testing.assert_allclose(dose(xa + xb), dose(xa) + dose(xb), rtol=1e-13, atol=1e-13)
    assert np.array_equal(dose(2 * xa), 2 * dose(xa))
    # angle blocks: D = [D_1 ... D_A]  =>  d = sum_a D_a x_a ; p = concat_a D_a^T g
    x = _x(A["n_b"], 7, 8.0)
    d_full = dose(x)
    g = np.random.default_rng(8).standard_normal(A["n_v"])
    p_full = oracle.price(A["vox"], A["beam"], A["val"], A["n_b"], g)
    d_sum = np.zeros(A["n_v"])
    spec = synth.config_spec(0)
    for a in range(spec.n_angles):
        blk = synth.generate(spec, angles=[a])
        B = as_np(blk)
        assert B["n_b"] == A["n_b"]
        lo, hi = A["aco"][a], A["aco"][a + 1]
        assert B["beam"].min() >= lo and B["beam"].max() < hi
        d_sum += oracle.dose(B["vox"], B["beam"], B["val"], A["n_v"], x)
        p_blk = oracle.price(B["vox"], B["beam"], B["val"], A["n_b"], g)
        np.testing.assert_allclose(p_blk[lo:hi], p_full[lo:hi], rtol=1e-12, atol=1e-12)
        assert not p_blk[:lo].any() and not p_blk[hi:].any()
    np.testing.assert_allclose(d_sum, d_full, rtol=1e-12, atol=1e-12)


# ---------------------------------------------------------------- P9: COO order invariance
def test_P9_permutation_invariance(cfg0):
    A = as_np(cfg0)
    x = _x(A["n_b"], 9, 14.0)
    ref = oracle.price_eval(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], x, A["sid"], A["T"], A["wo"],
                            A["wu"], A["lco"], A["aro"])
    perm = np.random.default_rng(10).permutation(A["vox"].size)
    ev = oracle.price_eval(A["vox"][perm], A["beam"][perm], A["val"][perm], A["n_v"], A["n_b"], x, A["sid"],
                           A["T"], A["wo"], A["wu"], A["lco"], A["aro"])
    np.testing.assert_allclose(ev.d, ref.d, rtol=1e-12)
    np.testing.assert_allclose(ev.p, ref.p, rtol=0, atol=1e-11 * np.abs(ref.p).max())
    assert abs(ev.F - ref.F) <= 1e-12 * ref.F
    assert np.array_equal(ev.L, ref.L) and np.array_equal(ev.R, ref.R) and ev.best_angle == ref.best_angle


# ---------------------------------------------------------------- O4 pins: P8, P10, P11
def _golden_rows():
    out = []
    for line in open(os.path.join(GOLDEN, "rows_adversarial.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        lhs, rhs = line.split("|")
        p = [float(t) for t in lhs.split()]
        L, R, V = rhs.split()
        out.append((p, int(L), int(R), float(V)))
    return out


def _select_one(p):
    p = np.asarray(p, np.float32)
    L, R, V = oracle.select_rows(p, np.array([0, p.size], np.int32))
    return int(L[0]), int(R[0]), float(V[0])


@pytest.mark.parametrize("case", _golden_rows())
def test_P11_hand_worked_rows(case):
    p, L, R, V = case
    assert _select_one(p) == (L, R, V)


def _brute_n3(p):
    """Independent O(n^3) enumeration: sums p[L:R] directly (no prefix sums), lexicographic (V,L,R)."""
    n = len(p)
    best = (0.0, 0, 0)
    for L in range(n + 1):
        for R in range(L, n + 1):
            V = 0.0
            for c in range(L, R):
                V += float(p[c])
            if (V, L, R) < best:
                best = (V, L, R)
    return best[1], best[2], best[0]


def test_P8_exhaustive_small_integer_rows():
    """Every row over {-2..2}^n, n <= 5: integer sums are exact in both enumerations."""
    for n in range(0, 6):
        for p in itertools.product([-2.0, -1.0, 0.0, 1.0, 2.0], repeat=n):
            assert _select_one(p) == _brute_n3(p), p


def test_P8_random_integer_rows_and_batched_offsets():
    rng = np.random.default_rng(11)
    lens = rng.integers(0, 9, size=200)
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    p = rng.integers(-6, 5, size=off[-1]).astype(np.float32)
    L, R, V = oracle.select_rows(p, off)
    for r in range(lens.size):
        assert (int(L[r]), int(R[r]), float(V[r])) == _brute_n3(p[off[r]:off[r + 1]]), r


def test_P8_config0_rows_against_direct_sums(cfg0):
    A = as_np(cfg0)
    x = _x(A["n_b"], 12, 14.0)             # x14: mixed-sign prices, partially open rows (C13)
    ev = oracle.price_eval(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], x, A["sid"], A["T"], A["wo"],
                           A["wu"], A["lco"], A["aro"])
    assert (ev.R > ev.L).any() and (ev.p_f32 > 0).any() and (ev.p_f32 < 0).any()
    for r in range(A["lco"].size - 1):
        row = ev.p_f32[A["lco"][r]:A["lco"][r + 1]].astype(np.float64)
        L, R, V = _brute_n3(row)
        assert abs(V - ev.row_price[r]) <= 1e-12 * max(1.0, np.abs(row).sum())
        if (L, R) != (ev.L[r], ev.R[r]):       # only a rounding-level tie may differ
            assert abs(row[min(L, ev.L[r]):max(R, ev.R[r])].sum() - V) <= 1e-9 * np.abs(row).sum()


def test_P10_selection_invariants():
    rng = np.random.default_rng(13)
    for _ in range(300):
        n = int(rng.integers(1, 40))
        p = (rng.standard_normal(n) * 10).astype(np.float32)
        p[rng.random(n) < 0.15] = 0.0
        L, R, V = _select_one(p)
        assert 0 <= L <= R <= n and V <= 0.0
        if p.min() < 0:
            assert V <= float(p.min())
            assert R > L and p[L] <= 0 and p[R - 1] < 0
        else:
            assert (L, R, V) == (0, 0, 0.0)
        # no single extension or contraction improves it
        S = np.concatenate([[0.0], np.cumsum(p.astype(np.float64))])
        assert V == S[R] - S[L]
        assert V <= (S[1:, None] - S[None, :-1])[np.tril_indices(n)].min() + 0.0
    assert _select_one(-np.ones(7)) == (0, 7, -7.0)
    assert _select_one(np.ones(7)) == (0, 0, 0.0)


def test_P12_angle_price_and_mask():
    rp = np.array([-1.0, -2.0, 0.0, -0.5, -4.0, 0.0, 0.0], np.float64)
    aro = np.array([0, 2, 4, 5, 7], np.int32)
    ap, best = oracle.angle_price(rp, aro)
    assert ap.tolist() == [-3.0, -0.5, -4.0, 0.0] and best == 2
    ap, best = oracle.angle_price(rp, aro, np.array([0, 0, 1, 0], np.uint8))
    assert ap[2] == np.inf and best == 0
    ap, best = oracle.angle_price(np.zeros(7), aro)
    assert best == -1                                   # no improving aperture: stop (L56)
    ap, best = oracle.angle_price(np.array([-1.0, -2.0, -3.0, 0, 0, 0, 0]), aro)
    assert best == 0 and ap[0] == ap[1] == -3.0           # tie -> smallest control point


def test_storage_closed_form_of_table2():
    """PAPER.md Table 2 (L198-L202): COO 12 B/nnz, CSR 8 B/nnz - pins FP32 values + int32 indices."""
    for nnz, coo_gib, csr_gib in [(608447419, 6.80, 4.53), (159839137, 1.79, 1.19)]:
        assert round(12 * nnz / 2 ** 30, 2) == coo_gib
        assert round(8 * nnz / 2 ** 30, 2) == csr_gib
