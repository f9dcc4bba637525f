"""GPU parity of the master problem (vmat_mp_*, NEXT-2) against oracle/master_problem.py.

The method is an iteration, so parity is checked (a) on the trace: objective value and step size of every
iteration, (b) on the returned iterate (y, z, F, iteration count, stopping rule).  The CUDA path sums in FP64 in
its own fixed order, so it differs from the FP64 oracle by summation order only: the tolerances are 1e-9
relative on the trace and on y (BB amplifies rounding differences over hundreds of iterations), 1e-5 / 1e-4 on
the FP32 dose z (`north_star`'s vector tolerance).
"""
import numpy as np
import pytest
import torch

import synth
from conftest import as_np
from helpers import assert_vec_close, ddc_from_arrays, obj_to_device
from oracle import master_problem as omp

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
TRACE_RTOL = 1e-9


@pytest.fixture(scope="module")
def vm():
    import paper_1503_01721_b200 as vm
    vm.load_library()
    return vm


def _random_mp(rng, n_v, m, n_struct=4, density=0.6):
    DA = (rng.random((n_v, m)) * (rng.random((n_v, m)) < density)).astype(np.float32)
    sid = rng.integers(0, n_struct, n_v).astype(np.uint8)
    T = np.array([30.0, 70.0, 20.0, 50.0], np.float32)[:n_struct]
    wo = np.array([0.2, 1.0, 0.05, 0.7], np.float32)[:n_struct]
    wu = np.array([0.0, 1.0, 0.0, 0.3], np.float32)[:n_struct]
    return DA, sid, T, wo, wu


def _solve_both(vm, DA, sid, T, wo, wu, y0, lo, hi, max_iter, eps_F, eps_y, m_cap=None):
    n_v, m = DA.shape
    ref = omp.solve(DA.astype(np.float64), y0, lo, hi, T[sid].astype(np.float64), wo[sid].astype(np.float64),
                    wu[sid].astype(np.float64), max_iter=max_iter, eps_F=eps_F, eps_y=eps_y)
    mp = vm.MasterProblem(n_v, m_cap or m, DEV)
    for k in range(m):
        mp.add_aperture(torch.from_numpy(np.ascontiguousarray(DA[:, k])).to(DEV), y0[k], lo[k], hi[k])
    obj = vm.Objective(torch.from_numpy(sid).to(DEV), torch.from_numpy(T).to(DEV), torch.from_numpy(wo).to(DEV),
                       torch.from_numpy(wu).to(DEV))
    z = torch.empty(n_v, dtype=torch.float32, device=DEV)
    sol = mp.solve(obj, max_iter=max_iter, eps_F=eps_F, eps_y=eps_y, z=z)
    Fh, dh = mp.history()
    return ref, sol, z.cpu().numpy(), Fh.numpy(), dh.numpy(), mp, obj


def _check(ref, sol, z, Fh, dh, trace_rtol=TRACE_RTOL):
    assert sol.n_iter == ref.n_iter and sol.reason == ref.reason
    assert np.allclose(Fh, np.array(ref.F_hist), rtol=trace_rtol, atol=0.0)
    assert np.allclose(dh, np.array(ref.delta_hist), rtol=trace_rtol, atol=0.0)
    scale = max(1.0, float(np.abs(ref.y).max()))
    assert np.abs(sol.y.numpy() - ref.y).max() <= trace_rtol * scale
    assert abs(sol.F - ref.F) <= trace_rtol * abs(ref.F)
    assert_vec_close("z", z, ref.z)


@pytest.mark.parametrize("n_v,m", [(1, 1), (37, 1), (1000, 3), (5000, 8), (3001, 31), (4000, 32), (2500, 33),
                                   (2000, 100), (1500, 257), (700, 384)])
def test_trace_and_solution_match_the_oracle(vm, n_v, m):
    """Every group size (G = 1 .. 32), every chunk count (1, 2, 4, 8, 12) and ragged voxel counts."""
    rng = np.random.default_rng(1000 + n_v + m)
    DA, sid, T, wo, wu = _random_mp(rng, n_v, m)
    lo, hi = np.zeros(m), np.full(m, 40.0)
    y0 = rng.uniform(0.0, 1.0, m)
    # 12 iterations: far from the rounding floor, where "F has stopped changing" would depend on summation order
    ref, sol, z, Fh, dh, mp, _ = _solve_both(vm, DA, sid, T, wo, wu, y0, lo, hi, max_iter=12, eps_F=0.0, eps_y=0.0)
    _check(ref, sol, z, Fh, dh)
    assert ref.n_iter == 12 or ref.reason == 1
    mp.close()


# ---- the pass kernel in its steady state (every instantiation runs >= 3 grid steps with a ragged tail)
# vmat_mp_pass_geometry reports, for m apertures, the number of voxel rows the whole grid takes per step of its
# grid-stride loop; a parity case only exercises the prefetch ring's wrap and the accumulation over steps when the
# reached voxels span several such steps (PAPER.md L139 steps 4 + 1, Eq. (6)-(10) L70-L101).
STEADY_CASES = [8, 32, 48, 64, 100, 128, 200, 256, 300, 384]


def _steady_problem(vm, m, rng, steps=3.4, dead_frac=0.3):
    rows = vm.mp_pass_geometry(m)["rows_per_grid_step"]
    n_reached_target = int(steps * rows) + 37                 # ragged tail: not a multiple of anything
    n_v = int(n_reached_target / (1.0 - dead_frac)) + 1
    DA, sid, T, wo, wu = _random_mp(rng, n_v, m, density=0.5)
    dead = rng.random(n_v) < dead_frac
    DA[dead] = 0.0
    DA[~dead, rng.integers(0, m)] += np.float32(0.125)        # every other row is reached for certain
    return DA, sid, T, wo, wu, rows


@pytest.mark.parametrize("m", STEADY_CASES)
def test_pass_kernel_steady_state_matches_the_oracle(vm, m):
    rng = np.random.default_rng(31000 + m)
    DA, sid, T, wo, wu, rows = _steady_problem(vm, m, rng)
    n_v = DA.shape[0]
    reached = int((DA != 0).any(axis=1).sum())
    assert reached >= 3.3 * rows and reached % rows != 0      # >= 3 full grid steps + a ragged one
    lo, hi = np.zeros(m), np.full(m, 40.0)
    y0 = rng.uniform(0.0, 1.0, m)
    ref, sol, z, Fh, dh, mp, _ = _solve_both(vm, DA, sid, T, wo, wu, y0, lo, hi, max_iter=12, eps_F=0.0, eps_y=0.0)
    print(f"\n[mp steady] m={m}: {n_v} voxels, {reached} reached = {reached / rows:.2f} grid steps of {rows} rows, "
          f"F {ref.F_hist[0]:.4e} -> {ref.F:.4e}")
    assert mp.n_reached_voxels == reached
    _check(ref, sol, z, Fh, dh)
    assert ref.n_iter == 12
    mp.close()


@pytest.mark.parametrize("n_v,m", [(1800, 129), (1200, 200), (900, 256), (2500, 64), (2100, 40), (1700, 160)])
def test_trace_matches_the_oracle_more_widths(vm, n_v, m):
    """Aperture counts the first parametrisation leaves out: 129..256 (two 16-byte chunks per lane) and 33..64."""
    rng = np.random.default_rng(2000 + n_v + m)
    DA, sid, T, wo, wu = _random_mp(rng, n_v, m)
    lo, hi = np.zeros(m), np.full(m, 40.0)
    y0 = rng.uniform(0.0, 1.0, m)
    ref, sol, z, Fh, dh, mp, _ = _solve_both(vm, DA, sid, T, wo, wu, y0, lo, hi, max_iter=12, eps_F=0.0, eps_y=0.0)
    _check(ref, sol, z, Fh, dh)
    mp.close()


def test_master_problem_at_the_bench_shape_config3(vm):
    """The shape bench.py times (`master_problem`): 128 apertures on config 3's voxel set (1.24e6 voxels), one per
    evenly spaced control point, random contiguous openings, columns by vmat_aperture_dose (Eq. (5)); 12 BB
    iterations against the oracle fed the SAME FP32 columns (downloaded from the device)."""
    m = 128
    ph = synth.generate(synth.config_spec(3), device=DEV)
    h = vm.vmat_ddc_create(ph.n_voxels, ph.n_beamlets, ph.coo_voxel, ph.coo_beamlet, ph.coo_val,
                           ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset, device=DEV)
    ph.coo_voxel = ph.coo_beamlet = ph.coo_val = None
    torch.cuda.empty_cache()
    n_v, n_a, n_rows = h.n_voxels, h.n_angles, h.n_leaf_rows
    gen = torch.Generator().manual_seed(20150301)
    lco = ph.leafrow_col_offset.to(torch.int64)
    lens = (lco[1:] - lco[:-1]).to(torch.float64)
    a, b = torch.rand(n_rows, generator=gen, dtype=torch.float64), torch.rand(n_rows, generator=gen, dtype=torch.float64)
    L = (torch.minimum(a, b) * lens).floor().to(torch.int32).to(DEV)
    R = (torch.maximum(a, b) * lens).ceil().to(torch.int32).to(DEV)
    mp = vm.MasterProblem(n_v, m, DEV)
    xs = torch.empty(h.n_beamlets, dtype=torch.float32, device=DEV)
    col = torch.empty(n_v, dtype=torch.float32, device=DEV)
    DA = np.empty((n_v, m), dtype=np.float64)
    for k in range(m):
        vm.vmat_aperture_dose(h, (k * n_a) // m, L, R, xs, col)
        mp.add_aperture(col, 0.0, 0.0, 50.0)
        DA[:, k] = col.cpu().numpy()
    h.close()
    A = dict(sid=ph.voxel_struct.numpy(), T=ph.struct_T.numpy(), wo=ph.struct_w_over.numpy(), wu=ph.struct_w_under.numpy())
    obj = obj_to_device(A, DEV)
    z = torch.empty(n_v, dtype=torch.float32, device=DEV)
    sol = mp.solve(obj, max_iter=12, eps_F=0.0, eps_y=0.0, z=z)
    Fh, dh = mp.history()
    rows = vm.mp_pass_geometry(m)["rows_per_grid_step"]
    reached = int((DA != 0).any(axis=1).sum())
    print(f"\n[mp cfg3] {reached} of {n_v} voxels reached = {reached / rows:.1f} grid steps of {rows} rows")
    assert mp.n_reached_voxels == reached and reached >= 3.3 * rows
    sid = A["sid"]
    ref = omp.solve(DA, np.zeros(m), np.zeros(m), np.full(m, 50.0), A["T"][sid].astype(np.float64),
                    A["wo"][sid].astype(np.float64), A["wu"][sid].astype(np.float64), max_iter=12, eps_F=0.0, eps_y=0.0)
    _check(ref, sol, z.cpu().numpy(), Fh.numpy(), dh.numpy())
    assert ref.n_iter == 12 and ref.F < 0.5 * ref.F_hist[0]
    mp.close()


def test_unaligned_structure_ids(vm):
    """voxel_struct at an address that is not a multiple of 16 (a view one byte into a buffer): the kernel's cp.async
    path for the structure ids needs aligned blocks and must fall back, with the same result."""
    rng = np.random.default_rng(123)
    n_v, m = 20011, 70
    DA, sid, T, wo, wu = _random_mp(rng, n_v, m)
    lo, hi, y0 = np.zeros(m), np.full(m, 40.0), rng.uniform(0.0, 1.0, m)
    ref, sol, z, Fh, dh, mp, obj = _solve_both(vm, DA, sid, T, wo, wu, y0, lo, hi, max_iter=8, eps_F=0.0, eps_y=0.0)
    buf = torch.zeros(n_v + 1, dtype=torch.uint8, device=DEV)
    buf[1:] = obj.voxel_struct
    view = buf[1:]
    assert view.data_ptr() % 16 != 0 and view.is_contiguous()
    mp.set_fluence(torch.from_numpy(y0))
    z2 = torch.empty(n_v, dtype=torch.float32, device=DEV)
    sol2 = mp.solve(vm.Objective(view, obj.T, obj.w_over, obj.w_under), max_iter=8, eps_F=0.0, eps_y=0.0, z=z2)
    Fh2, dh2 = mp.history()
    assert np.array_equal(Fh2.numpy(), Fh) and np.array_equal(dh2.numpy(), dh) and np.array_equal(z2.cpu().numpy(), z)
    assert torch.equal(sol2.y, sol.y)
    _check(ref, sol2, z2.cpu().numpy(), Fh2.numpy(), dh2.numpy())
    mp.close()


def test_each_stopping_rule(vm):
    rng = np.random.default_rng(5)
    DA, sid, T, wo, wu = _random_mp(rng, 3000, 12)
    lo, hi, y0 = np.zeros(12), np.full(12, 1e6), np.zeros(12)
    for kw, reason in ((dict(max_iter=7, eps_F=0.0, eps_y=0.0), 4), (dict(max_iter=5000, eps_F=1e-5, eps_y=0.0), 2),
                       (dict(max_iter=5000, eps_F=0.0, eps_y=1e-4), 3), (dict(max_iter=0, eps_F=0.0, eps_y=0.0), 4)):
        ref, sol, z, Fh, dh, mp, _ = _solve_both(vm, DA, sid, T, wo, wu, y0, lo, hi, **kw)
        assert ref.reason == reason
        _check(ref, sol, z, Fh, dh, trace_rtol=1e-8)
        mp.close()
    # nothing to gain (no under-dose penalty anywhere, everything at its lower bound): stationary at iteration 0
    ref, sol, z, Fh, dh, mp, _ = _solve_both(vm, DA, sid, T, wo, wu * 0, y0, lo, hi, max_iter=10, eps_F=0.0, eps_y=0.0)
    assert ref.reason == 1 and ref.n_iter == 0
    _check(ref, sol, z, Fh, dh)
    mp.close()


def test_active_bounds_and_convergence_to_the_kkt_point(vm):
    """Upper and lower bounds bind (Eq. (9)/(10)); run to convergence and compare with the oracle's optimum."""
    rng = np.random.default_rng(9)
    DA, sid, T, wo, wu = _random_mp(rng, 4000, 10)
    lo = np.full(10, 0.5)
    hi = np.array([3.0, 3.0, 3.0, 1e3, 1e3, 1e3, 1e3, 1e3, 1e3, 1e3])
    y0 = np.full(10, 0.5)
    ref, sol, z, Fh, dh, mp, obj = _solve_both(vm, DA, sid, T, wo, wu, y0, lo, hi, max_iter=3000, eps_F=0.0, eps_y=1e-11)
    assert ref.reason in (1, 2, 3)
    y = sol.y.numpy()
    assert np.all(y >= lo) and np.all(y <= hi) and ((y <= lo) | (y >= hi)).sum() >= 1
    assert abs(sol.F - ref.F) <= 1e-9 * ref.F
    assert np.abs(y - ref.y).max() <= 1e-6 * np.abs(ref.y).max()
    assert_vec_close("z", z, ref.z)
    # warm start (L56: the next outer iteration starts from this solution): solving again stops at once
    sol2 = mp.solve(obj, max_iter=50, eps_F=0.0, eps_y=1e-9)
    assert sol2.n_iter <= 3 and abs(sol2.F - sol.F) <= 1e-9 * sol.F
    mp.close()


def test_determinism_capacity_and_reset(vm):
    """Two solves give identical bits; spare capacity (m_cap > m) does not change a bit; reset() starts over."""
    rng = np.random.default_rng(21)
    DA, sid, T, wo, wu = _random_mp(rng, 2222, 9)
    lo, hi, y0 = np.zeros(9), np.full(9, 100.0), np.full(9, 0.25)
    outs = []
    for cap in (9, 9, 200):
        ref, sol, z, Fh, dh, mp, obj = _solve_both(vm, DA, sid, T, wo, wu, y0, lo, hi, max_iter=25, eps_F=0.0,
                                                   eps_y=0.0, m_cap=cap)
        outs.append((sol.y.numpy().copy(), z.copy(), Fh.copy(), dh.copy()))
        if cap == 200:
            mp.reset()
            assert mp.n_apertures == 0
            mp.add_aperture(torch.from_numpy(np.ascontiguousarray(DA[:, 0])).to(DEV), 0.0, 0.0, 100.0)
            one = mp.solve(obj, max_iter=10, eps_F=0.0, eps_y=0.0)
            ref1 = omp.solve(DA[:, :1].astype(np.float64), [0.0], [0.0], [100.0], T[sid].astype(np.float64),
                             wo[sid].astype(np.float64), wu[sid].astype(np.float64), max_iter=10, eps_F=0.0, eps_y=0.0)
            assert abs(one.y[0].item() - ref1.y[0]) <= 1e-9 * max(1.0, abs(ref1.y[0]))
        mp.close()
    for a, b in zip(outs[0], outs[1]):
        assert np.array_equal(a, b)
    for a, b in zip(outs[0], outs[2]):
        assert np.array_equal(a, b)


def test_argument_errors(vm):
    mp = vm.MasterProblem(10, 2, DEV)
    obj = vm.Objective(torch.zeros(10, dtype=torch.uint8, device=DEV), torch.ones(1, device=DEV),
                       torch.ones(1, device=DEV), torch.ones(1, device=DEV))
    with pytest.raises(vm.VmatError, match="no aperture"):
        mp.solve(obj)
    col = torch.ones(10, device=DEV)
    with pytest.raises(vm.VmatError, match="y_lo > y_hi"):
        mp.add_aperture(col, 0.0, 2.0, 1.0)
    for _ in range(8):                                       # capacity is rounded up to a multiple of 8
        mp.add_aperture(col, 0.0, 0.0, 1.0)
    with pytest.raises(vm.VmatError, match="full"):
        mp.add_aperture(col, 0.0, 0.0, 1.0)
    mp.close()
    with pytest.raises(vm.VmatError):
        vm.MasterProblem(10, 385, DEV)


def _compare_plans(A, plan, ref, h):
    """GPU plan against the oracle's: same control points in the same order, same openings, fluence rates / dose /
    objective within the FP32 tolerances (the GPU's master problem runs on FP32 aperture dose vectors, the
    oracle's on FP64 ones, so the iteration counts of the master problems may differ)."""
    assert plan.stop == ref.stop
    assert plan.angles.tolist() == ref.angles
    assert np.array_equal(plan.L.cpu().numpy(), ref.L) and np.array_equal(plan.R.cpu().numpy(), ref.R)
    assert plan.y.numel() == ref.y.size
    if ref.y.size:
        assert np.abs(plan.y.numpy() - ref.y).max() <= 1e-4 * max(1.0, np.abs(ref.y).max())
    assert np.allclose(plan.F_hist.numpy(), np.array(ref.F_hist), rtol=1e-5, atol=0.0)
    assert np.allclose(plan.aperture_price.numpy(), np.array(ref.aperture_price), rtol=1e-5, atol=0.0)
    assert_vec_close("z", plan.z.cpu().numpy(), ref.z)


def test_column_generation_on_config0(vm, cfg0):
    """The paper's loop (L56) on the tiny phantom, every step on the GPU (vmat_column_generation), against the
    oracle's loop, which runs on its own in FP64 from the COO triplets and never sees a GPU value."""
    from oracle import column_generation as ocg
    A = as_np(cfg0)
    h = ddc_from_arrays(A, DEV)
    obj = obj_to_device(A, DEV)
    n_a = len(A["aro"]) - 1
    mp = vm.MasterProblem(A["n_v"], n_a, DEV)
    for cap in (n_a, 3, 0):
        plan = vm.vmat_column_generation(h, mp, obj, cap, 0.0, 50.0)
        ref = ocg.run(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], A["sid"], A["T"], A["wo"], A["wu"], A["lco"],
                      A["aro"], max_apertures=cap, y_lo=0.0, y_hi=50.0)
        _compare_plans(A, plan, ref, h)
        assert mp.n_apertures == len(ref.angles)
        if cap == n_a:
            assert len(ref.angles) >= 3 and ref.F_hist[-1] < 0.01 * ref.F_hist[0]      # the plan covers the target
            assert vm.last_launch_count() > 10 * len(ref.angles)                       # every step ran on the device
    # tight upper bounds on the fluence rates: more apertures are needed and the bounds bind
    plan = vm.vmat_column_generation(h, mp, obj, n_a, 0.0, 6.0)
    ref = ocg.run(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], A["sid"], A["T"], A["wo"], A["wu"], A["lco"],
                  A["aro"], max_apertures=n_a, y_lo=0.0, y_hi=6.0)
    _compare_plans(A, plan, ref, h)
    assert (ref.y >= 6.0).any()
    mp.close()
    h.close()


def test_column_generation_on_config1_coarsened(vm):
    """The loop on the H&N-like phantom of config 1 coarsened by 3.2 (1.5e7 nnz, 180 control points): the first
    apertures against the oracle's loop (ragged leaf rows, thousands of voxels per beamlet)."""
    from oracle import column_generation as ocg
    ph = synth.generate(synth.config_spec(1, 3.2), device=DEV)
    A = as_np(ph)
    h = vm.vmat_ddc_create(ph.n_voxels, ph.n_beamlets, ph.coo_voxel, ph.coo_beamlet, ph.coo_val,
                           ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset, device=DEV)
    obj = obj_to_device(A, DEV)
    mp = vm.MasterProblem(A["n_v"], 8, DEV)
    plan = vm.vmat_column_generation(h, mp, obj, 5, 0.0, 100.0, mp_max_iter=500)
    ref = ocg.run(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], A["sid"], A["T"], A["wo"], A["wu"], A["lco"],
                  A["aro"], max_apertures=5, y_lo=0.0, y_hi=100.0, mp_max_iter=500)
    print(f"\n[cfg1/3.2] control points {ref.angles}, F {ref.F_hist[0]:.4e} -> {ref.F_hist[-1]:.4e}, "
          f"MP iterations {ref.mp_iters} (GPU {plan.mp_iters.tolist()})")
    _compare_plans(A, plan, ref, h)
    assert len(ref.angles) == 5 and ref.F_hist[-1] < 0.5 * ref.F_hist[0]
    mp.close()
    h.close()


def test_only_reached_voxels_are_visited(vm):
    """70 % of the voxels are reached by no aperture (all-zero rows of DA), among them under-dosed target voxels whose
    constant terms of Eq. (1) must still be in F; the count of reached voxels follows the apertures, also after a
    reset and after adding an aperture that reaches new voxels."""
    rng = np.random.default_rng(77)
    n_v, m = 6000, 40
    DA, sid, T, wo, wu = _random_mp(rng, n_v, m)
    dead = rng.random(n_v) < 0.7
    DA[dead] = 0.0
    reached = int((DA != 0).any(axis=1).sum())
    assert (wu[sid][dead] > 0).any()
    lo, hi = np.zeros(m), np.full(m, 40.0)
    y0 = rng.uniform(0.0, 1.0, m)
    ref, sol, z, Fh, dh, mp, obj = _solve_both(vm, DA, sid, T, wo, wu, y0, lo, hi, max_iter=15, eps_F=0.0, eps_y=0.0)
    _check(ref, sol, z, Fh, dh)
    assert mp.n_reached_voxels == reached and (z[dead] == 0).all()
    const = float((wu[sid][dead].astype(np.float64) * T[sid][dead].astype(np.float64) ** 2).sum())
    assert const > 0.1 * ref.F                                                  # the constant part matters here
    # one more aperture that reaches every voxel
    col = np.full(n_v, 0.25, np.float32)
    mp2_DA = np.concatenate([DA, col[:, None]], axis=1)
    mp.close()
    ref2, sol2, z2, Fh2, dh2, mp2, _ = _solve_both(vm, mp2_DA, sid, T, wo, wu, np.append(y0, 0.0), np.append(lo, 0.0),
                                                   np.append(hi, 40.0), max_iter=15, eps_F=0.0, eps_y=0.0)
    _check(ref2, sol2, z2, Fh2, dh2)
    assert mp2.n_reached_voxels == n_v
    # reset forgets the reached voxels
    mp2.reset()
    mp2.add_aperture(torch.from_numpy(np.ascontiguousarray(DA[:, 0])).to(DEV), 1.0, 0.0, 40.0)
    mp2.solve(obj, max_iter=3, eps_F=0.0, eps_y=0.0)
    assert mp2.n_reached_voxels == int((DA[:, 0] != 0).sum())
    mp2.close()
