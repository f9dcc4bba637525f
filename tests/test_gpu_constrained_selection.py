"""GPU parity of the constrained aperture selection (NEXT-3; vmat_select_apertures_constrained) against the oracle's
O6, bit for bit on the same FP32 price vector: hand-worked control points, random tiny control points with windows,
config 0 / coarsened config 1 with their real prices (fused protocol: the oracle is applied to the GPU's own p),
and the full-size config 3 on sampled control points plus properties that hold for every control point."""
import numpy as np
import pytest
import torch

import oracle
import synth
from conftest import as_np
from helpers import ddc_from_arrays, obj_to_device
from test_constrained_selection_oracle import parse_cases, satisfies_interdigitation

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def vm():
    import paper_1503_01721_b200 as vm
    vm.load_library()
    return vm


def selection_handle(vm, aro, lco, pos0):
    """A handle that holds only the offset tables (nnz = 0 is legal): enough for the selection calls."""
    aro, lco = np.asarray(aro, np.int32), np.asarray(lco, np.int32)
    e = torch.zeros(0, dtype=torch.int32, device=DEV)
    h = vm.vmat_ddc_create(1, int(lco[-1]), e, e, torch.zeros(0, dtype=torch.float32, device=DEV),
                           torch.from_numpy(lco[aro]), torch.from_numpy(aro), torch.from_numpy(lco), device=DEV)
    vm.vmat_ddc_set_leaf_geometry(h, torch.from_numpy(np.asarray(pos0, np.int32)))
    return h


def gpu_select(vm, h, p, interdig, mask=None, W=None):
    dev_i = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a, np.int32)).to(DEV)
    out = h.alloc_outputs()
    pt = p if torch.is_tensor(p) else torch.from_numpy(np.ascontiguousarray(p, np.float32)).to(DEV)
    m = None if mask is None else torch.from_numpy(np.ascontiguousarray(mask, np.uint8)).to(DEV)
    W = W or [None] * 4
    vm.vmat_select_apertures_constrained(h, pt, m, interdig, out.L, out.R, out.row_price, out.angle_price,
                                         out.best_angle, dev_i(W[0]), dev_i(W[1]), dev_i(W[2]), dev_i(W[3]))
    torch.cuda.synchronize()
    return (out.L.cpu().numpy(), out.R.cpu().numpy(), out.row_price.cpu().numpy(), out.angle_price.cpu().numpy(),
            int(out.best_angle.item()))


def assert_same(got, ref):
    for name, g, r in zip(("L", "R", "row_price", "angle_price"), got[:4], ref[:4]):
        assert np.array_equal(g, r), name                          # FP64 values: same operations in the same order
    assert got[4] == ref[4]


def test_hand_worked_control_points(vm):
    for interdig, pos0, rows, W, exp, price in parse_cases():
        lco = np.concatenate([[0], np.cumsum([len(r) for r in rows])])
        h = selection_handle(vm, [0, len(rows)], lco, pos0)
        p = np.array([v for r in rows for v in r], np.float32)
        L, R, rp, ap, best = gpu_select(vm, h, p, interdig, W=W)
        assert [[int(a), int(b)] for a, b in zip(L, R)] == exp
        assert ap[0] == price and best == (0 if price < 0 else -1)
        h.close()


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_random_control_points_with_windows(vm, seed):
    """Many small control points in one call: ragged rows, empty rows, shifted rows, windows (some infeasible), an
    occupied control point; integer and real prices."""
    rng = np.random.default_rng(1503 + seed)
    n_a = 300
    rows_per = rng.integers(0, 7, n_a)
    lens = [rng.integers(0, 9, k) for k in rows_per]
    aro = np.concatenate([[0], np.cumsum(rows_per)]).astype(np.int32)
    all_lens = np.concatenate(lens) if n_a else np.zeros(0, np.int64)
    lco = np.concatenate([[0], np.cumsum(all_lens)]).astype(np.int32)
    n_rows, n_b = int(aro[-1]), int(lco[-1])
    pos0 = rng.integers(0, 6, n_rows).astype(np.int32)
    p = (rng.integers(-4, 5, n_b) if seed == 0 else rng.normal(size=n_b) * 10.0).astype(np.float32)
    mask = np.zeros(n_a, np.uint8); mask[7] = 1
    lo = rng.integers(-2, 5, size=(2, n_rows))
    W = [lo[0], lo[0] + rng.integers(0, 9, n_rows), lo[1], lo[1] + rng.integers(0, 9, n_rows)]
    W = [w.astype(np.int32) for w in W]
    h = selection_handle(vm, aro, lco, pos0)
    n_inf = 0
    for interdig in (True, False):
        for win in (None, W, [W[0], None, None, W[3]]):
            kw = {} if win is None else {k: v for k, v in zip(("L_lo", "L_hi", "R_lo", "R_hi"), win) if v is not None}
            ref = oracle.select_constrained(p, aro, lco, pos0, interdig, angle_mask=mask, **kw)
            got = gpu_select(vm, h, p, interdig, mask, win)
            assert_same(got, ref)
            n_inf += int(np.isinf(ref[3]).sum())
    assert n_inf > 6                                               # infeasible control points were exercised
    h.close()


@pytest.mark.parametrize("scale", [1.0, 14.0, 16.0])
def test_config0_real_prices(vm, cfg0, scale):
    A = as_np(cfg0)
    h = ddc_from_arrays(A, DEV)
    vm.vmat_ddc_set_leaf_geometry(h, cfg0.leafrow_pos0)
    out = h.alloc_outputs()
    x = synth.draw_x(A["n_b"], 0, device=DEV, scale=scale)
    vm.vmat_price_eval(h, x, obj_to_device(A, DEV), out)
    p_gpu = out.p.cpu().numpy()
    u0 = cfg0.leafrow_pos0.numpy()
    for interdig in (True, False):
        ref = oracle.select_constrained(p_gpu, A["aro"], A["lco"], u0, interdig)     # fused protocol (C6 (ii))
        got = gpu_select(vm, h, out.p, interdig)
        assert_same(got, ref)
        if interdig:
            assert satisfies_interdigitation(got[0], got[1], u0, A["aro"])
            assert (got[3] >= out.angle_price.cpu().numpy()).all()
        else:                                                      # no constraint: the plain selection's apertures
            opened = out.R.cpu().numpy() > out.L.cpu().numpy()
            assert np.array_equal(got[0][opened], out.L.cpu().numpy()[opened])
            assert np.array_equal(got[2], out.row_price.cpu().numpy())
            assert np.array_equal(got[3], out.angle_price.cpu().numpy()) and got[4] == int(out.best_angle.item())
    h.close()


def test_config1_coarsened_real_prices(vm):
    """Config 1's geometry (ragged fields, 40 leaf rows, 180 control points) on a coarsened grid."""
    ph = synth.generate(synth.config_spec(1, scale=3.0), device=DEV)
    A = as_np(ph)
    h = ddc_from_arrays(A, DEV)
    vm.vmat_ddc_set_leaf_geometry(h, ph.leafrow_pos0)
    out = h.alloc_outputs()
    vm.vmat_price_eval(h, synth.draw_x(A["n_b"], 3, device=DEV, scale=0.55), obj_to_device(A, DEV), out)
    p_gpu = out.p.cpu().numpy()
    assert (p_gpu > 0).any() and (p_gpu < 0).any()                  # mixed signs: rows open partially
    u0 = ph.leafrow_pos0.numpy()
    rng = np.random.default_rng(5)
    n_rows = A["lco"].size - 1
    W = [rng.integers(-1, 3, n_rows).astype(np.int32), None, None, None]
    W[1] = (W[0] + rng.integers(2, 12, n_rows)).astype(np.int32)
    for interdig, win in ((True, None), (False, None), (True, W)):
        kw = {} if win is None else dict(L_lo=win[0], L_hi=win[1])
        ref = oracle.select_constrained(p_gpu, A["aro"], A["lco"], u0, interdig, **kw)
        assert_same(gpu_select(vm, h, out.p, interdig, W=win), ref)
    h.close()


def test_config3_full_size_fields_sampled(vm):
    """The field geometry of config 3 at full size (360 control points, 128-160 leaf rows of up to 130 beamlets: the
    largest tables the kernel takes) with a seeded smooth mixed-sign price vector: the oracle on sampled control
    points (it needs ~states^2 per row pair), properties on all of them."""
    from synth import phantom as P
    spec = synth.config_spec(3)
    cmins, cmaxs, aco, aro, lco = P._fields(spec)
    pos0 = torch.cat([torch.where(cx >= cn, cn, torch.zeros_like(cn)) for cn, cx in zip(cmins, cmaxs)]).numpy().astype(np.int32)
    aro, lco = aro.numpy().astype(np.int32), lco.numpy().astype(np.int32)
    n_b, n_a = int(lco[-1]), aro.size - 1
    j = np.arange(n_b, dtype=np.float64)
    u = synth.draw_x(n_b, 77).numpy().astype(np.float64)
    p = (np.sin(j * 0.37) + 0.6 * np.sin(j * 0.011) + (u - 0.5) - 0.1).astype(np.float32)
    h = selection_handle(vm, aro, lco, pos0)
    got = gpu_select(vm, h, p, True)
    free = gpu_select(vm, h, p, False)
    assert satisfies_interdigitation(got[0], got[1], pos0, aro, lco)
    assert (got[3] >= free[3]).all() and (got[3] > free[3]).any()   # the constraint binds somewhere
    lens = np.diff(lco)
    opened = got[1] > got[0]
    assert (got[0][opened] >= 0).all() and (got[1][opened] <= lens[opened]).all()
    Lf, Rf, rpf = oracle.select_rows(p, lco)                        # the unconstrained optimum is O4 / O5
    assert np.array_equal(free[2], rpf) and np.array_equal(free[0][Rf > Lf], Lf[Rf > Lf])
    sample = list(range(3, n_a, 8))                                 # 45 control points over both arcs
    mask = np.ones(n_a, np.uint8); mask[sample] = 0
    ref = oracle.select_constrained(p, aro, lco, pos0, True, angle_mask=mask)
    for k in sample:
        sl = slice(aro[k], aro[k + 1])
        assert np.array_equal(got[0][sl], ref[0][sl]) and np.array_equal(got[1][sl], ref[1][sl])
        assert np.array_equal(got[2][sl], ref[2][sl]) and got[3][k] == ref[3][k]
    h.close()


def test_config3_full_size_fields_all_control_points(vm):
    """As above, but O6 on ALL 360 control points of config 3 (about a minute of oracle time), with interdigitation
    and - second pass - with interdigitation plus seeded leaf windows."""
    import time
    from synth import phantom as P
    spec = synth.config_spec(3)
    cmins, cmaxs, aco, aro, lco = P._fields(spec)
    pos0 = torch.cat([torch.where(cx >= cn, cn, torch.zeros_like(cn)) for cn, cx in zip(cmins, cmaxs)]).numpy().astype(np.int32)
    aro, lco = aro.numpy().astype(np.int32), lco.numpy().astype(np.int32)
    n_b, n_rows = int(lco[-1]), lco.size - 1
    j = np.arange(n_b, dtype=np.float64)
    u = synth.draw_x(n_b, 78).numpy().astype(np.float64)
    p = (np.sin(j * 0.41) + 0.5 * np.sin(j * 0.013) + (u - 0.5) - 0.15).astype(np.float32)
    h = selection_handle(vm, aro, lco, pos0)
    rng = np.random.default_rng(11)
    # windows around a feasible aperture (the interdigitation-constrained optimum of a second price vector), a few
    # positions wide: they bind for most rows but leave every control point feasible
    p2 = (np.sin(j * 0.29 + 1.0) + 0.5 * np.sin(j * 0.017) + (u - 0.5) - 0.2).astype(np.float32)
    L2, R2 = gpu_select(vm, h, p2, True)[:2]
    W = [(L2 - rng.integers(0, 5, n_rows)).astype(np.int32), (L2 + rng.integers(0, 5, n_rows)).astype(np.int32),
         (R2 - rng.integers(0, 5, n_rows)).astype(np.int32), (R2 + rng.integers(0, 5, n_rows)).astype(np.int32)]
    for win in (None, W):
        t0 = time.time()
        kw = {} if win is None else dict(L_lo=win[0], L_hi=win[1], R_lo=win[2], R_hi=win[3])
        ref = oracle.select_constrained(p, aro, lco, pos0, True, **kw)
        got = gpu_select(vm, h, p, True, W=win)
        assert_same(got, ref)
        print(f"\n[cfg3 fields, all control points{' + windows' if win else ''}] oracle {time.time() - t0:.0f} s, "
              f"{int((ref[1] > ref[0]).sum())} open rows, {int(np.isinf(ref[3]).sum())} infeasible control points, "
              f"best {ref[4]}")
        assert (ref[1] > ref[0]).sum() > 1000 and not np.isinf(ref[3]).any()
    h.close()


def test_errors(vm):
    h = selection_handle(vm, [0, 1], [0, 3], [0])
    out = h.alloc_outputs()
    h2 = vm.vmat_ddc_create(1, 3, torch.zeros(0, dtype=torch.int32, device=DEV), torch.zeros(0, dtype=torch.int32, device=DEV),
                            torch.zeros(0, dtype=torch.float32, device=DEV), torch.tensor([0, 3]), torch.tensor([0, 1]),
                            torch.tensor([0, 3]), device=DEV)
    with pytest.raises(vm.VmatError):                               # geometry was never set
        vm.vmat_select_apertures_constrained(h2, torch.zeros(3, device=DEV), None, True, out.L, out.R, out.row_price,
                                             out.angle_price, out.best_angle)
    h3 = selection_handle(vm, [0, 2], [0, 3, 6], [0, 0])
    with pytest.raises(vm.VmatError):                               # a field range beyond 255 positions
        vm.vmat_ddc_set_leaf_geometry(h3, torch.tensor([0, 400], dtype=torch.int32))
    with pytest.raises(vm.VmatError):                               # 256 positions: one more than the packing holds
        vm.vmat_ddc_set_leaf_geometry(h3, torch.tensor([0, 252], dtype=torch.int32))
    for x in (h, h2, h3):
        x.close()


def test_field_range_at_the_limit_and_two_handles(vm):
    """A control point whose field range holds exactly 255 leaf positions (the most the 8-bit packing takes; the pair
    (255, 255) is the kernel's 'no predecessor' mark), against O6; and a SECOND handle with short rows created and
    used in between: the first one's launches must not be affected (the shared-memory attribute of the kernel
    belongs to the device, not to a handle)."""
    rng = np.random.default_rng(255)
    n0, n1 = 100, 120
    lco = np.array([0, n0, n0 + n1, n0 + n1 + 90], np.int32)
    pos0 = np.array([0, 134, 60], np.int32)                        # max pos0 + n = 254 -> 255 positions
    aro = np.array([0, 3], np.int32)
    h = selection_handle(vm, aro, lco, pos0)
    p = rng.integers(-3, 4, int(lco[-1])).astype(np.float32)
    small = selection_handle(vm, [0, 2], [0, 4, 8], [0, 1])        # lowers nothing
    ps = rng.integers(-3, 4, 8).astype(np.float32)
    assert_same(gpu_select(vm, small, ps, True), oracle.select_constrained(ps, [0, 2], [0, 4, 8], [0, 1], True))
    for interdig in (True, False):
        assert_same(gpu_select(vm, h, p, interdig), oracle.select_constrained(p, aro, lco, pos0, interdig))
    W = [np.array([0, 0, 0], np.int32), np.array([254, 254, 254], np.int32), np.array([0, 0, 0], np.int32),
         np.array([254, 254, 254], np.int32)]                      # windows over the whole range: closed pairs park at 254
    assert_same(gpu_select(vm, h, p, True, W=W), oracle.select_constrained(p, aro, lco, pos0, True, L_lo=W[0], L_hi=W[1],
                                                                          R_lo=W[2], R_hi=W[3]))
    p_pos = np.abs(p) + 1.0                                         # nothing to gain: every row closed somewhere feasible
    assert_same(gpu_select(vm, h, p_pos, True), oracle.select_constrained(p_pos, aro, lco, pos0, True))
    small.close()
    h.close()


# ---------------------------------------------------------------- leaf-travel windows and the constrained loop
def test_leaf_windows_against_the_oracle(vm):
    """vmat_leaf_windows against oracle.column_generation.leaf_windows, integer for integer: random occupied sets and
    openings on two arcs with ragged, partly empty rows."""
    from oracle import column_generation as ocg
    rng = np.random.default_rng(66)
    arcs = np.array([0, 23, 40], np.int32)
    rows_of = [5] * 23 + [7] * 17
    aro = np.concatenate([[0], np.cumsum(rows_of)]).astype(np.int32)
    n_rows = int(aro[-1])
    lens = rng.integers(0, 9, n_rows)
    lco = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    pos0 = rng.integers(0, 5, n_rows).astype(np.int32)
    h = selection_handle(vm, aro, lco, pos0)
    for trial, travel in enumerate((0, 1, 3, 50)):
        mask = (rng.random(40) < (0.1, 0.3, 0.6, 1.0)[trial]).astype(np.uint8)
        L = rng.integers(-2, 8, n_rows).astype(np.int32)
        R = (L + rng.integers(0, 6, n_rows)).astype(np.int32)
        ref = ocg.leaf_windows(mask, L, R, lco, aro, pos0, arcs, travel)
        dv = lambda a: torch.from_numpy(a).to(DEV)
        W = [torch.empty(n_rows, dtype=torch.int32, device=DEV) for _ in range(4)]
        vm.vmat_leaf_windows(h, dv(mask), dv(L), dv(R), torch.from_numpy(arcs), travel, *W)
        for got, want in zip(W, ref):
            assert np.array_equal(got.cpu().numpy(), want)
    with pytest.raises(vm.VmatError):                               # an arc whose control points differ in leaf rows
        vm.vmat_leaf_windows(h, dv(mask), dv(L), dv(R), torch.tensor([0, 30, 40]), 1, *W)
    h.close()


def _compare_constrained_plans(plan, ref):
    from helpers import assert_vec_close
    assert plan.stop == ref.stop
    assert plan.angles.tolist() == ref.angles
    assert np.array_equal(plan.L.cpu().numpy(), ref.L) and np.array_equal(plan.R.cpu().numpy(), ref.R)
    assert np.abs(plan.y.numpy() - ref.y).max() <= 1e-4 * max(1.0, np.abs(ref.y).max())
    assert np.allclose(plan.F_hist.numpy(), np.array(ref.F_hist), rtol=1e-5, atol=0.0)
    assert np.allclose(plan.aperture_price.numpy(), np.array(ref.aperture_price), rtol=1e-5, atol=0.0)
    assert_vec_close("z", plan.z.cpu().numpy(), ref.z)


@pytest.mark.parametrize("interdig,travel", [(True, 1), (True, -1), (False, 2)])
def test_constrained_column_generation_on_config0(vm, cfg0, interdig, travel):
    """The paper's loop (L56) with the pricing problem under hardware constraints, every step on the GPU, against the
    oracle's constrained loop (same control points in the same order, same leaf positions incl. parked closed rows)."""
    from oracle import column_generation as ocg
    A = as_np(cfg0)
    h = ddc_from_arrays(A, DEV)
    vm.vmat_ddc_set_leaf_geometry(h, cfg0.leafrow_pos0)
    obj = obj_to_device(A, DEV)
    n_a = len(A["aro"]) - 1
    mp = vm.MasterProblem(A["n_v"], n_a, DEV)
    plan = vm.vmat_column_generation(h, mp, obj, n_a, 0.0, 50.0, interdigitation=interdig, max_leaf_travel=travel,
                                     arc_angle_offset=cfg0.arc_angle_offset)
    ref = ocg.run(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], A["sid"], A["T"], A["wo"], A["wu"], A["lco"],
                  A["aro"], max_apertures=n_a, y_lo=0.0, y_hi=50.0, interdigitation=interdig, max_leaf_travel=travel,
                  leafrow_pos0=cfg0.leafrow_pos0.numpy(), arc_angle_offset=cfg0.arc_angle_offset.numpy())
    _compare_constrained_plans(plan, ref)
    assert len(ref.angles) >= 2
    mp.close()
    h.close()


def test_constrained_column_generation_on_config1_coarsened(vm):
    from oracle import column_generation as ocg
    ph = synth.generate(synth.config_spec(1, 3.2), device=DEV)
    A = as_np(ph)
    h = vm.vmat_ddc_create(ph.n_voxels, ph.n_beamlets, ph.coo_voxel, ph.coo_beamlet, ph.coo_val,
                           ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset, device=DEV)
    vm.vmat_ddc_set_leaf_geometry(h, ph.leafrow_pos0)
    obj = obj_to_device(A, DEV)
    mp = vm.MasterProblem(A["n_v"], 8, DEV)
    kw = dict(interdigitation=True, max_leaf_travel=1)
    plan = vm.vmat_column_generation(h, mp, obj, 5, 0.0, 100.0, mp_max_iter=500, arc_angle_offset=ph.arc_angle_offset, **kw)
    ref = ocg.run(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], A["sid"], A["T"], A["wo"], A["wu"], A["lco"],
                  A["aro"], max_apertures=5, y_lo=0.0, y_hi=100.0, mp_max_iter=500, leafrow_pos0=ph.leafrow_pos0.numpy(),
                  arc_angle_offset=ph.arc_angle_offset.numpy(), **kw)
    _compare_constrained_plans(plan, ref)
    assert len(ref.angles) == 5
    mp.close()
    h.close()


@pytest.mark.parametrize("constrained", [False, True])
def test_column_generation_on_config1_full(vm, constrained):
    """The loop (free, and under interdigitation + leaf travel) on the FULL config 1 (3.3e8 nnz, 180 control points, 434 688
    voxels): the first three apertures against the oracle's loop."""
    import time
    from oracle import column_generation as ocg
    ph = synth.generate(synth.config_spec(1), device=DEV)
    A = as_np(ph)
    h = vm.vmat_ddc_create(ph.n_voxels, ph.n_beamlets, ph.coo_voxel, ph.coo_beamlet, ph.coo_val,
                           ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset, device=DEV)
    ph.coo_voxel = ph.coo_beamlet = ph.coo_val = None
    vm.vmat_ddc_set_leaf_geometry(h, ph.leafrow_pos0)
    obj = obj_to_device(A, DEV)
    mp = vm.MasterProblem(A["n_v"], 8, DEV)
    kw = dict(interdigitation=True, max_leaf_travel=2) if constrained else {}
    okw = dict(leafrow_pos0=ph.leafrow_pos0.numpy(), arc_angle_offset=ph.arc_angle_offset.numpy(), **kw) if constrained else {}
    plan = vm.vmat_column_generation(h, mp, obj, 3, 0.0, 100.0, mp_max_iter=300,
                                     arc_angle_offset=ph.arc_angle_offset if constrained else None, **kw)
    t0 = time.time()
    ref = ocg.run(A["vox"], A["beam"], A["val"], A["n_v"], A["n_b"], A["sid"], A["T"], A["wo"], A["wu"], A["lco"],
                  A["aro"], max_apertures=3, y_lo=0.0, y_hi=100.0, mp_max_iter=300, **okw)
    print(f"\n[cfg1 full, {'constrained' if constrained else 'free'}] control points {ref.angles}, F {ref.F_hist[0]:.4e} -> "
          f"{ref.F_hist[-1]:.4e}, MP iterations {ref.mp_iters} (GPU {plan.mp_iters.tolist()}), oracle {time.time() - t0:.0f} s")
    if constrained:
        _compare_constrained_plans(plan, ref)
    else:
        from test_gpu_master_problem import _compare_plans
        _compare_plans(A, plan, ref, h)
    assert len(ref.angles) == 3 and ref.F_hist[-1] < ref.F_hist[0]
    mp.close()
    h.close()
