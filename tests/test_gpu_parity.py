"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json's: rel L2 <= 1e-5 and |delta| <= 1e-4 max|ref|
for FP32 vectors and F; leaf positions bit-exact under the protocol of DESIGN.md reading C6."""
import numpy as np
import pytest
import torch

import oracle
import synth
from conftest import as_np
from helpers import (assert_vec_close, check_selection_protocol, ddc_from_arrays, obj_to_device, oracle_eval,
                     REL_L2)

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def vm():
    import paper_1503_01721_b200 as vm
    vm.load_library()
    return vm


@pytest.fixture(scope="module")
def A0(cfg0):
    return as_np(cfg0)


@pytest.fixture(scope="module")
def h0(vm, A0):
    h = ddc_from_arrays(A0, DEV)
    yield h
    h.close()


def _x(n_b, k, scale=1.0):
    return synth.draw_x(n_b, k, scale=scale)


def _eval_gpu(vm, h, A, x, mask=None):
    obj = obj_to_device(A, DEV)
    out = h.alloc_outputs()
    m = None if mask is None else torch.from_numpy(np.asarray(mask, np.uint8)).to(DEV)
    vm.vmat_price_eval(h, x.to(DEV), obj, out, m)
    torch.cuda.synchronize()
    return out


def _check_eval(A, out, ev, mask=None):
    assert_vec_close("d", out.d.cpu().numpy(), ev.d)
    assert_vec_close("g", out.g.cpu().numpy(), ev.g)
    assert_vec_close("p", out.p.cpu().numpy(), ev.p)
    assert abs(out.F.item() - ev.F) <= REL_L2 * abs(ev.F) + 1e-300
    return check_selection_protocol(A, out, ev, mask)


# ------------------------------------------------------------------ A0 ingest / layout
def test_layouts_round_trip_config0(vm, A0, h0):
    """Both layouts expand back to exactly the input triplets; rows are in canonical order (P7, P9)."""
    key_in = np.sort(A0["vox"].astype(np.int64) * A0["n_b"] + A0["beam"])
    order = np.lexsort((A0["beam"], A0["vox"]))
    for which, rows in ((0, A0["n_v"]), (1, A0["n_b"])):
        ptr, idx, val = [t.numpy() for t in h0.export_csr(which)]
        assert ptr[0] == 0 and ptr[-1] == A0["vox"].size and (np.diff(ptr) >= 0).all()
        row = np.repeat(np.arange(rows), np.diff(ptr))
        v, b = (row, idx) if which == 0 else (idx, row)
        assert np.array_equal(np.sort(v.astype(np.int64) * A0["n_b"] + b), key_in)
        inner = np.diff(idx.astype(np.int64))
        same_row = np.diff(row) == 0
        assert (inner[same_row] > 0).all()                       # strictly ascending secondary index
        if which == 0:
            assert np.array_equal(val, A0["val"][order])
    info = h0.info
    assert info["bytes_csr_d"] == 8 * info["nnz"] + 8 * (info["n_voxels"] + 1)       # 8 B/nnz
    assert info["bytes_csr_dt"] == 8 * info["nnz"] + 8 * (info["n_beamlets"] + 1)


@pytest.mark.parametrize("bits", [16, 32])
def test_index_encodings_unpack_to_the_same_csr_and_give_the_same_bits(vm, A0, h0, bits):
    """int32 indices (the paper's 8 B/nnz, Table 2) and u16 offsets + one base per 32 entries (6.125 B) hold
    the same entries in the same order: same canonical CSR, and - config 0 needs no early-closed group -
    bit-identical outputs."""
    h = ddc_from_arrays(A0, DEV, index_bits=bits)
    info = h.info
    assert info["index_bits_d"] == info["index_bits_dt"] == bits
    for lay, rows in (("d", "n_voxels"), ("dt", "n_beamlets")):
        P = info[f"padded_{lay}"]
        assert P % 32 == 0 and info["nnz"] <= P
        per_entry = 6 * P + 4 * (P // 32) if bits == 16 else 8 * P
        seg_table = 4 * (info["n_dose_blocks"] + 1) if lay == "d" else 0
        assert info[f"bytes_stream_{lay}"] == per_entry + 8 * (info[rows] + 1) + seg_table
    assert info["padded_dt"] - info["nnz"] <= 31 * info["n_beamlets"]                  # < one group of pads per row
    for w in (0, 1):
        for a, b in zip(h.export_csr(w), h0.export_csr(w)):
            assert torch.equal(a, b)
    x = _x(A0["n_b"], 27, 14.0)
    o1, o2 = _eval_gpu(vm, h, A0, x), _eval_gpu(vm, h0, A0, x)
    for f in ("d", "g", "F", "p", "L", "R", "row_price", "angle_price", "best_angle"):
        assert torch.equal(getattr(o1, f), getattr(o2, f)), f
    h.close()


def test_ingest_host_and_device_coo_and_shuffle_give_identical_layouts(vm, A0, h0):
    perm = np.random.default_rng(3).permutation(A0["vox"].size)
    B = dict(A0, vox=A0["vox"][perm], beam=A0["beam"][perm], val=A0["val"][perm])
    ref = [t.numpy() for w in (0, 1) for t in h0.export_csr(w)]
    for on_dev in (True, False):
        h = ddc_from_arrays(B, DEV, coo_on_device=on_dev)
        got = [t.numpy() for w in (0, 1) for t in h.export_csr(w)]
        for a, b in zip(ref, got):
            assert np.array_equal(a, b)
        h.close()


def test_ingest_rejects_bad_input(vm, A0):
    def create(vox, beam, val, n_v=A0["n_v"], n_b=A0["n_b"]):
        return ddc_from_arrays(dict(A0, vox=vox, beam=beam, val=val, n_v=n_v, n_b=n_b), DEV)
    vox, beam, val = A0["vox"].copy(), A0["beam"].copy(), A0["val"].copy()
    bad = vox.copy(); bad[17] = A0["n_v"]
    with pytest.raises(vm.VmatError) as e:
        create(bad, beam, val)
    assert e.value.status == -2
    bad = beam.copy(); bad[5] = -1
    with pytest.raises(vm.VmatError) as e:
        create(vox, bad, val)
    assert e.value.status == -2
    badv = val.copy(); badv[100] = np.nan
    with pytest.raises(vm.VmatError) as e:
        create(vox, beam, badv)
    assert e.value.status == -6
    with pytest.raises(vm.VmatError) as e:                       # duplicate (voxel, beamlet) pair (C14)
        create(np.append(vox, vox[7]), np.append(beam, beam[7]), np.append(val, val[7]))
    assert e.value.status == -3
    lco = A0["lco"].copy(); lco[3] = lco[2] - 1
    with pytest.raises(vm.VmatError) as e:
        ddc_from_arrays(dict(A0, lco=lco), DEV)
    assert e.value.status == -1


# ------------------------------------------------------------------ per-call parity, config 0
@pytest.mark.parametrize("scale", [1.0, 8.0, 14.0, 16.0, 20.0])
def test_each_call_alone_config0(vm, A0, h0, scale):
    """Every C-ABI call on its own, fed the oracle's (FP32-rounded) input of that step."""
    x = _x(A0["n_b"], 21, scale)
    ev = oracle_eval(A0, x.numpy())
    obj = obj_to_device(A0, DEV)
    out = h0.alloc_outputs()
    # A1
    vm.vmat_dose(h0, x.to(DEV), out.d)
    assert_vec_close("d", out.d.cpu().numpy(), ev.d)
    # A2 on the oracle's d rounded to FP32
    d32 = ev.d.astype(np.float32)
    F_ref, g_ref = oracle.objective_grad(d32.astype(np.float64), A0["sid"], A0["T"], A0["wo"], A0["wu"])
    vm.vmat_objective_grad(h0, torch.from_numpy(d32).to(DEV), obj, out.g, out.F)
    assert_vec_close("g", out.g.cpu().numpy(), g_ref)
    assert abs(out.F.item() - F_ref) <= REL_L2 * abs(F_ref)
    # A3 on the oracle's g rounded to FP32
    g32 = ev.g.astype(np.float32)
    p_ref = oracle.price(A0["vox"], A0["beam"], A0["val"], A0["n_b"], g32.astype(np.float64))
    vm.vmat_price(h0, torch.from_numpy(g32).to(DEV), out.p)
    assert_vec_close("p", out.p.cpu().numpy(), p_ref)
    # A4 + A5 on the oracle's p rounded to FP32: bit-exact (C6 (i))
    vm.vmat_select_apertures(h0, torch.from_numpy(ev.p_f32).to(DEV), None, out.L, out.R, out.row_price,
                             out.angle_price, out.best_angle)
    torch.cuda.synchronize()
    assert np.array_equal(out.L.cpu().numpy(), ev.L) and np.array_equal(out.R.cpu().numpy(), ev.R)
    assert np.array_equal(out.row_price.cpu().numpy(), ev.row_price)
    assert np.array_equal(out.angle_price.cpu().numpy(), ev.angle_price)
    assert int(out.best_angle.item()) == ev.best_angle


@pytest.mark.parametrize("scale", [0.0, 1.0, 8.0, 14.0, 16.0, 20.0])
def test_price_eval_fused_config0(vm, A0, h0, scale):
    x = _x(A0["n_b"], 22, scale)
    ev = oracle_eval(A0, x.numpy())
    out = _eval_gpu(vm, h0, A0, x)
    n_diff = _check_eval(A0, out, ev)
    assert n_diff == 0
    if scale == 0.0:                                   # the paper's first iteration (L56): closed form
        assert (out.d == 0).all() and int(out.best_angle.item()) == ev.best_angle >= 0


def test_angle_mask(vm, A0, h0):
    x = _x(A0["n_b"], 23, 14.0)
    mask = np.zeros(A0["aro"].size - 1, np.uint8)
    ev0 = oracle_eval(A0, x.numpy())
    mask[ev0.best_angle] = 1                              # occupy the best control point (C7)
    mask[0] = 1
    ev = oracle_eval(A0, x.numpy(), mask)
    out = _eval_gpu(vm, h0, A0, x, mask)
    _check_eval(A0, out, ev, mask)
    assert int(out.best_angle.item()) == ev.best_angle != ev0.best_angle
    assert torch.isinf(out.angle_price[0]) and out.angle_price[0] > 0
    # unfused call, same mask
    o2 = h0.alloc_outputs()
    vm.vmat_select_apertures(h0, out.p, torch.from_numpy(mask).to(DEV), o2.L, o2.R, o2.row_price, o2.angle_price,
                             o2.best_angle)
    for a, b in ((o2.L, out.L), (o2.R, out.R), (o2.row_price, out.row_price), (o2.angle_price, out.angle_price),
                 (o2.best_angle, out.best_angle)):
        assert torch.equal(a, b)


def test_determinism_and_shuffle_invariance(vm, A0, h0):
    """Two runs are bit-identical, and so is a handle built from shuffled triplets (P9)."""
    x = _x(A0["n_b"], 24, 14.0)
    o1 = _eval_gpu(vm, h0, A0, x)
    o2 = _eval_gpu(vm, h0, A0, x)
    perm = np.random.default_rng(5).permutation(A0["vox"].size)
    hB = ddc_from_arrays(dict(A0, vox=A0["vox"][perm], beam=A0["beam"][perm], val=A0["val"][perm]), DEV)
    o3 = _eval_gpu(vm, hB, A0, x)
    hB.close()
    for f in ("d", "g", "F", "p", "L", "R", "row_price", "angle_price", "best_angle"):
        assert torch.equal(getattr(o1, f), getattr(o2, f)), f
        assert torch.equal(getattr(o1, f), getattr(o3, f)), f


def test_host_buffer_call_matches_device_call(vm, A0, h0):
    x = _x(A0["n_b"], 25, 14.0)
    out = _eval_gpu(vm, h0, A0, x)
    obj = obj_to_device(A0, DEV)
    xh = x.pin_memory()
    F = torch.empty(1, dtype=torch.float64).pin_memory()
    L = torch.empty(h0.n_leaf_rows, dtype=torch.int32).pin_memory()
    R = torch.empty(h0.n_leaf_rows, dtype=torch.int32).pin_memory()
    rp = torch.empty(h0.n_leaf_rows, dtype=torch.float64).pin_memory()
    ap = torch.empty(h0.n_angles, dtype=torch.float64).pin_memory()
    best = torch.empty(1, dtype=torch.int32).pin_memory()
    vm.vmat_price_eval_host(h0, xh, obj, F, L, R, rp, ap, best)
    assert F.item() == out.F.item() and best.item() == out.best_angle.item()
    assert torch.equal(L, out.L.cpu()) and torch.equal(R, out.R.cpu())
    assert torch.equal(rp, out.row_price.cpu()) and torch.equal(ap, out.angle_price.cpu())


def test_pipelined_host_call_matches_the_device_call(vm, A0, h0):
    """vmat_price_eval_host_submit / _wait: seven evaluations through the two slots, every result equal to the device
    call's bit for bit; a slot in flight refuses a second submit."""
    obj = obj_to_device(A0, DEV)
    xs = [_x(A0["n_b"], 40 + k, (1.0, 8.0, 14.0, 16.0)[k % 4]) for k in range(7)]
    refs = []
    for x in xs:
        o = _eval_gpu(vm, h0, A0, x)
        refs.append({f: getattr(o, f).cpu().clone() for f in ("F", "L", "R", "row_price", "angle_price", "best_angle")})
    pin = lambda n, dt: torch.empty(n, dtype=dt).pin_memory()
    hb = [dict(F=pin(1, torch.float64), L=pin(h0.n_leaf_rows, torch.int32), R=pin(h0.n_leaf_rows, torch.int32),
               rp=pin(h0.n_leaf_rows, torch.float64), ap=pin(h0.n_angles, torch.float64), b=pin(1, torch.int32)) for _ in range(2)]
    xh = [x.pin_memory() for x in xs]

    def check(k):
        o, r = hb[k % 2], refs[k]
        vm.vmat_price_eval_host_wait(h0, k % 2)
        assert o["F"].item() == r["F"].item() and o["b"].item() == r["best_angle"].item(), k
        assert torch.equal(o["L"], r["L"]) and torch.equal(o["R"], r["R"]), k
        assert torch.equal(o["rp"], r["row_price"]) and torch.equal(o["ap"], r["angle_price"]), k

    for k in range(7):
        if k >= 2:
            check(k - 2)
        o = hb[k % 2]
        vm.vmat_price_eval_host_submit(h0, k % 2, xh[k], obj, o["F"], o["L"], o["R"], o["rp"], o["ap"], o["b"])
    with pytest.raises(vm.VmatError, match="in flight"):
        o = hb[0]
        vm.vmat_price_eval_host_submit(h0, 0, xh[0], obj, o["F"], o["L"], o["R"], o["rp"], o["ap"], o["b"])
    check(5)
    check(6)
    vm.vmat_price_eval_host_wait(h0, 0)                          # waiting for an idle slot is a no-op


def test_aperture_dose(vm, A0, h0):
    """NEXT-1, Eq. (5): DA = sum of the columns of the beamlets inside the chosen aperture."""
    x = _x(A0["n_b"], 26, 14.0)
    out = _eval_gpu(vm, h0, A0, x)
    a = int(out.best_angle.item())
    assert a >= 0
    DA = torch.empty(h0.n_voxels, dtype=torch.float32, device=DEV)
    xs = torch.empty(h0.n_beamlets, dtype=torch.float32, device=DEV)
    vm.vmat_aperture_dose(h0, a, out.L, out.R, xs, DA)
    ind = np.zeros(A0["n_b"], np.float32)
    L, R = out.L.cpu().numpy(), out.R.cpu().numpy()
    for r in range(A0["aro"][a], A0["aro"][a + 1]):
        ind[A0["lco"][r] + L[r]:A0["lco"][r] + R[r]] = 1.0
    assert ind.sum() > 0
    assert np.array_equal(xs.cpu().numpy(), ind)
    ref = oracle.dose(A0["vox"], A0["beam"], A0["val"], A0["n_v"], ind)
    assert_vec_close("DA", DA.cpu().numpy(), ref)
    # the sums are exact fixed-point sums rounded once: within one FP32 rounding of the FP64 oracle, and order-free
    assert np.abs(DA.cpu().numpy().astype(np.float64) - ref).max() <= 2.0 ** -23 * np.abs(ref).max()
    DA2 = torch.empty_like(DA)
    vm.vmat_aperture_dose(h0, a, out.L, out.R, xs, DA2)
    assert torch.equal(DA, DA2)


def test_aperture_dose_signed_and_large_values(vm):
    """Eq. (5) on a random matrix with entries of both signs up to 1e6 (the fixed-point scale adapts to max |D_ij|),
    leaf rows of several lengths, openings incl. closed and full rows, for every control point."""
    rng = np.random.default_rng(55)
    n_v, rows = 700, [[5, 0, 9], [40, 3], [1], [33, 33, 2, 7]]
    lens = np.concatenate([np.array(r) for r in rows])
    n_b = int(lens.sum())
    lco = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    aro = np.concatenate([[0], np.cumsum([len(r) for r in rows])]).astype(np.int32)
    dense = rng.random((n_v, n_b)) < 0.3
    vox, beam = np.nonzero(dense)
    val = ((rng.random(vox.size) - 0.5) * 2e6).astype(np.float32)
    h = vm.vmat_ddc_create(n_v, n_b, torch.from_numpy(vox.astype(np.int32)).to(DEV), torch.from_numpy(beam.astype(np.int32)).to(DEV),
                           torch.from_numpy(val).to(DEV), torch.from_numpy(lco[aro]), torch.from_numpy(aro),
                           torch.from_numpy(lco), device=DEV)
    L = np.array([rng.integers(0, n + 1) for n in lens], np.int32)
    R = np.array([rng.integers(l, n + 1) for l, n in zip(L, lens)], np.int32)
    L[1], R[1] = 0, 0
    L[3], R[3] = 0, lens[3]
    DA = torch.empty(n_v, dtype=torch.float32, device=DEV)
    xs = torch.empty(n_b, dtype=torch.float32, device=DEV)
    for a in range(len(rows)):
        vm.vmat_aperture_dose(h, a, torch.from_numpy(L).to(DEV), torch.from_numpy(R).to(DEV), xs, DA)
        ind = np.zeros(n_b, np.float32)
        for r in range(aro[a], aro[a + 1]):
            ind[lco[r] + L[r]:lco[r] + R[r]] = 1.0
        ref = oracle.dose(vox.astype(np.int32), beam.astype(np.int32), val, n_v, ind)
        assert np.array_equal(xs.cpu().numpy(), ind)
        assert np.abs(DA.cpu().numpy().astype(np.float64) - ref).max() <= 2.0 ** -23 * max(np.abs(ref).max(), 1e-30)
    h.close()


def test_structure_id_contract_check(vm):
    """vmat_check_structure_ids: ids must index the per-structure tables (the compute calls do not re-check)."""
    sid = torch.tensor([0, 1, 2, 1, 0, 3], dtype=torch.uint8, device=DEV)
    t4 = torch.ones(4, device=DEV)
    vm.Objective(sid, t4, t4, t4).validate()
    t3 = torch.ones(3, device=DEV)
    with pytest.raises(vm.VmatError) as e:
        vm.Objective(sid, t3, t3, t3).validate()
    assert e.value.status == -2
    vm.Objective(torch.zeros(0, dtype=torch.uint8, device=DEV), t3, t3, t3).validate()


def test_schedule_setting_and_read_probe(vm, A0, h0):
    """vmat_ddc_set_schedule: argument check, what info reports, the automatic choice on a tiny matrix (one CTA per item);
    vmat_hbm_read_probe (libvmat_probe.so, bench.py's aid): runs, returns a plausible rate, rejects bad arguments."""
    assert h0.info["sm_affine_dose"] == 0 and h0.info["sm_affine_price"] == 0          # config 0: a handful of items
    g0 = (h0.info["grid_dose"], h0.info["grid_price"])
    h0.set_schedule(True)
    assert h0.info["sm_affine_dose"] == 1 and h0.info["sm_affine_price"] == 1
    assert h0.info["grid_dose"] <= g0[0] and h0.info["grid_price"] <= g0[1]            # persistent grids never exceed the items
    with pytest.raises(vm.VmatError):
        h0.set_schedule(2)
    h0.set_schedule(None)
    assert h0.info["sm_affine_dose"] == 0 and (h0.info["grid_dose"], h0.info["grid_price"]) == g0
    from paper_1503_01721_b200 import probe
    gbs, n_launch = probe.hbm_read_probe(256 << 20, 5)
    assert 500.0 < gbs < 20000.0, gbs
    assert n_launch == 6                                                                 # warm-up + 5 passes
    with pytest.raises(RuntimeError, match="1 MiB"):
        probe.hbm_read_probe(1000, 1)
