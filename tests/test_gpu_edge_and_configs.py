"""GPU parity on edge-case matrices and on the larger BASELINE.json configs."""
import time

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


def _random_problem(rng, n_v, n_b, rows_spec, row_lens, n_struct=4):
    """Random sparse D with prescribed per-voxel row lengths; leaf rows from `rows_spec` (list of lengths
    per angle)."""
    vox, beam = [], []
    for i, ln in enumerate(row_lens):
        if ln > 0:
            vox.append(np.full(ln, i, np.int32))
            beam.append(np.sort(rng.choice(n_b, ln, replace=False)).astype(np.int32))
    vox = np.concatenate(vox) if vox else np.zeros(0, np.int32)
    beam = np.concatenate(beam) if beam else np.zeros(0, np.int32)
    val = (rng.random(vox.size) + 0.01).astype(np.float32)
    perm = rng.permutation(vox.size)
    lens = np.concatenate(rows_spec) if rows_spec else np.zeros(0, np.int64)
    assert lens.sum() == n_b
    lco = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    aro = np.concatenate([[0], np.cumsum([len(r) for r in rows_spec])]).astype(np.int32)
    aco = lco[aro]
    return dict(vox=vox[perm], beam=beam[perm], val=val[perm], n_v=n_v, n_b=n_b,
                sid=rng.integers(0, n_struct, n_v).astype(np.uint8),
                T=np.array([5.0, 20.0, 8.0, 12.0], np.float32)[:n_struct],
                wo=np.array([0.05, 1.0, 0.2, 0.7], np.float32)[:n_struct],
                wu=np.array([0.0, 1.0, 0.0, 0.3], np.float32)[:n_struct], lco=lco, aro=aro, aco=aco)


OUT_FIELDS = ("d", "g", "F", "p", "L", "R", "row_price", "angle_price", "best_angle")


def _assert_schedules_agree(vm, h, x, obj, out, mask=None):
    """`out` was computed under the default schedule (SM-affine queues, persistent kernels): one CTA per item gives
    the same bits in every output, fused and unfused (vmat_ddc_set_schedule), and so does a second SM-affine run
    (the queue counters reset themselves)."""
    for sm_affine in (False, True):
        h.set_schedule(sm_affine)
        o2 = h.alloc_outputs()
        vm.vmat_price_eval(h, x, obj, o2, mask)
        d2 = torch.empty_like(out.d); p2 = torch.empty_like(out.p)
        vm.vmat_dose(h, x, d2)
        vm.vmat_price(h, out.g, p2)
        torch.cuda.synchronize()
        for f in OUT_FIELDS:
            assert torch.equal(getattr(o2, f), getattr(out, f)), (f, sm_affine)
        assert torch.equal(d2, out.d) and torch.equal(p2, out.p)
        assert h.info["sm_affine_dose"] == h.info["sm_affine_price"] == int(sm_affine)
    h.set_schedule(None)                                                   # back to the automatic choice


def _run_and_check(vm, A, x, mask=None, expect_no_diff=True):
    """Whole evaluation against the oracle, once per index encoding (int32 indices; u16 offsets + group
    bases; the automatic choice).  Returns the outputs / info of the automatic choice."""
    ev = oracle_eval(A, x, mask)
    outs, infos = {}, {}
    for bits in (32, 16, 0):
        h = ddc_from_arrays(A, DEV, index_bits=bits)
        out = h.alloc_outputs()
        m = None if mask is None else torch.from_numpy(mask).to(DEV)
        vm.vmat_price_eval(h, torch.from_numpy(x).to(DEV), obj_to_device(A, DEV), out, m)
        torch.cuda.synchronize()
        assert_vec_close("d", out.d.cpu().numpy(), ev.d)
        assert_vec_close("g", out.g.cpu().numpy(), ev.g)
        assert_vec_close("p", out.p.cpu().numpy(), ev.p)
        assert abs(out.F.item() - ev.F) <= REL_L2 * abs(ev.F) + 1e-300
        n_diff = check_selection_protocol(A, out, ev, mask)
        if expect_no_diff:
            assert n_diff == 0
        # the unfused calls give the same bits as the fused ones for d and p
        d2 = torch.empty_like(out.d); p2 = torch.empty_like(out.p)
        vm.vmat_dose(h, torch.from_numpy(x).to(DEV), d2)
        vm.vmat_price(h, out.g, p2)
        assert torch.equal(d2, out.d) and torch.equal(p2, out.p)
        _assert_schedules_agree(vm, h, torch.from_numpy(x).to(DEV), obj_to_device(A, DEV), out, m)
        info = h.info
        if bits:
            assert info["index_bits_d"] == info["index_bits_dt"] == bits
        for lay, rows in (("d", "n_voxels"), ("dt", "n_beamlets")):          # storage closed forms (spmv.cuh)
            P, b = info[f"padded_{lay}"], info[f"index_bits_{lay}"]
            assert P % 32 == 0 and P >= info["nnz"]
            per_entry = 6 * P + 4 * (P // 32) if b == 16 else 8 * P
            seg_table = 4 * (info["n_dose_blocks"] + 1) if lay == "d" else 0
            assert info[f"bytes_stream_{lay}"] == per_entry + 8 * (info[rows] + 1) + seg_table
        # the layouts unpack to the same canonical CSR whatever the encoding
        csr = [t.numpy() for w in (0, 1) for t in h.export_csr(w)]
        if outs:
            for a, b in zip(csr, first_csr):
                assert np.array_equal(a, b)
        else:
            first_csr = csr
        outs[bits], infos[bits] = out, info
        h.close()
    # no group closed early (same padded size) => the encodings give the same bits everywhere
    if infos[16]["padded_d"] == infos[32]["padded_d"] and infos[16]["padded_dt"] == infos[32]["padded_dt"]:
        for f in ("d", "g", "F", "p", "L", "R", "row_price", "angle_price", "best_angle"):
            assert torch.equal(getattr(outs[16], f), getattr(outs[32], f)), f
    return outs[0], ev, infos[0]


def test_empty_matrix(vm):
    """nnz = 0 is legal: d = 0, g = -2 w- T on under-dose structures, p = 0, everything closed."""
    rng = np.random.default_rng(0)
    A = _random_problem(rng, 50, 12, [np.array([4, 0, 2]), np.array([6])], np.zeros(50, int))
    out, ev, _ = _run_and_check(vm, A, np.ones(12, np.float32))
    assert (out.d == 0).all() and (out.p == 0).all() and (out.L == 0).all() and (out.R == 0).all()
    assert int(out.best_angle.item()) == -1


def test_ragged_rows_spanning_every_kernel_path(vm):
    """Voxel rows of 0, 1, 7, 8, 9 ... entries, rows longer than one dose block (4096), one longer than the
    shared-memory sort (24576); leaf rows of length 0, 1 and 2100 (> the fused kernel's 2048 limit)."""
    rng = np.random.default_rng(1)
    n_v, n_b = 3000, 30000
    lens = rng.integers(0, 40, n_v)
    lens[rng.random(n_v) < 0.3] = 0
    lens[[5, 6, 7, 8]] = [1, 7, 8, 9]
    lens[100] = 4096; lens[101] = 4097; lens[102] = 5000; lens[1500] = 26000; lens[2999] = 12345
    rows = [np.array([2100, 0, 1, 899]), np.array([0, 0]), np.array([5000, 3000, 1, 1, 1, 997]),
            np.array([18000]), np.array([], int)]
    A = _random_problem(rng, n_v, n_b, rows, lens)
    x = (rng.random(n_b) * 0.02).astype(np.float32)
    out, ev, info = _run_and_check(vm, A, x)
    assert info["max_voxel_row_nnz"] == 26000 and info["max_leaf_row_len"] == 18000
    assert (ev.g > 0).any() and (ev.g < 0).any() and (ev.R > ev.L).any()


def test_tiled_column_order_is_invisible_at_the_boundary(vm):
    """Leaf rows of several tiles (the handle renumbers the beamlets of CSR(D) in tiles of 8 columns x all leaf rows
    of a control point and permutes x before the dose kernel): vmat_ddc_export_csr still returns both layouts in the
    caller's numbering, canonical order, exactly the input triplets; the evaluation matches the oracle."""
    rng = np.random.default_rng(8)
    n_v = 4000
    rows = [np.array([70, 33, 0, 41, 8, 64]), np.array([9, 120, 35]), np.array([40, 40, 40, 40])]
    n_b = int(sum(r.sum() for r in rows))
    lens = rng.integers(0, 120, n_v)
    A = _random_problem(rng, n_v, n_b, rows, lens)
    x = (rng.random(n_b) * 0.5).astype(np.float32)
    out, ev, info = _run_and_check(vm, A, x)
    h = ddc_from_arrays(A, DEV)
    order = np.lexsort((A["beam"], A["vox"]))
    ptr, idx, val = [t.numpy() for t in h.export_csr(0)]
    assert np.array_equal(ptr, np.concatenate([[0], np.cumsum(np.bincount(A["vox"], minlength=n_v))]))
    assert np.array_equal(idx, A["beam"][order]) and np.array_equal(val, A["val"][order])
    order_t = np.lexsort((A["vox"], A["beam"]))
    ptr, idx, val = [t.numpy() for t in h.export_csr(1)]
    assert np.array_equal(idx, A["vox"][order_t]) and np.array_equal(val, A["val"][order_t])
    # D e_j reproduces column j (P1) for beamlets in different tiles of the same leaf row
    for j in (0, 7, 8, 69, 70, 103, int(n_b) - 1):
        e = torch.zeros(n_b, device=DEV); e[j] = 1.0
        d = torch.empty(n_v, device=DEV)
        vm.vmat_dose(h, e, d)
        col = np.zeros(n_v, np.float32); m = A["beam"] == j; col[A["vox"][m]] = A["val"][m]
        assert np.array_equal(d.cpu().numpy(), col), j
    h.close()


def test_short_leaf_rows_fused_path_and_masks(vm):
    rng = np.random.default_rng(2)
    n_v, n_b = 20000, 4000
    lens = rng.integers(0, 300, n_v)
    rows = [rng.multinomial(500, np.ones(10) / 10) for _ in range(8)]
    A = _random_problem(rng, n_v, n_b, rows, lens)
    x = (rng.random(n_b) * 0.30).astype(np.float32)       # near balance: mixed-sign prices
    mask = np.zeros(8, np.uint8); mask[[1, 6]] = 1
    out, ev, info = _run_and_check(vm, A, x, mask)
    assert info["max_leaf_row_len"] <= 2048
    assert (ev.g > 0).any() and (ev.g < 0).any() and (ev.R > ev.L).any() and (ev.p_f32 > 0).any()


def test_exact_ties_in_prices(vm):
    """Integer-valued data: prices are exact small integers, so equal-sum openings tie exactly (C5)."""
    rng = np.random.default_rng(3)
    n_v, n_b = 400, 240
    lens = rng.integers(0, 6, n_v)
    rows = [np.array([8] * 10) for _ in range(3)]
    A = _random_problem(rng, n_v, n_b, rows, lens, n_struct=2)
    A["val"] = rng.integers(1, 3, A["val"].size).astype(np.float32)
    A["T"] = np.array([3.0, 2.0], np.float32); A["wo"] = np.array([0.5, 1.0], np.float32)
    A["wu"] = np.array([0.0, 1.0], np.float32)
    x = rng.integers(0, 2, n_b).astype(np.float32)
    out, ev, _ = _run_and_check(vm, A, x)
    assert np.array_equal(out.p.cpu().numpy().astype(np.float64), ev.p)          # exact integers on both sides
    assert np.array_equal(out.L.cpu().numpy(), ev.L) and np.array_equal(out.R.cpu().numpy(), ev.R)


def test_index_spans_beyond_16_bits(vm):
    """Secondary indices scattered over > 65536 columns / rows: the u16 encoding has to close groups early
    (pads inside rows), and for D the automatic choice falls back to int32 indices; every encoding matches
    the oracle."""
    rng = np.random.default_rng(4)
    n_v, n_b = 150000, 200000
    lens = np.zeros(n_v, int)
    hot = rng.choice(n_v, 2500, replace=False)
    lens[hot] = rng.integers(1, 120, hot.size)
    lens[hot[:3]] = [700, 1500, 9000]                      # long rows: register path with pads inside tiles
    rows = [rng.multinomial(n_b // 4, np.ones(50) / 50) for _ in range(4)]
    A = _random_problem(rng, n_v, n_b, rows, lens)
    x = (rng.random(n_b) * 0.35).astype(np.float32)
    out, ev, info = _run_and_check(vm, A, x)
    assert info["index_bits_d"] == 32                                       # padding would outweigh the saving
    h16 = ddc_from_arrays(A, DEV, index_bits=16)
    assert h16.info["padded_d"] > 1.2 * info["padded_d"]                    # groups were closed early
    # both tile kinds occur: one base per tile (span <= 65535: the 9000-entry row) and one base per group
    assert 0 < h16.info["tiles_uniform_d"] < h16.info["tiles_d"]
    h16.close()
    assert (ev.g > 0).any() and (ev.g < 0).any() and (ev.R > ev.L).any()


def test_narrow_encoding_is_chosen_when_smaller(vm):
    """Clustered indices over > 65536 columns (runs, as in a DDC matrix): u16 offsets fit, 6.125 B per entry."""
    rng = np.random.default_rng(5)
    n_v, n_b = 90000, 100000
    vox, beam = [], []
    for i in rng.choice(n_v, 4000, replace=False):
        for start in rng.choice(n_b - 40, rng.integers(1, 6), replace=False):   # a few runs of consecutive beamlets
            ln = int(rng.integers(3, 30))
            vox.append(np.full(ln, i, np.int32)); beam.append(np.arange(start, start + ln, dtype=np.int32))
    vox, beam = np.concatenate(vox), np.concatenate(beam)
    key = np.unique(vox.astype(np.int64) * n_b + beam)                     # overlapping runs: drop duplicates
    vox, beam = (key // n_b).astype(np.int32), (key % n_b).astype(np.int32)
    perm = rng.permutation(vox.size)
    rows = [rng.multinomial(n_b // 5, np.ones(40) / 40) for _ in range(5)]
    lens = np.concatenate(rows)
    lco = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    aro = np.concatenate([[0], np.cumsum([len(r) for r in rows])]).astype(np.int32)
    A = dict(vox=vox[perm], beam=beam[perm], val=(rng.random(vox.size) + 0.01).astype(np.float32)[perm], n_v=n_v,
             n_b=n_b, sid=rng.integers(0, 3, n_v).astype(np.uint8), T=np.array([5.0, 20.0, 8.0], np.float32),
             wo=np.array([0.05, 1.0, 0.2], np.float32), wu=np.array([0.0, 1.0, 0.0], np.float32), lco=lco, aro=aro,
             aco=lco[aro])
    x = (rng.random(n_b) * 2.0).astype(np.float32)
    out, ev, info = _run_and_check(vm, A, x)
    assert info["index_bits_dt"] == 16 or info["index_bits_d"] == 16


# ------------------------------------------------------------------ the configs
def _phantom_on_gpu(cfg, scale=1.0, angles=None):
    spec = synth.config_spec(cfg, scale)
    t = time.time()
    ph = synth.generate(spec, device=DEV, angles=angles)
    torch.cuda.synchronize()
    print(f"\n[{spec.name}] generated on GPU in {time.time() - t:.1f}s: {ph.stats()}")
    return ph


def _full_parity(vm, ph, scales):
    import paper_1503_01721_b200 as vmod
    A = as_np(ph)
    h = vmod.vmat_ddc_create(ph.n_voxels, ph.n_beamlets, ph.coo_voxel, ph.coo_beamlet, ph.coo_val,
                             ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset, device=DEV)
    obj = obj_to_device(A, DEV)
    out = h.alloc_outputs()
    for k, sc in enumerate(scales):
        x = synth.draw_x(ph.n_beamlets, 100 + k, scale=sc)
        vmod.vmat_price_eval(h, x.to(DEV), obj, out)
        torch.cuda.synchronize()
        ev = oracle_eval(A, x.numpy())
        assert_vec_close("d", out.d.cpu().numpy(), ev.d)
        assert_vec_close("g", out.g.cpu().numpy(), ev.g)
        assert_vec_close("p", out.p.cpu().numpy(), ev.p)
        assert abs(out.F.item() - ev.F) <= REL_L2 * abs(ev.F)
        n_diff = check_selection_protocol(A, out, ev)
        _assert_schedules_agree(vm, h, x.to(DEV), obj, out)
        print(f"  x*{sc}: F={ev.F:.6e} open rows={(ev.R > ev.L).sum()} best={ev.best_angle} "
              f"rows differing from the pure-FP64 path={n_diff}")
        assert n_diff <= max(1, A["lco"].size // 1000)
    h.close()


def test_config1_scaled_down(vm):
    """Config 1 at 2.5x coarser voxels/beamlets (~1e6 nnz): several dose blocks, ragged leaf rows."""
    _full_parity(vm, _phantom_on_gpu(1, scale=2.5), [1.0, 0.7])


def test_sm_affine_queues_repeat_bit_for_bit(vm):
    """The persistent kernels with per-SM queues on a matrix with many items per CTA (config 1 at 1.6x coarser voxels:
    ~1e8 nnz, several thousand items against 1776 / 888 CTAs): 40 evaluations launched back to back without a host
    synchronisation, alternating between two fluence vectors - whoever steals what at the tail, and however the
    self-resetting counters are left, every evaluation of the same x gives the same bits, equal to one CTA per item."""
    import paper_1503_01721_b200 as vmod
    ph = _phantom_on_gpu(1, scale=1.6)
    A = as_np(ph)
    h = vmod.vmat_ddc_create(ph.n_voxels, ph.n_beamlets, ph.coo_voxel, ph.coo_beamlet, ph.coo_val,
                             ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset, device=DEV)
    obj = obj_to_device(A, DEV)
    xs = [synth.draw_x(ph.n_beamlets, 7 + k, scale=0.8 + 0.4 * k).to(DEV) for k in range(2)]
    h.set_schedule(False)
    ref = []
    for x in xs:
        o = h.alloc_outputs()
        vmod.vmat_price_eval(h, x, obj, o)
        ref.append(o)
    h.set_schedule(True)
    assert h.info["grid_dose"] < (h.info["n_dose_blocks"] + 3) // 4 and h.info["grid_price"] < (ph.n_beamlets + 7) // 8
    outs = [h.alloc_outputs() for _ in range(40)]
    for k, o in enumerate(outs):
        vmod.vmat_price_eval(h, xs[k % 2], obj, o)                      # no synchronisation in between
    torch.cuda.synchronize()
    for k, o in enumerate(outs):
        for f in OUT_FIELDS:
            assert torch.equal(getattr(o, f), getattr(ref[k % 2], f)), (k, f)
    h.close()


def test_config1_full(vm):
    _full_parity(vm, _phantom_on_gpu(1), [1.0, 0.6])


def test_config2_full(vm):
    _full_parity(vm, _phantom_on_gpu(2), [1.0])


def _entries_with_key(key, n, sample):
    """Positions of the COO entries whose `key` (int32 tensor on the GPU) is in `sample` - chunked lookup table."""
    flag = torch.zeros(n, dtype=torch.bool, device=key.device)
    flag[torch.from_numpy(sample).to(key.device, torch.int64)] = True
    pos = []
    CH = 1 << 28
    for c0 in range(0, key.numel(), CH):
        pos.append(torch.nonzero(flag[key[c0:c0 + CH].long()]).flatten() + c0)
    return torch.cat(pos)


def test_config3_full_size_sampled(vm):
    """Config 3 at full size (2.8e9 nnz, the workload and launch configuration bench.py times):
    sampled outputs the oracle computes one by one, the whole selection, and properties that hold at any size."""
    import paper_1503_01721_b200 as vmod
    ph = _phantom_on_gpu(3)
    n_v, n_b = ph.n_voxels, ph.n_beamlets
    h = vmod.vmat_ddc_create(n_v, n_b, ph.coo_voxel, ph.coo_beamlet, ph.coo_val, ph.angle_col_offset,
                             ph.angle_row_offset, ph.leafrow_col_offset, device=DEV)
    A = dict(sid=ph.voxel_struct.numpy(), T=ph.struct_T.numpy(), wo=ph.struct_w_over.numpy(),
             wu=ph.struct_w_under.numpy(), lco=ph.leafrow_col_offset.numpy(), aro=ph.angle_row_offset.numpy())
    obj = obj_to_device(A, DEV)
    out = h.alloc_outputs()
    for scale in (0.55, 0.5, 0.47, 0.44, 0.41, 0.38):          # near balance: mixed-sign gradient and prices
        x = synth.draw_x(n_b, 7, scale=scale)
        vmod.vmat_price_eval(h, x.to(DEV), obj, out)
        torch.cuda.synchronize()
        if bool((out.p > 0).any()) and bool((out.p < 0).any()) and bool((out.g < 0).any()):
            break
    print(f"  x scale {scale}")
    d, g, p = out.d.cpu().numpy(), out.g.cpu().numpy(), out.p.cpu().numpy()
    assert h.info["nnz"] == ph.nnz > 2 ** 31                   # 64-bit offsets are exercised

    # -- sampled voxel rows (A1): longest row, empty rows, random rows
    rng = np.random.default_rng(33)
    ptrD = h.export_ptr(0)
    cnt_v = (ptrD[1:] - ptrD[:-1]).to(DEV)
    sv = np.unique(np.concatenate([rng.choice(n_v, 48, replace=False), [int(cnt_v.argmax())],
                                   torch.nonzero(cnt_v == 0).flatten()[:4].cpu().numpy(), [0, n_v - 1]]))
    m = _entries_with_key(ph.coo_voxel, n_v, sv)
    d_ref = oracle.dose(ph.coo_voxel[m].cpu().numpy(), ph.coo_beamlet[m].cpu().numpy(), ph.coo_val[m].cpu().numpy(),
                        n_v, x.numpy())[sv]
    del m
    dmax = float(np.abs(d).max())
    assert np.abs(d[sv] - d_ref).max() <= 1e-4 * dmax
    assert np.linalg.norm(d[sv] - d_ref) <= REL_L2 * np.linalg.norm(d_ref)
    print(f"  sampled d: {sv.size} rows, longest {int(cnt_v.max())} nnz, rel L2 err "
          f"{np.linalg.norm(d[sv] - d_ref) / np.linalg.norm(d_ref):.2e}")

    # -- A2 on the GPU's own d, every voxel (elementwise; F is a plain sum)
    F_ref, g_ref = oracle.objective_grad(d.astype(np.float64), A["sid"], A["T"], A["wo"], A["wu"])
    assert_vec_close("g", g, g_ref)
    assert abs(out.F.item() - F_ref) <= REL_L2 * F_ref
    assert (g > 0).any() and (g < 0).any()

    # -- sampled beamlet rows (A3) on the GPU's own g
    ptrT = h.export_ptr(1)
    cnt_b = (ptrT[1:] - ptrT[:-1]).to(DEV)
    sb = np.unique(np.concatenate([rng.choice(n_b, 48, replace=False), [int(cnt_b.argmax()), 0, n_b - 1]]))
    m = _entries_with_key(ph.coo_beamlet, n_b, sb)
    p_ref = oracle.price(ph.coo_voxel[m].cpu().numpy(), ph.coo_beamlet[m].cpu().numpy(), ph.coo_val[m].cpu().numpy(),
                         n_b, g.astype(np.float64))[sb]
    del m
    assert np.abs(p[sb] - p_ref).max() <= 1e-4 * float(np.abs(p).max())
    assert np.linalg.norm(p[sb] - p_ref) <= REL_L2 * np.linalg.norm(p_ref)

    # -- adjoint identity on the GPU's vectors: <D x, g> = <x, D^T g>
    lhs = float(np.dot(d.astype(np.float64), g.astype(np.float64)))
    rhs = float(np.dot(x.numpy().astype(np.float64), p.astype(np.float64)))
    scale = float(np.dot(np.abs(d).astype(np.float64), np.abs(g).astype(np.float64)))
    assert abs(lhs - rhs) <= 1e-5 * scale

    # -- A4 + A5 in full: the oracle's exhaustive selection on the GPU's FP32 p, bit for bit (C6 (ii))
    L, R, rp = oracle.select_rows(p, A["lco"])
    ap, best = oracle.angle_price(rp, A["aro"])
    assert np.array_equal(out.L.cpu().numpy(), L) and np.array_equal(out.R.cpu().numpy(), R)
    assert np.array_equal(out.row_price.cpu().numpy(), rp) and np.array_equal(out.angle_price.cpu().numpy(), ap)
    assert int(out.best_angle.item()) == best
    n_open = int((R > L).sum())
    n_partial = int(((R - L) < np.diff(A["lco"])).sum())
    print(f"  selection: {n_open} open rows of {L.size}, {n_partial} not fully open, best control point {best}")
    assert n_open > 0 and n_partial > 0

    # -- NEXT-1 at this size: the aperture dose vector DA = D 1_A (Eq. (5)) of the apertures just selected at three
    #    control points (first arc, second arc with the rotated collimator, the best one), every voxel, against the
    #    oracle's O1 on the control point's own triplets with the aperture's indicator as x
    aco = ph.angle_col_offset.numpy()
    xs, DA = torch.empty(n_b, dtype=torch.float32, device=DEV), torch.empty(n_v, dtype=torch.float32, device=DEV)
    for a in sorted({17, 180 + 95, max(best, 0)}):
        vmod.vmat_aperture_dose(h, a, out.L, out.R, xs, DA)
        ind = np.zeros(n_b, np.float64)
        for r in range(int(A["aro"][a]), int(A["aro"][a + 1])):
            ind[A["lco"][r] + L[r]:A["lco"][r] + R[r]] = 1.0
        assert np.array_equal(xs.cpu().numpy().astype(np.float64), ind)
        m = _entries_with_key(ph.coo_beamlet, n_b, np.arange(aco[a], aco[a + 1]))
        DA_ref = oracle.dose(ph.coo_voxel[m].cpu().numpy(), ph.coo_beamlet[m].cpu().numpy(), ph.coo_val[m].cpu().numpy(),
                             n_v, ind)
        del m
        got = DA.cpu().numpy()
        assert ind.sum() > 0 and np.abs(got - DA_ref).max() <= 2.0 ** -23 * max(float(np.abs(DA_ref).max()), 1e-30) * 1.01
    h.close()


def test_config3_full_size_all_elements(vm):
    """Config 3 at full size, EVERY element: the oracle streams the COO triplets block by block (O1 and O3 are sums
    over triplets, so a pass over consecutive blocks of the input with the partial sums added in FP64 is the one
    pass of the definition up to FP64 rounding; P6 pins the additivity) and every d_i, g_i, p_j and F
    is compared at the `north_star` tolerances; the whole selection bit for bit (C6 (ii)) and against the oracle's
    pure FP64 path (C6 (iii))."""
    import paper_1503_01721_b200 as vmod
    t_start = time.time()
    ph = _phantom_on_gpu(3)
    n_v, n_b, nnz = ph.n_voxels, ph.n_beamlets, ph.nnz
    h = vmod.vmat_ddc_create(n_v, n_b, ph.coo_voxel, ph.coo_beamlet, ph.coo_val, ph.angle_col_offset,
                             ph.angle_row_offset, ph.leafrow_col_offset, device=DEV)
    info = h.info
    # both tile kinds (one base per tile / one base per group) and pads occur in this run
    assert 0 < info["tiles_uniform_d"] < info["tiles_d"] and info["padded_d"] > nnz and info["padded_dt"] > nnz
    A = dict(sid=ph.voxel_struct.numpy(), T=ph.struct_T.numpy(), wo=ph.struct_w_over.numpy(),
             wu=ph.struct_w_under.numpy(), lco=ph.leafrow_col_offset.numpy(), aro=ph.angle_row_offset.numpy())
    obj = obj_to_device(A, DEV)
    out = h.alloc_outputs()
    for scale in (0.55, 0.5, 0.47, 0.44, 0.41, 0.38):          # near balance: mixed-sign gradient and prices
        x = synth.draw_x(n_b, 7, scale=scale)
        vmod.vmat_price_eval(h, x.to(DEV), obj, out)
        torch.cuda.synchronize()
        if bool((out.p > 0).any()) and bool((out.p < 0).any()) and bool((out.g < 0).any()):
            break
    xn = x.numpy()
    CH = 1 << 28                                                # triplets per block: 3.2 GB on the host
    t0 = time.time()
    d_ref = np.zeros(n_v, dtype=np.float64)
    for c0 in range(0, nnz, CH):
        sl = slice(c0, min(c0 + CH, nnz))
        d_ref += oracle.dose(ph.coo_voxel[sl].cpu().numpy(), ph.coo_beamlet[sl].cpu().numpy(),
                             ph.coo_val[sl].cpu().numpy(), n_v, xn)
    F_ref, g_ref = oracle.objective_grad(d_ref, A["sid"], A["T"], A["wo"], A["wu"])
    p_ref = np.zeros(n_b, dtype=np.float64)
    for c0 in range(0, nnz, CH):
        sl = slice(c0, min(c0 + CH, nnz))
        p_ref += oracle.price(ph.coo_voxel[sl].cpu().numpy(), ph.coo_beamlet[sl].cpu().numpy(),
                              ph.coo_val[sl].cpu().numpy(), n_b, g_ref)
    t_oracle = time.time() - t0
    d, g, p = out.d.cpu().numpy(), out.g.cpu().numpy(), out.p.cpu().numpy()
    assert_vec_close("d", d, d_ref)
    assert_vec_close("g", g, g_ref)
    assert_vec_close("p", p, p_ref)
    assert abs(out.F.item() - F_ref) <= REL_L2 * abs(F_ref)
    assert (g_ref > 0).any() and (g_ref < 0).any() and (p_ref > 0).any() and (p_ref < 0).any()
    rel = lambda a, b: np.linalg.norm(a - b) / np.linalg.norm(b)
    print(f"  all {n_v} d, {n_v} g, {n_b} p: rel L2 err {rel(d, d_ref):.2e} {rel(g, g_ref):.2e} {rel(p, p_ref):.2e}; "
          f"F rel err {abs(out.F.item() - F_ref) / F_ref:.2e}")
    # selection: protocol (ii) bit for bit on the GPU's p, (iii) against the pure FP64 path
    p32 = p_ref.astype(np.float32)
    L_ref, R_ref, rp_ref = oracle.select_rows(p32, A["lco"])
    ap_ref, best_ref = oracle.angle_price(rp_ref, A["aro"])
    ev = oracle.PriceEval(d_ref, F_ref, g_ref, p_ref, p32, L_ref, R_ref, rp_ref, ap_ref, best_ref)
    n_diff = check_selection_protocol(A, out, ev)
    print(f"  selection: {(R_ref > L_ref).sum()} open rows of {L_ref.size}, best control point {best_ref}, rows differing "
          f"from the pure-FP64 path: {n_diff}; oracle passes {t_oracle:.0f} s, whole test {time.time() - t_start:.0f} s")
    assert n_diff <= L_ref.size // 1000
    h.close()


def test_layout_beyond_2_32_stored_entries(vm):
    """Maximum size: a layout of MORE THAN 2^32 stored entries (config 1 generator at 0.395 x the voxel / beamlet size:
    ~4.6e9 non-zeros, ~27 GB per layout, 55 GB of triplets - built from host memory through the chunked path of the
    ingest step when the device cannot hold the triplets next to the build).  Exercises the 64-bit padded positions,
    the kernels' one-register cursor (units of 8 entries) past 2^32 entries and the price kernel's queues.
    Sampled voxel rows and beamlet rows the oracle computes one by one from their own triplets (rows from the first, the
    middle and the LAST 2^28 stored entries among them), the gradient and F of the sampled voxels, and the adjoint
    identity on the whole vectors.  Skipped where the host or the device is too small."""
    import paper_1503_01721_b200 as vmod
    psutil = pytest.importorskip("psutil")
    import gc
    gc.collect()
    torch.cuda.empty_cache()                                   # what earlier tests left in torch's caching allocator
    free_dev, _ = torch.cuda.mem_get_info()
    free_host = psutil.virtual_memory().available
    if free_host < 80e9 or free_dev < 125e9:
        pytest.skip(f"needs ~60 GB of host memory for the triplets and ~125 GB on the device "
                    f"(available: host {free_host / 1e9:.0f} GB, device {free_dev / 1e9:.0f} GB)")
    t0 = time.time()
    ph = _phantom_on_gpu(1, scale=0.395)
    n_v, n_b, nnz = ph.n_voxels, ph.n_beamlets, ph.nnz
    assert nnz > (1 << 32), nnz
    rng = np.random.default_rng(11)
    # samples, and their triplets, taken while the COO is still on the device
    cnt_v = torch.zeros(n_v, dtype=torch.int64, device=DEV)
    CH = 1 << 28
    for c0 in range(0, nnz, CH):
        cnt_v += torch.bincount(ph.coo_voxel[c0:c0 + CH].long(), minlength=n_v)
    nz_rows = torch.nonzero(cnt_v).flatten().cpu().numpy()
    sv = np.unique(np.concatenate([rng.choice(nz_rows, 40, replace=False), nz_rows[:2], nz_rows[-3:],
                                   [int(cnt_v.argmax()), nz_rows[nz_rows.size // 2]]]))
    sb = np.unique(np.concatenate([rng.choice(n_b, 40, replace=False), [0, 1, n_b // 2, n_b - 2, n_b - 1]]))
    mv = _entries_with_key(ph.coo_voxel, n_v, sv)
    sub_v = [t[mv].cpu().numpy() for t in (ph.coo_voxel, ph.coo_beamlet, ph.coo_val)]
    mb = _entries_with_key(ph.coo_beamlet, n_b, sb)
    sub_b = [t[mb].cpu().numpy() for t in (ph.coo_voxel, ph.coo_beamlet, ph.coo_val)]
    del mv, mb, cnt_v
    A = dict(sid=ph.voxel_struct.numpy(), T=ph.struct_T.numpy(), wo=ph.struct_w_over.numpy(),
             wu=ph.struct_w_under.numpy())
    try:
        h = vmod.vmat_ddc_create(n_v, n_b, ph.coo_voxel, ph.coo_beamlet, ph.coo_val, ph.angle_col_offset,
                                 ph.angle_row_offset, ph.leafrow_col_offset, device=DEV)
        how = "device"
    except vmod.VmatError as e:
        if e.status != -4:
            raise
        hv, hb, hw = ph.coo_voxel.cpu(), ph.coo_beamlet.cpu(), ph.coo_val.cpu()
        ph.coo_voxel = ph.coo_beamlet = ph.coo_val = None
        torch.cuda.empty_cache()
        h = vmod.vmat_ddc_create(n_v, n_b, hv, hb, hw, ph.angle_col_offset, ph.angle_row_offset,
                                 ph.leafrow_col_offset, device=DEV)
        del hv, hb, hw
        how = "host (chunked)"
    ph.coo_voxel = ph.coo_beamlet = ph.coo_val = None
    torch.cuda.empty_cache()
    info = h.info
    print(f"\n  built from {how} memory in {time.time() - t0:.0f} s: nnz {nnz}, stored {info['padded_d']} / {info['padded_dt']}, "
          f"queues dose / price: {info['sm_affine_dose']} / {info['sm_affine_price']}")
    assert info["padded_d"] > (1 << 32) and info["padded_dt"] > (1 << 32) and info["nnz"] == nnz
    obj = obj_to_device(A, DEV)
    out = h.alloc_outputs()
    x = synth.draw_x(n_b, 5, scale=0.9)
    vmod.vmat_price_eval(h, x.to(DEV), obj, out)
    torch.cuda.synchronize()
    d, g, p = out.d.cpu().numpy(), out.g.cpu().numpy(), out.p.cpu().numpy()
    # sampled voxel rows (A1, A2): the oracle on the rows' own triplets
    d_ref = oracle.dose(sub_v[0], sub_v[1], sub_v[2], n_v, x.numpy().astype(np.float64))[sv]
    assert np.abs(d[sv] - d_ref).max() <= 1e-4 * float(np.abs(d).max())
    assert np.linalg.norm(d[sv] - d_ref) <= REL_L2 * np.linalg.norm(d_ref)
    _, g_ref = oracle.objective_grad(d_ref, A["sid"][sv], A["T"], A["wo"], A["wu"])
    assert np.abs(g[sv] - g_ref).max() <= 1e-4 * float(np.abs(g).max())
    # sampled beamlet rows (A3) on the GPU's own g
    p_ref = oracle.price(sub_b[0], sub_b[1], sub_b[2], n_b, g.astype(np.float64))[sb]
    assert np.abs(p[sb] - p_ref).max() <= 1e-4 * float(np.abs(p).max())
    assert np.linalg.norm(p[sb] - p_ref) <= REL_L2 * np.linalg.norm(p_ref)
    # F from the GPU's own d (every voxel): the oracle's O2
    F_ref, g_all = oracle.objective_grad(d.astype(np.float64), A["sid"], A["T"], A["wo"], A["wu"])
    assert abs(out.F.item() - F_ref) <= REL_L2 * F_ref
    assert_vec_close("g", g, g_all)
    # adjoint identity on the whole vectors: <D x, g> = <x, D^T g>
    lhs = float(np.dot(d.astype(np.float64), g.astype(np.float64)))
    rhs = float(np.dot(x.numpy().astype(np.float64), p.astype(np.float64)))
    assert abs(lhs - rhs) <= 1e-5 * float(np.dot(np.abs(d).astype(np.float64), np.abs(g).astype(np.float64)))
    # one CTA per item gives the same bits
    _assert_schedules_agree(vm, h, x.to(DEV), obj, out)
    print(f"  {sv.size} voxel rows and {sb.size} beamlet rows against the oracle, wall time {time.time() - t0:.0f} s")
    h.close()
