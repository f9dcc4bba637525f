"""NEXT-4 on one GPU: the angle-sharded evaluation with its column blocks evaluated one after the other (no rank
waits on another: the all-reduce of the dose is stood in for by a torch add of the partial doses, in this test only),
against the oracle and against the unsharded handle; and a single block through ShardedDDC.price_eval, which must be
vmat_price_eval bit for bit."""
import numpy as np
import pytest
import torch

import oracle
import synth
from conftest import as_np
from helpers import assert_vec_close, ddc_from_arrays, obj_to_device, oracle_eval, REL_L2

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def vm():
    import paper_1503_01721_b200 as vm
    vm.load_library()
    return vm


def _shards(ph, A, n_shards):
    from paper_1503_01721_b200 import sharded
    nnz_per_angle = np.bincount(np.searchsorted(A["aco"], A["beam"], side="right") - 1, minlength=ph.n_angles)
    offs = sharded.partition_angles(nnz_per_angle, n_shards)
    cv, cb, cval = (torch.from_numpy(A[k]).to(DEV) for k in ("vox", "beam", "val"))
    return offs, [sharded.ShardedDDC.create(ph.n_voxels, ph.n_beamlets, cv, cb, cval, ph.angle_col_offset,
                                            ph.angle_row_offset, ph.leafrow_col_offset, offs[m], offs[m + 1], device=DEV)
                  for m in range(n_shards)]


@pytest.mark.parametrize("n_shards,scale", [(2, 14.0), (3, 1.0), (8, 16.0)])
def test_blocks_add_up_to_the_unsharded_evaluation(vm, cfg0, n_shards, scale):
    from paper_1503_01721_b200 import sharded
    A = as_np(cfg0)
    obj = obj_to_device(A, DEV)
    x = synth.draw_x(A["n_b"], 9, device=DEV, scale=scale)
    ev = oracle_eval(A, x.cpu().numpy())
    offs, shards = _shards(cfg0, A, n_shards)
    assert sum(s.h.nnz for s in shards) == A["vox"].size
    outs = [s.h.alloc_outputs() for s in shards]
    for s, o in zip(shards, outs):                                   # rank m: d_m = D_m x_m
        vm.vmat_dose(s.h, x[s.block.beamlet_lo:s.block.beamlet_hi].contiguous(), o.d)
    d = torch.stack([o.d for o in outs]).sum(0)                      # all: d = sum_m d_m (stand-in for the all-reduce)
    assert_vec_close("d", d.cpu().numpy(), ev.d)
    cands = []
    for s, o in zip(shards, outs):
        o.d.copy_(d)
        vm.vmat_objective_grad(s.h, o.d, obj, o.g, o.F)
        vm.vmat_price_select(s.h, o.g, o)
        torch.cuda.synchronize()
        b = s.block
        assert_vec_close("g", o.g.cpu().numpy(), ev.g)
        assert abs(o.F.item() - ev.F) <= REL_L2 * abs(ev.F)
        p_loc = o.p.cpu().numpy()
        pmax = np.abs(ev.p).max()
        assert np.abs(p_loc - ev.p[b.beamlet_lo:b.beamlet_hi]).max() <= 1e-4 * pmax
        # selection protocol (C6 (ii)) on the block: the oracle applied to the GPU's own local prices
        L, R, rp = oracle.select_rows(p_loc, b.leafrow_col_offset.numpy())
        ap, lbest = oracle.angle_price(rp, b.angle_row_offset.numpy())
        assert np.array_equal(o.L.cpu().numpy(), L) and np.array_equal(o.R.cpu().numpy(), R)
        assert np.array_equal(o.row_price.cpu().numpy(), rp) and np.array_equal(o.angle_price.cpu().numpy(), ap)
        assert int(o.best_angle.item()) == lbest
        assert np.array_equal(L, ev.L[b.row_lo:b.row_hi]) and np.array_equal(R, ev.R[b.row_lo:b.row_hi])
        pair = torch.empty(2, dtype=torch.float64, device=DEV)
        vm.vmat_best_pair(s.h, o, b.angle_lo, pair)                   # {price, global control point} or {0, -1}
        assert pair.tolist() == ([float(ap[lbest]), float(lbest + b.angle_lo)] if lbest >= 0 else [0.0, -1.0])
        cands.append(pair)
    # the A5 rule over the blocks' candidates, on the device (what merge_best runs on the all-gathered pairs)
    best = torch.empty(2, dtype=torch.float64, device=DEV)
    vm.vmat_merge_best(torch.stack(cands).contiguous(), best)
    k, price = sharded.best_to_host(best)
    assert k == ev.best_angle
    if k >= 0:
        assert abs(price - ev.angle_price[k]) <= 1e-4 * abs(ev.angle_price[k])
    for s in shards:
        s.close()


def test_one_block_is_the_unsharded_call(vm, cfg0):
    A = as_np(cfg0)
    obj = obj_to_device(A, DEV)
    x = synth.draw_x(A["n_b"], 2, device=DEV, scale=14.0)
    h = ddc_from_arrays(A, DEV)
    ref = h.alloc_outputs()
    vm.vmat_price_eval(h, x, obj, ref)
    _, (s,) = _shards(cfg0, A, 1)
    out = s.h.alloc_outputs()
    from paper_1503_01721_b200 import sharded
    best, price = sharded.best_to_host(s.price_eval(x, obj, out))
    for name in ("d", "g", "F", "p", "L", "R", "row_price", "angle_price", "best_angle"):
        assert torch.equal(getattr(out, name), getattr(ref, name)), name
    assert best == int(ref.best_angle.item()) and price == float(ref.angle_price[best].item())
    s.close()
    h.close()


def test_merge_rule_on_the_device(vm):
    """vmat_merge_best against hand-worked candidate lists: smallest price, ties -> smallest control point, candidates
    without a control point never win, none below 0 -> {0, -1}."""
    cases = [([[-1.0, 7.0], [-3.0, 2.0], [-3.0, 1.0]], [-3.0, 1.0]), ([[0.0, -1.0], [-0.5, 9.0]], [-0.5, 9.0]),
             ([[0.0, -1.0], [0.0, -1.0]], [0.0, -1.0]), ([[-2.0, 5.0]], [-2.0, 5.0]), ([[-2.0, 5.0], [-2.0, 3.0], [0.0, -1.0]], [-2.0, 3.0])]
    for pairs, want in cases:
        best = torch.empty(2, dtype=torch.float64, device=DEV)
        vm.vmat_merge_best(torch.tensor(pairs, dtype=torch.float64, device=DEV), best)
        assert best.tolist() == want


def test_merge_rule_on_random_candidate_lists(vm):
    """vmat_merge_best against the A5 rule written out on the host (the aperture with the lowest
    price; ties -> smallest control point; none below 0 -> {0, -1}) on seeded candidate lists of 1..64 ranks, prices
    drawn from a few values so that ties across ranks are the rule, with ranks that report no candidate mixed in."""
    rng = np.random.default_rng(20260306)
    for case in range(300):
        n = int(rng.integers(1, 65))
        prices = rng.choice([-3.5, -1.25, -1.0, -0.5, -2.0 ** -40, 0.0], size=n)
        cps = rng.permutation(4 * n)[:n].astype(np.float64)
        none = (prices >= 0.0) | (rng.random(n) < 0.15)
        prices[none], cps[none] = 0.0, -1.0
        want = [0.0, -1.0]
        for pr, k in zip(prices.tolist(), cps.tolist()):                 # the rule, one candidate at a time
            if k >= 0 and pr < 0.0 and (pr < want[0] or (pr == want[0] and k < want[1])):
                want = [pr, k]
        best = torch.empty(2, dtype=torch.float64, device=DEV)
        vm.vmat_merge_best(torch.from_numpy(np.stack([prices, cps], 1)).to(DEV).contiguous(), best)
        assert best.tolist() == want, case


def test_collective_path_on_one_gpu_with_nccl(tmp_path):
    """ShardedDDC.price_eval through a REAL torch.distributed process group of world size 1 with the nccl backend: the
    all-reduce of the dose and the all-gather of the candidates run (not the no-process-group bypass), and the result
    is the unsharded call bit for bit (tests/_nccl1_worker.py)."""
    import json, os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29593", RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(root, "tests", "_nccl1_worker.py")], cwd=root, env=env,
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    res = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1])
    assert res["backend"] == "nccl" and res["world"] == 1 and res["collectives_ran"] >= 2
    assert res["equal"] and res["best"] == res["best_ref"] and res["price"] == res["price_ref"]
