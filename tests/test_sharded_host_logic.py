"""NEXT-4, N > 1 on the CPU: the angle-sharded evaluation's host logic (partition of the control points, re-based offset
tables, all-reduce of the dose, merge of the best control points) with world size 2 over gloo, plus unit tests of the
partition and the merge rule."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

from paper_1503_01721_b200 import sharded

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_angles():
    assert sharded.partition_angles([1] * 8, 2) == [0, 4, 8]
    assert sharded.partition_angles([1] * 8, 1) == [0, 8]
    assert sharded.partition_angles([1] * 9, 3) == [0, 3, 6, 9]
    offs = sharded.partition_angles([10, 1, 1, 1, 1, 10, 1, 1], 2)          # balanced by weight, not by count
    assert offs[0] == 0 and offs[-1] == 8 and abs(sum([10, 1, 1, 1, 1, 10, 1, 1][:offs[1]]) - 13) <= 5
    offs = sharded.partition_angles([1, 1], 4)                               # more ranks than control points
    assert offs[0] == 0 and offs[-1] == 2 and all(b >= a for a, b in zip(offs, offs[1:])) and len(offs) == 5
    rng = np.random.default_rng(0)
    for _ in range(50):
        w = rng.integers(0, 100, rng.integers(1, 40))
        k = int(rng.integers(1, 9))
        offs = sharded.partition_angles(w, k)
        assert len(offs) == k + 1 and offs[0] == 0 and offs[-1] == len(w)
        assert all(b >= a for a, b in zip(offs, offs[1:]))
        if w.sum() > 0:                                                      # no block is heavier than its share + one angle
            assert max(w[a:b].sum() for a, b in zip(offs, offs[1:])) <= w.sum() / k + w.max()


def test_local_block_rebases_the_offset_tables():
    aco = torch.tensor([0, 6, 6, 15, 20]); aro = torch.tensor([0, 2, 2, 5, 6])
    lco = torch.tensor([0, 3, 6, 9, 12, 15, 20])
    b = sharded.local_block(aco, aro, lco, 2, 4)
    assert (b.beamlet_lo, b.beamlet_hi, b.row_lo, b.row_hi) == (6, 20, 2, 6)
    assert b.angle_col_offset.tolist() == [0, 9, 14] and b.angle_row_offset.tolist() == [0, 3, 4]
    assert b.leafrow_col_offset.tolist() == [0, 3, 6, 9, 14]
    e = sharded.local_block(aco, aro, lco, 1, 2)                             # a control point without beamlets
    assert e.angle_col_offset.tolist() == [0, 0] and e.leafrow_col_offset.tolist() == [0]


def test_gather_pairs_without_a_process_group():
    pair = torch.tensor([-2.5, 13.0], dtype=torch.float64)
    assert sharded.gather_pairs(pair).tolist() == [[-2.5, 13.0]]


@pytest.mark.parametrize("xscale", ["14", "1"])
def test_two_ranks_reproduce_the_unsharded_evaluation(tmp_path, xscale):
    env = dict(os.environ, VMAT_TEST_OUT=str(tmp_path / "out"), VMAT_TEST_XSCALE=xscale)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", "29587", os.path.join(ROOT, "tests", "_shard_worker.py")]
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    res = [json.loads(lines[0]), json.load(open(str(tmp_path / "out") + ".1"))]
    assert res[0]["offs"] == res[1]["offs"] and res[0]["offs"][0] == 0 and res[0]["offs"][-1] == 8
    assert res[0]["block"][1] == res[1]["block"][0] and res[0]["block"][3] == res[1]["block"][2]   # blocks tile the matrix
    assert res[0]["nnz_local"] + res[1]["nnz_local"] == res[0]["nnz"] and min(r_["nnz_local"] for r_ in res) > 0
    for r_ in res:
        assert r_["d_err"] < 1e-12 and r_["F_err"] < 1e-12 and r_["p_err"] < 1e-12 and r_["ap_err"] < 1e-6
        assert r_["LR_equal"]
        assert r_["best"] == r_["best_ref"] and abs(r_["best_price"] - r_["best_price_ref"]) <= 1e-9 * abs(r_["best_price_ref"])
    assert res[0]["best"] == res[1]["best"]                                   # every rank knows the winner
