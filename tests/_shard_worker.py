"""Worker of test_sharded_host_logic.py: the host logic of the angle-sharded evaluation (paper_1503_01721_b200/sharded.py:
partition, re-based offset tables, the all-reduce of the dose, the all-gather of the candidate control points) under
torch.distributed.run with gloo.  No GPU here, so every rank's kernels are stood in for by the oracle applied to the
rank's own column block - which is exactly the angle-block additivity of PAPER.md L119 (pin P6)."""
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import oracle
import synth
from paper_1503_01721_b200 import sharded

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ph = synth.generate(synth.config_spec(0))
vox, beam, val = ph.coo_voxel.numpy(), ph.coo_beamlet.numpy(), ph.coo_val.numpy()
sid, T, wo, wu = ph.voxel_struct.numpy(), ph.struct_T.numpy(), ph.struct_w_over.numpy(), ph.struct_w_under.numpy()
aco, aro, lco = ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset
x = synth.draw_x(ph.n_beamlets, 5, scale=float(os.environ.get("VMAT_TEST_XSCALE", "14"))).numpy()
nnz_per_angle = np.bincount(np.searchsorted(aco.numpy(), beam, side="right") - 1, minlength=ph.n_angles)
offs = sharded.partition_angles(nnz_per_angle, world)
blk = sharded.local_block(aco, aro, lco, offs[rank], offs[rank + 1])
keep = (beam >= blk.beamlet_lo) & (beam < blk.beamlet_hi)
lbeam = (beam[keep] - blk.beamlet_lo).astype(np.int32)
n_b_local = blk.beamlet_hi - blk.beamlet_lo
# rank m: d_m = D_m x_m; all: d = sum_m d_m
d = torch.from_numpy(oracle.dose(vox[keep], lbeam, val[keep], ph.n_voxels, x[blk.beamlet_lo:blk.beamlet_hi]))
dist.all_reduce(d, op=dist.ReduceOp.SUM)
F, g = oracle.objective_grad(d.numpy(), sid, T, wo, wu)
p = oracle.price(vox[keep], lbeam, val[keep], n_b_local, g)
L, R, rp = oracle.select_rows(p.astype(np.float32), blk.leafrow_col_offset.numpy())
ap, lbest = oracle.angle_price(rp, blk.angle_row_offset.numpy())
# every rank's candidate {price, global control point}; the exchange is sharded.gather_pairs; the A5 rule over the
# gathered candidates (vmat_merge_best on a GPU) is stood in for by the oracle's O5 with one "control point" per rank
pair = torch.tensor([ap[lbest] if lbest >= 0 else 0.0, float(lbest + blk.angle_lo) if lbest >= 0 else -1.0], dtype=torch.float64)
pairs = sharded.gather_pairs(pair).numpy()
_, win = oracle.angle_price(pairs[:, 0].copy(), np.arange(world + 1, dtype=np.int32))
best, best_price = (int(pairs[win, 1]), float(pairs[win, 0])) if win >= 0 else (-1, 0.0)
# the unsharded evaluation
ev = oracle.price_eval(vox, beam, val, ph.n_voxels, ph.n_beamlets, x, sid, T, wo, wu, lco.numpy(), aro.numpy())
res = {
    "rank": rank, "offs": offs, "block": [blk.angle_lo, blk.angle_hi, blk.beamlet_lo, blk.beamlet_hi, blk.row_lo, blk.row_hi],
    "d_err": float(np.abs(d.numpy() - ev.d).max() / np.abs(ev.d).max()), "F_err": abs(F - ev.F) / abs(ev.F),
    "p_err": float(np.abs(p - ev.p[blk.beamlet_lo:blk.beamlet_hi]).max() / np.abs(ev.p).max()),
    "LR_equal": bool(np.array_equal(L, ev.L[blk.row_lo:blk.row_hi]) and np.array_equal(R, ev.R[blk.row_lo:blk.row_hi])),
    "ap_err": float(np.abs(ap - ev.angle_price[blk.angle_lo:blk.angle_hi]).max()),
    "best": best, "best_ref": ev.best_angle, "best_price": best_price,
    "best_price_ref": float(ev.angle_price[ev.best_angle]) if ev.best_angle >= 0 else 0.0,
    "nnz_local": int(keep.sum()), "nnz": int(beam.size),
}
dist.barrier()
if rank == 0:
    print(json.dumps(res))
else:
    with open(os.environ["VMAT_TEST_OUT"] + f".{rank}", "w") as f:
        json.dump(res, f)
dist.destroy_process_group()
