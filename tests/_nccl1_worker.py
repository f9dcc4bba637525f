"""Worker of test_gpu_sharded.py::test_collective_path_on_one_gpu_with_nccl: one rank, backend nccl.  The process group
is real, so ShardedDDC.price_eval takes its collective path (all-reduce of d, all-gather of the candidates)."""
import json
import os
import sys

import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import synth
import paper_1503_01721_b200 as vm
from paper_1503_01721_b200 import sharded

vm.load_library()
torch.cuda.set_device(0)
dev = torch.device("cuda:0")
dist.init_process_group("nccl", device_id=dev)
calls = {"n": 0}
for name in ("all_reduce", "all_gather_into_tensor"):            # count the collectives price_eval issues
    orig = getattr(dist, name)

    def wrap(*a, _o=orig, **k):
        calls["n"] += 1
        return _o(*a, **k)
    setattr(dist, name, wrap)
ph = synth.generate(synth.config_spec(0))
sh = sharded.ShardedDDC.create(ph.n_voxels, ph.n_beamlets, ph.coo_voxel.to(dev), ph.coo_beamlet.to(dev), ph.coo_val.to(dev),
                               ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset, 0, ph.n_angles, device=dev)
obj = vm.Objective(ph.voxel_struct.to(dev), ph.struct_T.to(dev), ph.struct_w_over.to(dev), ph.struct_w_under.to(dev))
x = synth.draw_x(ph.n_beamlets, 2, device=dev, scale=14.0)
out, ref = sh.h.alloc_outputs(), sh.h.alloc_outputs()
best, price = sharded.best_to_host(sh.price_eval(x, obj, out))
vm.vmat_price_eval(sh.h, x, obj, ref)
torch.cuda.synchronize()
equal = all(torch.equal(getattr(out, n), getattr(ref, n)) for n in ("d", "g", "F", "p", "L", "R", "row_price", "angle_price", "best_angle"))
b = int(ref.best_angle.item())
print(json.dumps({"backend": dist.get_backend(), "world": dist.get_world_size(), "collectives_ran": calls["n"], "equal": equal,
                  "best": best, "price": price, "best_ref": b, "price_ref": float(ref.angle_price[b].item()) if b >= 0 else 0.0}))
sh.close()
dist.destroy_process_group()
