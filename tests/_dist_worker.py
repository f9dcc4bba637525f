"""Worker of test_multi_rank_host_logic.py: run under torch.distributed.run with the gloo backend."""
import json
import os
import sys

import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
# every rank draws its own fluence sequence
idx = [bench.rank_eval_index(rank, k) for k in range(3)]
# max over ranks of the device time (here: fake per-rank times)
t = bench.reduce_max([10.0 + rank, 20.0 - rank], dist, torch.device("cpu"))
dist.barrier()
line = bench.aggregate(world, 50, t[0])
if rank == 0:
    print(json.dumps({"idx0": idx, "t": t, "value": line["value"], "ms_per_step": line["ms_per_step"]}))
else:
    # other ranks report their indices through a file so the test can check disjointness
    with open(os.environ["VMAT_TEST_OUT"] + f".{rank}", "w") as f:
        json.dump({"idx": idx}, f)
dist.destroy_process_group()
