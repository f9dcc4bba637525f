"""Angle-sharded price evaluation over several GPUs (NEXT-4).

The DDC matrix is split by control point into column blocks D = [D_1 ... D_M] (L119), one block per rank; every rank
holds both layouts of its block.  One evaluation:

    rank m:   d_m = D_m x_m                              vmat_dose            (its own beamlets only)
    all:      d = sum_m d_m                              all-reduce(sum), n_voxels floats   <- the one exchange step
    rank m:   F, g = objective(d)                        vmat_objective_grad  (redundantly on every rank, as in L127)
    rank m:   p_m = D_m^T g, row openings, aperture      vmat_price_select    (its own control points only)
              prices of its control points
    all:      best control point                         all-gather of one (price, control point) pair per rank

In the paper this exchange is the broadcast of z over a P2P tree and the gather of the prices to GPU 1 (L127);
here it is NCCL over NVLink (a 5 MB all-reduce next to two kernels that stream tens of GB).  Everything numerical runs
in the library's kernels; this module only partitions the control points, re-bases the offset tables and calls
torch.distributed; the A5 rule over the gathered candidates runs on the device too (vmat_best_pair, vmat_merge_best), so
an evaluation never synchronises with the host.  With no process group (one rank) the collectives are skipped and the
result is the unsharded one.

`north_star` fixes one GPU for the hot path, so the bench's default for N > 1 stays "replicas only"; this path is for
matrices beyond one GPU (`bench.py --parallelism angle-shards`).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Optional, Sequence

import torch

from . import (DDC, Objective, PriceEvalOut, last_launch_count, vmat_best_pair, vmat_ddc_create, vmat_dose, vmat_merge_best,
               vmat_objective_grad, vmat_price_select)


def partition_angles(weight_per_angle: Sequence[float], world: int) -> List[int]:
    """Contiguous blocks of control points, one per rank, balanced by `weight_per_angle` (non-zeros, or beamlets, of
    every control point): boundary m is the first control point at which the running weight reaches m/world of the
    total.  Returns world+1 offsets; blocks may be empty when world > number of control points."""
    w = [float(v) for v in weight_per_angle]
    n, total = len(w), float(sum(w))
    offs, acc, k = [0], 0.0, 0
    for m in range(1, world):
        target = total * m / world
        while k < n and acc + w[k] * 0.5 < target:
            acc += w[k]
            k += 1
        offs.append(k)
    offs.append(n)
    return offs


@dataclass
class LocalBlock:
    """Offset tables of one rank's column block, re-based to start at 0."""
    angle_lo: int
    angle_hi: int
    beamlet_lo: int
    beamlet_hi: int
    row_lo: int
    row_hi: int
    angle_col_offset: torch.Tensor      # int32 [n_local_angles + 1]
    angle_row_offset: torch.Tensor
    leafrow_col_offset: torch.Tensor    # int32 [n_local_rows + 1]


def local_block(angle_col_offset: torch.Tensor, angle_row_offset: torch.Tensor, leafrow_col_offset: torch.Tensor,
                angle_lo: int, angle_hi: int) -> LocalBlock:
    aco, aro, lco = (t.to(torch.int64).cpu() for t in (angle_col_offset, angle_row_offset, leafrow_col_offset))
    b0, b1 = int(aco[angle_lo]), int(aco[angle_hi])
    r0, r1 = int(aro[angle_lo]), int(aro[angle_hi])
    return LocalBlock(angle_lo, angle_hi, b0, b1, r0, r1,
                      (aco[angle_lo:angle_hi + 1] - b0).to(torch.int32),
                      (aro[angle_lo:angle_hi + 1] - r0).to(torch.int32),
                      (lco[r0:r1 + 1] - b0).to(torch.int32))


def gather_pairs(pair: torch.Tensor, group=None) -> torch.Tensor:
    """All-gather of one candidate pair {aperture price, global control point} (float64 [2]) per rank -> [world, 2] on
    the pair's device (CUDA for NCCL, CPU for gloo).  Communication only; one rank without a process group: [1, 2]."""
    import torch.distributed as dist
    if group is None and not (dist.is_available() and dist.is_initialized()):
        return pair.reshape(1, 2)
    world = dist.get_world_size(group)
    pairs = torch.empty(world * 2, dtype=torch.float64, device=pair.device)
    dist.all_gather_into_tensor(pairs, pair.contiguous(), group=group)
    return pairs.reshape(world, 2)


def merge_best(pair: torch.Tensor, group=None) -> torch.Tensor:
    """Best control point over all ranks from every rank's candidate pair (device float64 [2], from vmat_best_pair):
    one all-gather, then the A5 rule on the device (vmat_merge_best).  Returns a device float64 [2] = {price, global
    control point or -1}; nothing comes to the host."""
    pairs = gather_pairs(pair, group)
    best = torch.empty(2, dtype=torch.float64, device=pair.device)
    vmat_merge_best(pairs.contiguous(), best)
    return best


def best_to_host(best: torch.Tensor) -> tuple:
    """(global control point or -1, its aperture price) from the device pair; this is the synchronising read."""
    p, k = best.cpu().tolist()
    return int(k), float(p)


class ShardedDDC:
    """One rank's column block of D plus the two collectives of an evaluation."""

    def __init__(self, handle: DDC, block: LocalBlock, n_angles_total: int, n_beamlets_total: int, group=None):
        self.h, self.block, self.group = handle, block, group
        self.n_angles_total, self.n_beamlets_total = n_angles_total, n_beamlets_total
        self.n_voxels = handle.n_voxels
        self._pair = None
        self.last_launches = 0

    @classmethod
    def create(cls, n_voxels: int, n_beamlets: int, coo_voxel: torch.Tensor, coo_beamlet: torch.Tensor,
               coo_val: torch.Tensor, angle_col_offset: torch.Tensor, angle_row_offset: torch.Tensor,
               leafrow_col_offset: torch.Tensor, angle_lo: int, angle_hi: int, device=None, index_bits: int = 0,
               group=None) -> "ShardedDDC":
        """Builds this rank's handle from COO triplets in GLOBAL beamlet numbering; triplets of other ranks' control
        points are dropped, so the caller may pass the whole matrix or only its own block."""
        blk = local_block(angle_col_offset, angle_row_offset, leafrow_col_offset, angle_lo, angle_hi)
        keep = (coo_beamlet >= blk.beamlet_lo) & (coo_beamlet < blk.beamlet_hi)
        if not bool(keep.all()):
            coo_voxel, coo_beamlet, coo_val = coo_voxel[keep], coo_beamlet[keep], coo_val[keep]
        local_beamlet = (coo_beamlet - blk.beamlet_lo).to(torch.int32)
        h = vmat_ddc_create(n_voxels, blk.beamlet_hi - blk.beamlet_lo, coo_voxel.contiguous(), local_beamlet.contiguous(),
                            coo_val.contiguous(), blk.angle_col_offset, blk.angle_row_offset, blk.leafrow_col_offset,
                            device=device, index_bits=index_bits)
        return cls(h, blk, int(angle_col_offset.numel()) - 1, int(n_beamlets), group)

    def _dist(self):
        import torch.distributed as dist
        return dist if (dist.is_available() and dist.is_initialized()) else None

    def price_eval(self, x_local: torch.Tensor, obj: Objective, out: PriceEvalOut,
                   angle_mask_local: Optional[torch.Tensor] = None):
        """One evaluation; `x_local` and the beamlet / leaf-row / control-point outputs in `out` are this rank's block
        (local numbering), d, g and F are the global ones.  Returns a device float64 [2] = {aperture price, best control
        point in global numbering or -1} after the second exchange; no host synchronisation (`best_to_host` reads it)."""
        dist = self._dist()
        vmat_dose(self.h, x_local, out.d)
        n = last_launch_count()
        if dist is not None:
            dist.all_reduce(out.d, op=dist.ReduceOp.SUM, group=self.group)          # d = sum_m D_m x_m
        vmat_objective_grad(self.h, out.d, obj, out.g, out.F)
        n += last_launch_count()
        vmat_price_select(self.h, out.g, out, angle_mask_local)
        n += last_launch_count()
        if self._pair is None:
            self._pair = torch.empty(2, dtype=torch.float64, device=out.d.device)
        vmat_best_pair(self.h, out, self.block.angle_lo, self._pair)
        n += last_launch_count()
        best = merge_best(self._pair, self.group)
        self.last_launches = n + last_launch_count()         # libvmat kernels of this evaluation (vmat_last_launch_count)
        return best

    def close(self):
        self.h.close()
