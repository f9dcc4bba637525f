"""Run structure of the secondary indices of the two stored layouts (host-side count, no GPU).

    python -m synth.index_runs [--config 3] [--angles 12] [--scale 1.0]

Question: the layouts store 2.125 B of index per entry (u16 offset + one int32 base
per 32 entries) next to the 4 B value.  The indices come in runs (a beamlet's voxels are x-runs of a raster line; a
voxel's beamlets are patches, contiguous in the tiled column order of CSR(D)).  Would a run-aware encoding - per group of
32 consecutive entries of a row a 32-bit break mask plus the start of every run - be smaller, and by how much?

Counted on the synthetic triplets of `--angles` evenly spaced control points of the config (rows of D^T belong to one
control point, so for D^T the sample is exact per row; a row of D holds one patch per control point, so the sample has
the patches of the sampled control points back to back: the same runs, cut into groups of 32 at other places).
Restates, for the count only, the tiled column order of CSR(D) (csrc/api.cu: per control point, tiles of 8 columns x all
leaf rows).  Prints one JSON object; profiles/r3_index_runs.md holds the output and what follows from it."""
from __future__ import annotations

import argparse
import json

import numpy as np

import synth

GROUP, TILE_GROUPS, COL_TILE = 32, 8, 8


def tiled_column_order(aco, aro, lco):
    """perm[j] = position of beamlet j in the column order of CSR(D)."""
    perm = np.arange(int(aco[-1]), dtype=np.int64)
    for a in range(len(aco) - 1):
        ra, rb = int(aro[a]), int(aro[a + 1])
        j0, j1 = int(aco[a]), int(aco[a + 1])
        if j1 == j0:
            continue
        j = np.arange(j0, j1)
        r = np.searchsorted(lco[ra:rb + 1], j, side="right") - 1           # leaf row within the control point
        c = j - lco[ra + r]
        key = (c // COL_TILE) * ((rb - ra) * COL_TILE) + r * COL_TILE + c % COL_TILE
        perm[j0 + np.argsort(key, kind="stable")] = j0 + np.arange(j1 - j0)
    return perm


def run_stats(row, idx):
    """row, idx: the entries of a layout sorted by (row, idx).  Groups of 32 consecutive entries of a row."""
    n = row.size
    new_row = np.ones(n, bool)
    new_row[1:] = row[1:] != row[:-1]
    row_start = np.flatnonzero(new_row)
    pos = np.arange(n) - np.repeat(row_start, np.diff(np.append(row_start, n)))
    brk = np.ones(n, bool)                                                    # entry starts a run
    brk[1:] = (idx[1:] != idx[:-1] + 1) | new_row[1:]
    run_start_pos = np.flatnonzero(brk)
    run_len = np.diff(np.append(run_start_pos, n))
    brk_g = brk | (pos % GROUP == 0)                                          # a group boundary cuts a run
    new_group = new_row | (pos % GROUP == 0)
    gid = np.cumsum(new_group) - 1
    runs_per_group = np.bincount(gid, weights=brk_g).astype(np.int64)
    n_groups = runs_per_group.size
    new_tile = new_row | (pos % (GROUP * TILE_GROUPS) == 0)
    tid_of_group = (np.cumsum(new_tile) - 1)[np.flatnonzero(new_group)]
    n_tiles = int(tid_of_group[-1]) + 1
    hist = np.bincount(np.minimum(runs_per_group, 33), minlength=34)
    out = {
        "entries": int(n), "rows": int(row_start.size), "groups_of_32": int(n_groups), "tiles_of_256": n_tiles,
        "runs": int(run_len.size), "mean_run_length": float(n / run_len.size),
        "entries_in_runs_of_at_least_8": float(run_len[run_len >= 8].sum() / n),
        "mean_runs_per_group": float(runs_per_group.mean()),
        "groups_with_at_most": {str(k): float((runs_per_group <= k).mean()) for k in (1, 2, 3, 4, 6, 8, 12, 16)},
        "histogram_runs_per_group": {str(k): int(v) for k, v in enumerate(hist) if v and k > 0},
        "stored_now_index_bytes_per_entry": 2.125,
    }
    # candidate encodings, index bytes per stored entry (the 4 B value comes on top)
    enc = {"variable: mask + int32 start per run": float((4 + 4 * runs_per_group).sum() / (GROUP * n_groups)),
           "variable: mask + u16 start per run + int32 base per tile": float(
               (4 + 2 * runs_per_group).sum() / (GROUP * n_groups) + 4.0 / (GROUP * TILE_GROUPS))}
    for K in (1, 2, 3, 4, 6, 8):
        bad_groups = runs_per_group > K
        tile_bad = np.bincount(tid_of_group, weights=bad_groups, minlength=n_tiles) > 0
        ok = 1.0 - float(tile_bad.mean())
        for name, hdr in (("int32", 4 + 4 * K), ("u16 + tile base", 4 + 2 * K + 0.5)):
            enc[f"fixed: mask + {K} {name} starts per group, u16 fallback per tile"] = \
                ok * hdr / GROUP + (1.0 - ok) * 2.125
        enc[f"tiles with every group <= {K} runs"] = ok
    out["candidate_index_bytes_per_entry"] = enc
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--angles", type=int, default=12)
    ap.add_argument("--scale", type=float, default=1.0)
    args = ap.parse_args()
    spec = synth.config_spec(args.config, args.scale)
    n_a = spec.n_angles
    k = min(args.angles, n_a)
    angles = sorted(set(int(round(i * n_a / k)) % n_a for i in range(k)))
    ph = synth.generate(spec, device="cpu", angles=angles)
    vox = ph.coo_voxel.numpy().astype(np.int64)
    beam = ph.coo_beamlet.numpy().astype(np.int64)
    aco, aro, lco = (t.numpy().astype(np.int64) for t in (ph.angle_col_offset, ph.angle_row_offset, ph.leafrow_col_offset))
    res = {"workload": spec.name, "control_points_sampled": angles, "of": n_a, "nnz_sampled": int(vox.size)}
    o = np.lexsort((vox, beam))                                               # CSR(D^T): rows = beamlets, index = voxel
    res["csr_dt (rows = beamlets, index = voxel)"] = run_stats(beam[o], vox[o])
    col = tiled_column_order(aco, aro, lco)[beam]
    o = np.lexsort((col, vox))                                                # CSR(D): rows = voxels, index = tiled column
    res["csr_d (rows = voxels, index = beamlet in the tiled column order)"] = run_stats(vox[o], col[o])
    o = np.lexsort((beam, vox))
    res["csr_d, caller's column order (for comparison)"] = run_stats(vox[o], beam[o])
    print(json.dumps(res, indent=1))


if __name__ == "__main__":
    main()
