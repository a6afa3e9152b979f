"""Multi-GPU sharding of the sector tracker.

The 36 sectors are tracked "individually" and drift windows are independent, so the unit
of work is the sector instance and the path needs NO data-path collective: every rank tracks its own instances.
This module is host logic only (which instances a rank owns, how per-rank timings and counts are combined); it works
with any torch.distributed backend (nccl on the GPU box, gloo in the CPU tests).
"""
from __future__ import annotations

import numpy as np


def window_seeds(windows_per_rank: int, seed0: int, rank: int) -> list[int]:
    """Weak scaling: rank r generates and tracks windows seed0 + r*W ... seed0 + (r+1)*W - 1 (disjoint across ranks)."""
    return [seed0 + rank * windows_per_rank + i for i in range(windows_per_rank)]


def partition_instances(row_offsets: np.ndarray, n_inst: int, n_rows: int, world: int, rank: int, unit: int = 36):
    """Strong-scaling split of one job: contiguous blocks of `unit` instances (one event/window = 36 sectors), blocks
    dealt to ranks so that cluster counts are balanced (greedy prefix split on the cumulative cluster count).

    Returns (inst0, n_inst_local, cluster0, n_clusters_local).  Ranks beyond the number of blocks get empty ranges."""
    n_blocks = -(-n_inst // unit)
    ends = np.array([int(row_offsets[min((b + 1) * unit, n_inst) * n_rows]) for b in range(n_blocks)], dtype=np.int64)
    total = int(ends[-1]) if n_blocks else 0
    # block boundary k_r = first block index whose cumulative end reaches r/world of the clusters
    cuts = [0]
    for r in range(1, world):
        target = total * r / world
        k = int(np.searchsorted(ends, target, side="left")) + 1 if n_blocks else 0
        k = min(max(k, cuts[-1]), n_blocks)
        cuts.append(k)
    cuts.append(n_blocks)
    b0, b1 = cuts[rank], cuts[rank + 1]
    inst0, inst1 = min(b0 * unit, n_inst), min(b1 * unit, n_inst)
    c0, c1 = int(row_offsets[inst0 * n_rows]), int(row_offsets[inst1 * n_rows])
    return inst0, inst1 - inst0, c0, c1 - c0


def local_problem(clusters: np.ndarray, row_offsets: np.ndarray, n_rows: int, inst0: int, n_inst_local: int):
    """The rank's slice of a job as a self-contained tracker input (row offsets rebased to 0)."""
    ro = row_offsets[inst0 * n_rows:(inst0 + n_inst_local) * n_rows + 1]
    c0 = int(ro[0])
    return clusters[c0:int(ro[-1])], (ro - c0).astype(np.int32)


def combine_step(ms_local: float, units_local: int, device=None):
    """(max over ranks of the step time, total units over ranks) -- the bench contract's whole-job aggregate.
    Without an initialised process group this is the identity."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), int(units_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    n = torch.tensor([int(units_local)], dtype=torch.int64, device=device)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t.item()), int(n.item())


def gather_counts(counts_local: np.ndarray, device=None) -> np.ndarray:
    """Per-rank tpc counts[] -> [world, n] on every rank (the only thing a consumer needs to place per-rank track
    lists into one job-wide numbering: track base of rank r = sum of n_tracks of ranks < r)."""
    import torch
    import torch.distributed as dist
    c = torch.as_tensor(np.asarray(counts_local, dtype=np.int64), device=device)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return c.cpu().numpy()[None, :]
    out = [torch.empty_like(c) for _ in range(dist.get_world_size())]
    dist.all_gather(out, c)
    return torch.stack(out).cpu().numpy()
