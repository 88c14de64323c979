"""Cell-range sharding of the collision step across ranks.

Cells are independent units and the step needs no exchange, so a rank owns a contiguous
range of global cell ids and the particles sorted into them; weights and the chi table are
replicated.  The only arithmetic here is integer bookkeeping: which cells go where.  A rank passes
`cell_base = c0` in its parameter struct, so its Philox counters carry GLOBAL cell ids and the
sharded run draws exactly the randoms of the unsharded one (results are bit-identical).

`allreduce_diagnostics` is the one (optional) collective: a sum of per-rank scalars (total energy,
momentum, collided pairs) outside the data path.
"""
from __future__ import annotations

import numpy as np


def pairs_per_cell(counts: np.ndarray, pairs_req: int = -1) -> np.ndarray:
    """M_k = min(M_req, floor(N_k / 2)) (M_req = -1: floor(N_k / 2)); SURVEY 8(c) step 3."""
    half = np.asarray(counts, dtype=np.int64) // 2
    return half if pairs_req < 0 else np.minimum(half, pairs_req)


def partition_cells(counts: np.ndarray, world: int, pairs_req: int = -1) -> np.ndarray:
    """Split [0, K) into `world` contiguous ranges balanced by sum of M_k.

    Returns bounds[world + 1] with bounds[0] = 0, bounds[world] = K, non-decreasing; rank r owns
    cells [bounds[r], bounds[r + 1]).  Deterministic, identical on every rank."""
    if world < 1:
        raise ValueError("world must be >= 1")
    m = pairs_per_cell(counts, pairs_req)
    cum = np.concatenate([[0], np.cumsum(m)])
    total = int(cum[-1])
    K = len(m)
    bounds = np.zeros(world + 1, dtype=np.int64)
    bounds[world] = K
    for r in range(1, world):
        # first cell boundary whose pair prefix reaches r/world of the total
        bounds[r] = int(np.searchsorted(cum, (total * r + world - 1) // world, side="left"))
    return np.maximum.accumulate(np.minimum(bounds, K))


def shard_sorted(cell_start: np.ndarray, arrays, bounds: np.ndarray, rank: int):
    """Slice the cell-sorted arrays of a population for `rank`.

    Returns (cell_base, local_cell_start, [local arrays]); local_cell_start[0] = 0."""
    c0, c1 = int(bounds[rank]), int(bounds[rank + 1])
    q0, q1 = int(cell_start[c0]), int(cell_start[c1])
    local_cs = (np.asarray(cell_start[c0:c1 + 1], dtype=np.int64) - q0).astype(np.int32)
    return c0, local_cs, [np.ascontiguousarray(a[q0:q1]) for a in arrays]


def allreduce_diagnostics(values, group=None):
    """Sum a small vector of per-rank float64 diagnostics over the ranks (NCCL on GPUs, gloo on CPU)."""
    import torch
    import torch.distributed as dist
    t = torch.as_tensor(np.asarray(values, dtype=np.float64))
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        if dist.get_backend(group) == "nccl":
            t = t.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t.cpu().numpy()
