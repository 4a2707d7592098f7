"""Axial scan (BASELINE.json config 4): D_scan = sum over source positions of D_p.

Source positions are independent problems, so the only multi-GPU decomposition this path has is by
position: rank r takes positions r, r + world, ...; one all-reduce(sum) of the dose
map at the end is the only exchange step. A single projection does not shard ("replicas only").
Host logic only; every arithmetic step runs in the CUDA library through `dos.Context`.
"""
from __future__ import annotations


def shard_positions(n_pos: int, rank: int, world: int):
    """Round-robin partition of positions 0..n_pos-1: disjoint, complete, sizes differ by at most 1."""
    if not (0 <= rank < world):
        raise ValueError("rank outside 0..world-1")
    return list(range(rank, n_pos, world))


def run_scan(ctx, problem, positions, dose, n_iter=None):
    """Runs the hot path for the listed positions on `ctx`, summing the dose maps into `dose` (device tensor
    [nz][ny][nx]); with no positions the map is zeroed. Positions go through the library ctx.n_batch at a time
    (dos_uncollided_batch: one set of sweep launches serves the whole batch). Only enqueues work."""
    n_iter = problem["n_iter"] if n_iter is None else n_iter
    if not positions:
        dose.zero_()
    nb = max(1, int(getattr(ctx, "n_batch", 1)))
    for n in range(0, len(positions), nb):
        chunk = [problem["sources"][s] for s in positions[n:n + nb]]
        if len(chunk) == 1:
            ctx.dos_uncollided(chunk[0], problem["spectrum"])
        else:
            ctx.dos_uncollided_batch(chunk, problem["spectrum"])
        ctx.dos_solve(n_iter)
        ctx.dos_dose(dose, accumulate=(n > 0))
    return dose


def all_reduce_dose(dose):
    """Sum of the ranks' partial dose maps (NCCL over NVLink on GPUs, gloo on CPU tensors); no-op when
    torch.distributed is not initialised."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(dose, op=dist.ReduceOp.SUM)
    return dose
