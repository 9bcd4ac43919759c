"""Host logic of the N > 1 path (replicas only).

The independent unit of the paper's workload is the right-hand side: a propagator is 12 columns, one per
(spin, colour) point source ("12 columns"; reading C13: column = 3*spin + colour). With N ranks every
rank owns a full context built from the same seeded gauge field and takes the columns dealt to it round-robin;
there is no data-path collective. This module holds only that dealing and the max-over-ranks reduction of a
device time (the one thing torch.distributed is used for besides the barrier).
"""
from __future__ import annotations

N_COLUMNS = 12


def columns_for_rank(rank: int, world: int, n_columns: int = N_COLUMNS) -> list[int]:
    """Columns (3*spin + colour) solved by `rank` of `world`: rank, rank + world, ... With world > n_columns the
    surplus ranks repeat columns (rank mod n_columns) so that every replica has work (weak scaling)."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError(f"bad rank/world {rank}/{world}")
    cols = list(range(rank, n_columns, world))
    return cols if cols else [rank % n_columns]


def spin_colour(column: int) -> tuple[int, int]:
    if not 0 <= column < N_COLUMNS:
        raise ValueError(f"column {column} out of range")
    return divmod(column, 3)


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """max of a per-rank scalar (device-timed milliseconds) over all ranks; identity without a process group."""
    if dist is None or not dist.is_initialized():
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
