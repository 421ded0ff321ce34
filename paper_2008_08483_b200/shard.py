"""Cell sharding for N > 1 GPUs: one process per GPU, contiguous slices of cells, NO collective
on the data path (cells are independent: PAPER.md:9, 37, 66, 235).

Only host-side arithmetic lives here; `torch.distributed` is used for the timing reduction
(max over ranks) and nothing else.
"""
from __future__ import annotations


def cell_slice(n_total: int, rank: int, world: int) -> tuple[int, int]:
    """[lo, hi) of the cells rank `rank` owns out of n_total: contiguous, sizes differ by at
    most one, earlier ranks take the larger shares.  SoA columns are sliced by offset
    (T[lo:hi], P[lo:hi], Y[:, lo:hi])."""
    if world < 1 or not 0 <= rank < world or n_total < 0:
        raise ValueError("bad shard request: n_total=%d rank=%d world=%d" % (n_total, rank, world))
    base, extra = divmod(n_total, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def rank_cells(n: int, rank: int, world: int, scaling: str = "weak") -> tuple[int, int, int, int]:
    """What rank `rank` works on, as (n_generate, lo, hi, seed_offset): it draws n_generate cells
    with its state seed offset by seed_offset and keeps [lo, hi).
      "weak":   every rank has its own n cells (a different seeded batch per rank: the paper's
                "MPI rank offloads ... a given number of cells");
      "strong": ONE seeded batch of n cells in all, rank r takes cell_slice(n, r, world) of it
                (contiguous slices of N/G cells, SoA columns by offset).
    No collective on the data path in either mode."""
    if scaling == "weak":
        if world < 1 or not 0 <= rank < world or n < 0:
            raise ValueError("bad shard request: n=%d rank=%d world=%d" % (n, rank, world))
        return n, 0, n, rank
    if scaling == "strong":
        lo, hi = cell_slice(n, rank, world)
        return n, lo, hi, 0
    raise ValueError("scaling must be 'weak' or 'strong', got %r" % (scaling,))


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of a scalar (the multi-GPU timing rule); identity without a group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
