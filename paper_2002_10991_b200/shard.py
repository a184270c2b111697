"""Host-side logic of the multi-GPU path: eigenvector columns are independent
(PAPER.md:134, :138), so N GPUs each back-transform their own columns with a replicated reflector
stream -- no data-path collective; only the timing is reduced (max over ranks).  No arithmetic of
the method lives here."""
from __future__ import annotations


def column_shard(nev: int, rank: int, world: int, slab: int = 8):
    """Columns [col0, col0 + ncols) of rank ``rank`` when ``nev`` columns are split over ``world``
    ranks in units of ``slab`` columns (the kernels' DMMA granularity), as evenly as possible; the
    last non-empty shard takes the ragged tail.  Every column belongs to exactly one rank."""
    if world < 1 or not (0 <= rank < world) or nev < 0 or slab < 1:
        raise ValueError("bad shard arguments")
    nslab = (nev + slab - 1) // slab
    s0 = nslab * rank // world
    s1 = nslab * (rank + 1) // world
    col0 = min(s0 * slab, nev)
    col1 = min(s1 * slab, nev)
    return col0, col1 - col0


def max_over_ranks(value: float, dist=None, device: str = "cpu") -> float:
    """MAX all-reduce of one float (the timed interval); identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(flops_per_rank: float, world: int, max_seconds: float) -> float:
    """Whole-job FLOP/s of a weak-scaling run: every rank did ``flops_per_rank`` in ``max_seconds``."""
    return world * flops_per_rank / max_seconds
