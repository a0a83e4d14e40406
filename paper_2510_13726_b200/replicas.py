"""N > 1: replicas only.  The path does not shard (BASELINE.json north_star: one GPU, no
decomposition, no collectives; the paper's own weak-scaling layout is one rotor per GPU,
PAPER.md:421).  Each rank steps an independent lattice; the only cross-rank traffic is the
barrier and the max-over-ranks reduction of the timed region."""
from __future__ import annotations


def max_over_ranks(ms_local: float, device=None) -> float:
    """Max of a per-rank duration over all ranks (identity without an initialised process group)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local)
    t = torch.tensor([ms_local], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_mlups(cells_per_rank: int, steps: int, ms_max: float, world: int) -> float:
    """Whole-job throughput: the units all ranks processed / the slowest rank's time."""
    return world * cells_per_rank * steps / (ms_max * 1e3)
