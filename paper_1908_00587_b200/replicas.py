"""Host-side plumbing of multi-GPU runs (the path does not shard in v1, so N GPUs run N
independent replicas -- one process per GPU, no data-path collective).  Only bookkeeping lives here: the
per-rank seed, the barrier, and the max-over-ranks reduction of a device-measured time.  Works with any
``torch.distributed`` backend (NCCL on GPUs; gloo in the CPU tests)."""
from __future__ import annotations


def rank_config(cfg: dict, rank: int) -> dict:
    """The replica of ``rank``: same physics and sizes, its own seeded synthetic state."""
    return dict(cfg, seed=cfg["seed"] + 1000 * rank)


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX all-reduce of a per-rank scalar (a time measured on the device); identity without a group."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(world: int, units_per_rank: float, seconds_max: float) -> float:
    """Whole-job throughput: every rank processed ``units_per_rank`` units in at most ``seconds_max``."""
    return world * units_per_rank / seconds_max
