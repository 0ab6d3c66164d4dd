"""Multi-GPU plumbing: rays are independent ("large ensemble of independent problems"; the paper's own
multi-device run splits the ensemble, L195), so ranks trace disjoint ray batches and the data path has NO collective.
The only communication is bookkeeping: a barrier and a max-over-ranks of the timed interval.
No arithmetic of the method lives here."""
from __future__ import annotations


def ray_range(n_rays: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous partition of [0, n_rays) into `world` ranges whose sizes differ by at most one ray (strong scaling of
    one ensemble).  Returns (begin, end) for `rank`."""
    if world < 1 or not (0 <= rank < world) or n_rays < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, n_rays >= 0")
    base, rem = divmod(n_rays, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def rank_seed(base_seed: int, rank: int) -> int:
    """Seed of rank `rank`'s own batch when every rank traces a full-size batch (weak scaling, bench.py)."""
    return int(base_seed) + 7919 * int(rank)


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of a host scalar over the default process group (a no-op without a group)."""
    if dist is None or not dist.is_initialized():
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, dist=None, device=None) -> float:
    if dist is None or not dist.is_initialized():
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
