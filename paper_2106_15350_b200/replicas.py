"""Host logic of the multi-GPU ("replicas only") mode: candidates are independent (one trial per
kernel set), `north_star` rules out sharding one search over GPUs, so every rank searches its OWN batch of candidate
kernel sets on the same images.  The only collectives are the timing barrier and a max over ranks; no arithmetic of
the method lives here.  Works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations


def first_candidate(rank: int, n_cand_per_rank: int) -> int:
    """index of the first candidate kernel set of `rank` in the global stream of seeded kernel sets."""
    if rank < 0 or n_cand_per_rank < 1:
        raise ValueError("rank >= 0 and n_cand_per_rank >= 1 required")
    return rank * n_cand_per_rank


def max_over_ranks(value: float, device=None) -> float:
    """max of a per-rank scalar over all ranks (the job's time is its slowest rank's); identity without a group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(world: int, n_cand_per_rank: int, steps: int, seconds_max_over_ranks: float) -> float:
    """whole-job candidates/s: all ranks' candidates over the slowest rank's time (weak scaling)."""
    return world * n_cand_per_rank * steps / seconds_max_over_ranks


def global_best(acc_best: float, index_best: int, rank: int, n_cand_per_rank: int, device=None):
    """(accuracy, global candidate index) of the best candidate over all ranks; ties -> lowest global index
    (R13).  Every rank passes its local best; returns the same pair on every rank."""
    import torch
    import torch.distributed as dist
    g = first_candidate(rank, n_cand_per_rank) + int(index_best)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(acc_best), g
    world = dist.get_world_size()
    mine = torch.tensor([float(acc_best), float(g)], dtype=torch.float64, device=device if device is not None else "cpu")
    allv = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(allv, mine)
    best = max(allv, key=lambda t: (float(t[0]), -float(t[1])))
    return float(best[0]), int(best[1])
