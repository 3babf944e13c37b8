"""History sharding over ranks: host-side plumbing only, no physics.

Histories are independent and the Philox stream is keyed by the global history id, so a run of N histories
splits into contiguous id ranges, one per rank (`history_offset` option of libpmc).  Each rank produces its own
mean dose (Gy per primary of ITS share) and standard error; the plan dose is their history-weighted mean:

    D     = sum_r n_r D_r / sum_r n_r
    sigma = sqrt( sum_r (n_r / N)^2 sigma_r^2 )

which needs one all-reduce(sum) of two grids — the only exchange step of the path (PAPER.md:L266, L270 mention
multi-GPU only as deployment).  Works on CPU tensors over gloo (tests) and CUDA tensors over NCCL (bench).
"""
from __future__ import annotations


def shard_histories(n_total: int, rank: int, world: int):
    """Contiguous split of history ids [0, n_total) -> (offset, count) of `rank`; counts differ by at most 1."""
    if world < 1 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n_total, world)
    count = base + (1 if rank < rem else 0)
    offset = rank * base + min(rank, rem)
    return offset, count


def weak_shard(n_per_rank: int, rank: int):
    """Weak scaling: every rank runs n_per_rank histories with disjoint global ids."""
    return rank * n_per_rank, n_per_rank


def combine_dose(dose, sigma, n_local: int, group=None):
    """All-reduce the per-rank (dose, sigma) into the plan's (dose, sigma).  In place; returns (dose, sigma, N)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return dose, sigma, n_local
    n = torch.tensor([float(n_local)], dtype=torch.float64, device=dose.device)
    dist.all_reduce(n, group=group)
    n_tot = float(n.item())
    w = n_local / n_tot if n_tot > 0 else 0.0
    dose.mul_(w)
    sigma.mul_(w).square_()
    dist.all_reduce(dose, group=group)
    dist.all_reduce(sigma, group=group)
    sigma.sqrt_()
    return dose, sigma, int(round(n_tot))
