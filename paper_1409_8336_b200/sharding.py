"""History sharding over ranks: host-side plumbing only, no physics.

Histories are independent and the Philox stream is keyed by the global history id, so a run of N histories
splits into contiguous id ranges, one per rank (`history_offset` option of libpmc).  Each rank produces its own
mean dose (Gy per primary of ITS share) and standard error; the plan dose is their history-weighted mean:

    D     = sum_r n_r D_r / sum_r n_r
    sigma = sqrt( sum_r (n_r / N)^2 sigma_r^2 )

which needs one all-reduce(sum) of one packed buffer (two grids and the history count) — the only exchange step of the path (PAPER.md:L266, L270 mention
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
    """ONE all-reduce(sum) of a packed buffer [n_r D_r | (n_r sigma_r)^2 | n_r] turns the per-rank (dose, sigma) into the
    plan's: D = sum n_r D_r / N, sigma = sqrt(sum (n_r sigma_r)^2) / N.  In place; returns (dose, sigma, N).
    (n_r travels as two fp32 words of 16 bits each so that the sum over ranks is exact in the fp32 buffer.)"""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return dose, sigma, n_local
    nv = dose.numel()
    buf = torch.empty(2 * nv + 2, dtype=torch.float32, device=dose.device)
    torch.mul(dose.reshape(-1), float(n_local), out=buf[:nv])
    torch.mul(sigma.reshape(-1), float(n_local), out=buf[nv:2 * nv]); buf[nv:2 * nv].square_()
    buf[2 * nv] = float(n_local >> 16); buf[2 * nv + 1] = float(n_local & 0xFFFF)
    dist.all_reduce(buf, group=group)
    tail = buf[2 * nv:].tolist()
    n_tot = int(round(tail[0])) * 65536 + int(round(tail[1]))
    inv = 1.0 / n_tot if n_tot > 0 else 0.0
    dose.copy_((buf[:nv] * inv).reshape(dose.shape))
    sigma.copy_((buf[nv:2 * nv].sqrt_() * inv).reshape(sigma.shape))
    return dose, sigma, n_tot
