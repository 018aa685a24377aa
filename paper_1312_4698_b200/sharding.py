"""Trajectory sharding across ranks (the paper names multi-GPU as future work).

Trajectories are independent, so each rank runs the whole path on its own block of
trajectories with no data-path collective.  The only exchange is one sum of k + 1 doubles at the end:
Eq. 11's 1/n_good is per job, so a rank's spectrum I_r (normalised by its own n_good_r) is re-weighted,

    I = sum_r n_good_r I_r / sum_r n_good_r .

Host logic only (torch.distributed plumbing); covered by a world_size-2 gloo test on CPU.
"""
from __future__ import annotations


def shard_bounds(ntraj: int, rank: int, world: int):
    """Contiguous block [lo, hi) of trajectories for `rank`; sizes differ by at most one."""
    base, rem = divmod(int(ntraj), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def combine_shards(spectra, n_goods):
    """The same re-weighting without a process group: spectra[r] (normalised by n_goods[r]) of every shard, in rank order.
    Returns (I, n_good).  combine_spectra is this sum carried by one all-reduce."""
    import torch

    acc = torch.zeros_like(spectra[0])
    n_good = 0
    for I_r, n_r in zip(spectra, n_goods):  # fixed rank order
        acc = acc + I_r * float(n_r)
        n_good += int(n_r)
    if n_good == 0:
        return torch.zeros_like(spectra[0]), 0
    return acc / float(n_good), n_good


def combine_spectra(I_local, n_good_local: int, group=None):
    """All-reduce of (n_good_r * I_r, n_good_r): returns (I, n_good) of the whole job on every rank.

    I_local: 1-D float64 torch tensor (CPU for gloo, CUDA for nccl).  A rank with n_good_r = 0 contributes zero.
    """
    import torch
    import torch.distributed as dist

    buf = torch.empty(I_local.numel() + 1, dtype=torch.float64, device=I_local.device)
    buf[:-1] = I_local * float(n_good_local)
    buf[-1] = float(n_good_local)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(buf, op=dist.ReduceOp.SUM, group=group)
    n_good = int(round(buf[-1].item()))
    if n_good == 0:
        return torch.zeros_like(I_local), 0
    return buf[:-1] / buf[-1], n_good
