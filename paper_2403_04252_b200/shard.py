"""Data-parallel sharding of trajectories over ranks (impact parameters are
independent, "one rank per impact parameter").  Host logic only -- no arithmetic of the method.

The path has exactly one exchange step: the final amplitudes c(z_max) of every trajectory are gathered on all ranks
before wpccc_probabilities integrates the cross sections over b.  Everything before it is rank-local.
"""
from __future__ import annotations

import numpy as np


def shard_indices(n_traj: int, rank: int, world: int) -> np.ndarray:
    """Round-robin: rank r owns trajectories r, r + world, ...  (interleaves small and large b, whose cost differs)."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world of %d" % (rank, world))
    return np.arange(rank, n_traj, world, dtype=np.int64)


def shard_sizes(n_traj: int, world: int) -> list:
    return [len(range(r, n_traj, world)) for r in range(world)]


def gather_amplitudes(C_local, n_traj: int, rank: int, world: int, group=None):
    """all_gather of the per-rank amplitude blocks [n_local, N] (complex128 as a real view) into [n_traj, N] in the
    original trajectory order.  Works on any torch.distributed backend (NCCL on the GPUs, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist

    if world == 1:
        return C_local
    sizes = shard_sizes(n_traj, world)
    N = C_local.shape[1]
    n_max = max(sizes)
    send = torch.zeros((n_max, N, 2), dtype=torch.float64, device=C_local.device)
    if C_local.shape[0]:
        send[: C_local.shape[0]] = torch.view_as_real(C_local)
    recv = [torch.empty_like(send) for _ in range(world)]
    dist.all_gather(recv, send, group=group)
    out = torch.empty((n_traj, N, 2), dtype=torch.float64, device=C_local.device)
    for r in range(world):
        idx = torch.as_tensor(shard_indices(n_traj, r, world), device=C_local.device)
        if sizes[r]:
            out[idx] = recv[r][: sizes[r]]
    return torch.view_as_complex(out)
