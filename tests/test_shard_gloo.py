"""-m "not gpu": the N > 1 path (trajectory sharding + the one exchange step, the all-gather of the final amplitudes)
on two gloo ranks on the CPU.  SURVEY.md 8(e); PAPER.md L106 (impact parameters are independent)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2403_04252_b200.shard import gather_amplitudes, shard_indices, shard_sizes


def test_round_robin_partition_is_exact():
    for n in (0, 1, 5, 16, 33):
        for world in (1, 2, 3, 8):
            idx = [shard_indices(n, r, world) for r in range(world)]
            assert sorted(np.concatenate(idx).tolist()) == list(range(n))
            assert [len(i) for i in idx] == shard_sizes(n, world)
    with pytest.raises(ValueError):
        shard_indices(4, 2, 2)


def _worker(rank, world, port, n_traj, N, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    full = torch.arange(n_traj * N, dtype=torch.float64).reshape(n_traj, N)
    full = torch.complex(full, -0.5 * full)
    mine = torch.as_tensor(shard_indices(n_traj, rank, world))
    got = gather_amplitudes(full[mine].clone(), n_traj, rank, world)
    q.put((rank, bool(torch.equal(got, full))))
    dist.destroy_process_group()


@pytest.mark.parametrize("n_traj", [5, 16])
def test_gather_amplitudes_two_gloo_ranks(n_traj):
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, n_traj, 7, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
    assert res == [(0, True), (1, True)]
