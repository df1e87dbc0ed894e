"""Multi-GPU host logic: block lists shard by independent blocks, one all-gather.
world_size-2 gloo on CPU; the projector is a stand-in (the oracle), since only the partition /
gather logic is under test here."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_20519_b200.sharding import assign_blocks, project_sharded


def test_assign_blocks_balances_by_cube():
    sizes = [1296, 2401] + [36] * 64
    owned = assign_blocks(sizes, 2)
    assert sorted(owned[0] + owned[1]) == list(range(len(sizes)))
    assert 1 in owned[0] and 0 in owned[1]            # largest first, then the other rank
    load = [sum(sizes[b] ** 3 for b in o) for o in owned]
    assert load[1] <= load[0]
    assert all(b in owned[1] for b in range(2, 66))   # small ones fill the lighter rank
    assert assign_blocks([], 4) == [[], [], [], []]
    assert assign_blocks([5], 3) == [[0], [], []]


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, sizes, sv, want):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle

    def projector(szs, t):
        return torch.from_numpy(oracle.project(list(szs), t.numpy()))

    out = project_sharded(sizes, torch.from_numpy(sv), projector=projector)
    assert np.array_equal(out.numpy(), want), rank
    dist.destroy_process_group()


def test_project_sharded_gloo_world2(orc):
    rng = np.random.default_rng(3)
    sizes = [12, 5, 1, 9, 0, 7]
    mats = []
    for n in sizes:
        g = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
        mats.append(0.5 * (g + g.conj().T))
    sv = np.concatenate([orc.pack(m) for m in mats])
    want = orc.project(sizes, sv)
    mp.spawn(_worker, args=(2, _free_port(), sizes, sv, want), nprocs=2, join=True)
