"""The exchanges of the sharded lattice (paper_1210_8018_b200/sharded.py) on CPU: the
torch.distributed plumbing under gloo with world_size 2 and 4 must move the same data as the in-process
reference (LocalComm), in particular with 2 ranks, where the lower and the upper neighbour are the same peer.
No GPU, no liblgf compute."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1210_8018_b200 import sharded


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_data(world, r, n=6, h=5):
    """Distinct numbers everywhere: block q of rank r, its two halo messages."""
    blocks = torch.arange(world * n, dtype=torch.float64).view(world, n) + 1000.0 * r
    to_lower = torch.arange(h, dtype=torch.float64) + 100.0 * r + 0.25
    to_upper = torch.arange(h, dtype=torch.float64) + 100.0 * r + 0.75
    # complex, as the fields and links are: the transport must not depend on the element type
    return torch.complex(blocks, -blocks), torch.complex(to_lower, to_upper), torch.complex(to_upper, to_lower)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        comm = sharded.TorchDistComm()
        assert comm.world == world and comm.local_ranks == [rank]
        res = sharded.exchange_selftest(comm, world, [_rank_data(world, rank)])[0]
        out[rank] = tuple(t.clone() for t in res)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4])
def test_torch_dist_exchanges_equal_the_in_process_reference(world):
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        got = {r: out[r] for r in range(world)}
    ref = sharded.exchange_selftest(sharded.LocalComm(world), world, [_rank_data(world, r) for r in range(world)])
    for r in range(world):
        for a, b in zip(got[r], ref[r]):
            assert torch.equal(a, b)


def test_in_process_reference_is_what_the_layout_needs():
    """all_to_all: rank r receives block r of every rank q, in rank order (the transposed field is
    [source = t range][...]); halo: from_upper = upper neighbour's to_lower, from_lower = lower neighbour's to_upper."""
    world = 4
    data = [_rank_data(world, r) for r in range(world)]
    ref = sharded.exchange_selftest(sharded.LocalComm(world), world, data)
    for r in range(world):
        recv, fu, fl, tot = ref[r]
        for q in range(world):
            assert torch.equal(recv[q], data[q][0][r])
        assert torch.equal(fu, data[(r + 1) % world][1]) and torch.equal(fl, data[(r - 1) % world][2])
        assert tot.item() == sum(d[0].real.sum().item() for d in data)


def test_slab_of_takes_whole_time_slices():
    import numpy as np

    N = (4, 4, 2, 8)
    V = 4 * 4 * 2 * 8
    U = np.arange(V)
    for world in (1, 2, 4):
        parts = [sharded.slab_of(U, N, world, r) for r in range(world)]
        assert np.array_equal(np.concatenate(parts), U)
        t = parts[-1] // (4 * 4 * 2)
        assert t.min() == 8 - 8 // world and t.max() == 7
