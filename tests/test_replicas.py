"""N > 1 path on CPU: replica sharding and the max-over-ranks timing reduction under gloo,
world_size 2.  No GPU, no liblgf compute."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1210_8018_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import gen

        seed = replicas.replica_seed(gen.BASE_SEED + 4, rank)
        U = gen.gen_links(4, 0.3, seed)
        mine = replicas.shard_ensemble(5, rank, world)
        # rank r pretends its step took (1 + r) ms over 100 units per lattice
        times, units = replicas.reduce_timing([1.0 + rank, 10.0 - rank], 100 * len(mine))
        out[rank] = (seed, float(abs(U).sum()), mine, times, units)
    finally:
        dist.destroy_process_group()


def test_replicas_gloo_world2():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert r0[0] != r1[0] and r0[1] != r1[1]              # distinct lattices per rank
    assert sorted(r0[2] + r1[2]) == [0, 1, 2, 3, 4]       # ensemble covered once, ragged tail
    assert r0[3] == r1[3] == [2.0, 10.0]                  # max over ranks
    assert r0[4] == r1[4] == 500.0                        # sum of work over ranks


def test_single_process_is_identity():
    t, u = replicas.reduce_timing([3.5], 7)
    assert t == [3.5] and u == 7.0
    assert replicas.replica_seed(10, 0) == 10
    assert replicas.shard_ensemble(3, 1, 4) == [1] and replicas.shard_ensemble(3, 3, 4) == []
