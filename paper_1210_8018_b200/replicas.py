"""Replica sharding for N > 1 GPUs: every rank fixes its own lattice.

There is no data-path collective: the lattices of an ensemble are independent problems
(SURVEY 8(e)).  The only communication is the timing reduction of the benchmark: the step time
is the MAX over ranks, the work is the SUM over ranks.  Works with any torch.distributed
backend (nccl on GPUs, gloo in the CPU tests); with no process group it is the identity.
"""
import torch
import torch.distributed as dist

SEED_STRIDE = 7919


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of the lattice that rank `rank` fixes (rank 0 keeps the workload's own seed)."""
    return int(base_seed) + SEED_STRIDE * int(rank)


def shard_ensemble(n_lattices: int, rank: int, world: int):
    """Indices of the lattices of an ensemble that `rank` fixes: round-robin, ragged tail allowed."""
    return list(range(int(rank), int(n_lattices), int(world)))


def reduce_timing(times_ms, units, device="cpu"):
    """(max over ranks of each time, sum over ranks of units).

    times_ms: sequence of this rank's times; units: this rank's work (e.g. sites * steps)."""
    t = torch.tensor([float(x) for x in times_ms], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return [float(x) for x in t], float(u[0])
