"""One lattice sharded over several GPUs in t-slabs (the B200 analogue of the paper's
distributed CPU program, which runs its FFTs through PFFT over MPI).

Rank r of R holds the time slices [r Nt/R, (r+1) Nt/R) of every array, between one halo slice below and one
above.  All arithmetic runs in the kernels of liblgf.so (`lgf_shard_step`); this module is the plumbing
between the steps, per iteration of Algorithm 1:

    (x,y) forward FFT           local: an (x,y) plane lies inside one time slice
    pack, ALL-TO-ALL            the 4 packed fields go from t-slabs to y-slabs (rank q gets rows [q Ny/R, (q+1) Ny/R))
    (z,t) forward, mask, inverse   local on the y-slab
    ALL-TO-ALL, unpack          back to t-slabs
    (x,y) inverse FFT + g(x)    local
    HALO of g                   slice 1 -> lower neighbour's upper halo, slice Nt/R -> upper neighbour's lower halo
    fused link update + measure local; gives this rank's part of F and theta
    HALO of the new t-links     slice Nt/R -> upper neighbour's lower halo (U_t(x - t) of its first slice)
    ALL-REDUCE (sum) of F, theta, then the stop decision, the same on every rank

Two all-to-alls of the packed field (64 B per site in FP64) and three one-slice halos per iteration: at 32^4 on
8 GPUs that is 8.4 MB per GPU per transpose against about 40 us of compute, communication-bound; the layout
pays from 64^4 up, or when a lattice does not fit one GPU.  Independent lattices should use
replicas.py instead: no communication at all.

`Comm` does the exchanges.  `TorchDistComm` uses torch.distributed (NCCL on GPUs; gloo in the CPU test of the
plumbing) with one slab per process.  `LocalComm` holds all R slabs in ONE process on one GPU and performs the same
exchanges as device copies: the steps of the ranks are launched one after another, nothing waits on a peer, so
this is how the sharded path is verified on a single GPU (tests/test_gpu_sharded.py).
"""
import numpy as np

from . import lgf


class LocalComm:
    """All ranks in this process: exchanges are copies between the ranks' buffers."""

    def __init__(self, world):
        self.world = int(world)
        self.local_ranks = list(range(self.world))

    def all_to_all(self, dst, src):
        """dst[r] block q <- src[q] block r (equal contiguous blocks)."""
        R = self.world
        for r in range(R):
            d = dst[r].view(R, -1)
            for q in range(R):
                d[q].copy_(src[q].view(R, -1)[r])

    def halo(self, to_lower, to_upper, from_upper, from_lower):
        """from_upper[r] <- to_lower[r+1], from_lower[r] <- to_upper[r-1] (periodic in the rank index)."""
        R = self.world
        for r in range(R):
            if to_lower is not None:
                from_upper[r].copy_(to_lower[(r + 1) % R])
            if to_upper is not None:
                from_lower[r].copy_(to_upper[(r - 1) % R])

    def all_reduce_sum(self, bufs):
        total = bufs[0].clone()
        for b in bufs[1:]:
            total += b
        for b in bufs:
            b.copy_(total)


class TorchDistComm:
    """One rank per process over torch.distributed (backend nccl on GPUs, gloo in the CPU test)."""

    def __init__(self, group=None):
        import torch.distributed as dist

        self.dist = dist
        self.group = group
        self.world = dist.get_world_size(group)
        self.rank = dist.get_rank(group)
        self.local_ranks = [self.rank]

    @staticmethod
    def _bytes(t):
        """Transport view: collectives move bytes, whatever the element type (complex tensors are not supported by every backend)."""
        import torch

        return t.view(torch.uint8) if t.is_complex() else t

    def all_to_all(self, dst, src):
        self.dist.all_to_all_single(self._bytes(dst[0]), self._bytes(src[0]), group=self.group)

    def halo(self, to_lower, to_upper, from_upper, from_lower):
        dist, R, r = self.dist, self.world, self.rank
        lo, up = (r - 1) % R, (r + 1) % R
        ops = []
        # per peer, sends and receives are matched in the order they are posted; with R = 2 both neighbours
        # are the same rank, and its first message (its to_lower) is this rank's from_upper
        B = self._bytes
        if to_lower is not None:
            ops.append(dist.P2POp(dist.isend, B(to_lower[0]), lo, group=self.group))
        if to_upper is not None:
            ops.append(dist.P2POp(dist.isend, B(to_upper[0]), up, group=self.group))
        if to_lower is not None:
            ops.append(dist.P2POp(dist.irecv, B(from_upper[0]), up, group=self.group))
        if to_upper is not None:
            ops.append(dist.P2POp(dist.irecv, B(from_lower[0]), lo, group=self.group))
        for w in dist.batch_isend_irecv(ops):
            w.wait()

    def all_reduce_sum(self, bufs):
        self.dist.all_reduce(bufs[0], op=self.dist.ReduceOp.SUM, group=self.group)


def slab_of(U, N, world, rank):
    """The time slices of `rank` out of an interchange array over the whole lattice ([V, ...], t slowest)."""
    V = N[0] * N[1] * N[2] * N[3]
    per = V // world
    return U[rank * per:(rank + 1) * per]


class ShardedGaugeFixer:
    """Algorithm 1 on one lattice sharded in t-slabs.  `comm.local_ranks` are the slabs this process holds (one
    with TorchDistComm, all of them with LocalComm); every method takes / returns one array per local slab."""

    def __init__(self, N, comm, precision="fp64", recon=18, devices=None, **opts):
        import torch

        self.torch = torch
        self.N = lgf._dims(N)
        self.comm = comm
        R = comm.world
        if self.N[3] % R or self.N[1] % R:
            raise ValueError("the number of ranks must divide Nt and Ny")
        devices = devices or ["cuda:0"] * len(comm.local_ranks)
        self.fixers = [lgf.GaugeFixer(self.N, precision=precision, recon=recon, shard=(R, r), device=d, **opts)
                       for r, d in zip(comm.local_ranks, devices)]
        self.cdt = self.fixers[0].torch_dtype
        self.info = self.fixers[0].shard_info()
        self.loaded = False

    # ---- views of the exchanged regions
    def _planes(self, f, region, arrays, t):
        """[arrays] views of time slice t of every array of a region (g: 6 arrays; t-links: NE arrays of mu = 3)."""
        i = self.info
        a = f.shard_region(region, self.cdt).view(-1, i["stored_sites"])
        return a[arrays, t * i["slice_sites"]:(t + 1) * i["slice_sites"]]

    def _exchange_tlinks(self):
        """U_t of the last own slice -> lower halo of the upper neighbour (the U_t(x - t) of its first slice)."""
        i = self.info
        ne, nt = i["ne"], i["own_slices"]
        rows = slice(3 * ne, 4 * ne)
        send, recv = [], []
        for f in self.fixers:
            f.stream.synchronize()
            send.append(self._planes(f, lgf.REGION_LINKS, rows, nt).contiguous())
            recv.append(self.torch.empty_like(send[-1]))
        self.comm.halo(None, send, None, recv)
        for f, r in zip(self.fixers, recv):
            self._planes(f, lgf.REGION_LINKS, rows, 0).copy_(r)
        self.torch.cuda.synchronize()       # the copies ran on torch's stream, the next step runs on the library's

    def _exchange_g(self):
        i = self.info
        nt = i["own_slices"]
        rows = slice(0, 6)
        lo, up, fu, fl = [], [], [], []
        for f in self.fixers:
            f.stream.synchronize()
            lo.append(self._planes(f, lgf.REGION_G, rows, 1).contiguous())
            up.append(self._planes(f, lgf.REGION_G, rows, nt).contiguous())
            fu.append(self.torch.empty_like(lo[-1]))
            fl.append(self.torch.empty_like(lo[-1]))
        self.comm.halo(lo, up, fu, fl)
        for f, a, b in zip(self.fixers, fu, fl):
            self._planes(f, lgf.REGION_G, rows, nt + 1).copy_(a)
            self._planes(f, lgf.REGION_G, rows, 0).copy_(b)
        self.torch.cuda.synchronize()

    def _sync(self):
        for f in self.fixers:
            f.stream.synchronize()
        self.torch.cuda.synchronize()

    def _all_reduce(self):
        self._sync()
        self.comm.all_reduce_sum([f.shard_region(lgf.REGION_CTRL, self.torch.float64) for f in self.fixers])

    def _step(self, step, alpha=0.0, eps=-1.0):
        for f in self.fixers:
            f.shard_step(step, alpha, eps)

    # ---- the calls of the single-GPU binding, per slab
    def load_links(self, slabs, eps=-1.0):
        """slabs[i]: links of local rank i, [V/R, 4, 3, 3] (or [V/R, 4, 2, 3]); then the initial measure."""
        for f, U in zip(self.fixers, slabs):
            f.load_links(U)
        self._exchange_tlinks()
        self._step(lgf.SHARD_MEASURE)
        self._all_reduce()
        self._step(lgf.SHARD_RESET, eps=eps)
        self.loaded = True
        return self.result()

    def get_links(self):
        return [f.get_links() for f in self.fixers]

    def result(self):
        return self.fixers[0].shard_result()

    def iterate_once(self, alpha, eps=-1.0):
        T = self.torch
        self._step(lgf.SHARD_XY_FWD)
        self._step(lgf.SHARD_PACK)
        self._sync()
        send = [f.shard_region(lgf.REGION_XSEND, self.cdt) for f in self.fixers]
        recv = [f.shard_region(lgf.REGION_XRECV, self.cdt) for f in self.fixers]
        self.comm.all_to_all(recv, send)
        T.cuda.synchronize()
        self._step(lgf.SHARD_ZT)
        self._sync()
        self.comm.all_to_all(send, recv)
        T.cuda.synchronize()
        self._step(lgf.SHARD_UNPACK)
        self._step(lgf.SHARD_XY_INV_G, alpha=alpha)
        self._exchange_g()
        T.cuda.synchronize()
        self._step(lgf.SHARD_LINK, alpha=alpha)
        self._exchange_tlinks()
        self._all_reduce()
        self._step(lgf.SHARD_FINISH, eps=eps)

    def iterate(self, alpha, n):
        for _ in range(int(n)):
            self.iterate_once(alpha)
        return self.result()

    def fix(self, alpha=0.08, eps=1e-15, max_iter=100000):
        """Algorithm 1: iterate while theta > eps; the decision is the device's, read every iteration."""
        self._step(lgf.SHARD_RESET, eps=eps)
        r = self.result()
        n = 0
        while not r.converged and n < max_iter:
            self.iterate_once(alpha, eps)
            r = self.result()
            n += 1
        return r

    def close(self):
        for f in self.fixers:
            f.close()


def exchange_selftest(comm, world, rank_data):
    """The exchanges alone, on host or device tensors, for the CPU test of the plumbing: `rank_data[r]` gives
    (send block matrix [R, n], to_lower, to_upper) per local rank; returns what each local rank receives."""
    import torch

    send = [d[0].contiguous().view(-1) for d in rank_data]
    recv = [torch.empty_like(s) for s in send]
    comm.all_to_all(recv, send)
    lo = [d[1] for d in rank_data]
    up = [d[2] for d in rank_data]
    fu = [torch.empty_like(x) for x in lo]
    fl = [torch.empty_like(x) for x in up]
    comm.halo(lo, up, fu, fl)
    tot = [d[0].real.sum().reshape(1).clone() if d[0].is_complex() else d[0].sum().reshape(1).clone() for d in rank_data]
    comm.all_reduce_sum(tot)
    return [(r.view(world, -1), a, b, t) for r, a, b, t in zip(recv, fu, fl, tot)]
