"""Communicators for t-sharded contexts (include/gf.h, "t-shards"): plumbing only.

A sharded run needs, between the shards, a stream-ordered barrier and the in-place sum of a small host array
(2 * Nt_global .. 6 * Nt_global doubles per check).  libgf.so links no communication library: the caller hands it
two callbacks (gf_comm).  This module builds them

  * for several shards driven by the threads of one process (`ThreadComm`; the shards share one CUDA stream, so the
    enqueue order is the execution order and the barrier only has to order the host threads), and
  * for one process per GPU over torch.distributed (`TorchDistComm`; NCCL: the barrier is an all-reduce of one element
    enqueued on the context's stream, gloo: a host barrier after a stream synchronisation),

and the partition of N_t over the ranks.  No arithmetic of the method lives here.
"""
from __future__ import annotations

import ctypes
import threading

import numpy as np

from . import gf


def partition_t(Nt_global: int, n_shards: int):
    """[(t0, Nt_local)] for every shard: contiguous, even first slice and even extent (the colouring of a store is
    the global one), as equal as that allows."""
    if Nt_global % 2 or n_shards < 1 or Nt_global // 2 < n_shards:
        raise ValueError(f"cannot split Nt = {Nt_global} into {n_shards} shards of even extent")
    pairs, rem = divmod(Nt_global // 2, n_shards)
    out, t0 = [], 0
    for k in range(n_shards):
        n = 2 * (pairs + (1 if k < rem else 0))
        out.append((t0, n))
        t0 += n
    return out


def _as_array(buf, n):
    return np.ctypeslib.as_array(buf, shape=(n,))


class ThreadComm:
    """Shards of one process, one host thread per shard, all on ONE CUDA stream."""

    class _Shared:
        def __init__(self, n):
            self.n = n
            self.barrier = threading.Barrier(n)
            self.slots = [None] * n

    def __init__(self, shared: "ThreadComm._Shared", rank: int):
        self.shared, self.rank = shared, rank
        self._b = gf.GF_BARRIER_FN(self._barrier)
        self._a = gf.GF_ALLREDUCE_FN(self._allreduce)
        self.comm = gf.gf_comm(self._b, self._a, None)

    @classmethod
    def group(cls, n):
        sh = cls._Shared(n)
        return [cls(sh, r) for r in range(n)]

    def _barrier(self, _user):
        self.shared.barrier.wait()

    def _allreduce(self, _user, buf, n):
        a = _as_array(buf, n)
        self.shared.slots[self.rank] = a.copy()
        self.shared.barrier.wait()
        total = np.zeros(n)
        for s in self.shared.slots:       # rank order on every thread: the same bits everywhere
            total += s
        self.shared.barrier.wait()
        a[:] = total


class TorchDistComm:
    """One process per shard over torch.distributed (NCCL on GPUs; gloo for the CPU-side tests)."""

    def __init__(self, dist, device=None, stream=None):
        self.dist, self.device, self.stream = dist, device, stream
        self.nccl = dist.get_backend() == "nccl"
        import torch
        self.torch = torch
        self.flag = torch.zeros(1, device=device) if self.nccl else None
        self.calls = {"barrier": 0, "allreduce": 0}
        self._b = gf.GF_BARRIER_FN(self._barrier)
        self._a = gf.GF_ALLREDUCE_FN(self._allreduce)
        self.comm = gf.gf_comm(self._b, self._a, None)

    def _barrier(self, _user):
        self.calls["barrier"] += 1
        if self.nccl:
            # stream-ordered: the collective waits for the work enqueued on the context's stream and the stream waits
            # for the collective (async_op=False), the host does not
            with self.torch.cuda.stream(self.stream):
                self.dist.all_reduce(self.flag)
        else:
            if self.stream is not None:
                self.stream.synchronize()
            self.dist.barrier()

    def _allreduce(self, _user, buf, n):
        self.calls["allreduce"] += 1
        a = _as_array(buf, n)
        t = self.torch.from_numpy(a.copy())
        if self.nccl:
            with self.torch.cuda.stream(self.stream):
                d = t.to(self.device)
                self.dist.all_reduce(d)
                t = d.cpu()
        else:
            self.dist.all_reduce(t)
        a[:] = t.numpy()


def exchange_handles(dist, handle: "gf.gf_shard_handle"):
    """All-gather the exported stores of the shards (one per rank, rank k = k-th slab) and return the handles of the
    shards below and above this rank's (periodic).  Marshalling only: the handles are opaque bytes."""
    world, rank = dist.get_world_size(), dist.get_rank()
    blobs = [None] * world
    dist.all_gather_object(blobs, bytes(handle))
    hs = [gf.gf_shard_handle.from_buffer_copy(b) for b in blobs]
    return hs[(rank - 1) % world], hs[(rank + 1) % world]


def make_rank_shard(dist, device, stream, Nx, Ny, Nz, Nt_global, force_comm=False, **kw):
    """One process per GPU: this rank's shard of the lattice, attached to its neighbours' stores through CUDA IPC
    mappings (NVLink peer access) and wired to torch.distributed.  -> (GaugeFixer, TorchDistComm, (t0, Nt_local)).
    A single rank needs no communicator and gets none, unless force_comm asks for it: the whole call path of the
    multi-rank run (the collective issued from the library's callback once per half-sweep, the device-tensor sum of
    the slice arrays) then runs on one GPU, which is how it is tested and timed where only one GPU is at hand."""
    world, rank = dist.get_world_size(), dist.get_rank()
    t0, n = partition_t(Nt_global, world)[rank]
    fx = gf.GaugeFixer(Nx, Ny, Nz, n, cuda_stream=stream, shard=(t0, Nt_global), **kw)
    if world == 1:
        fx.attach(fx, fx)
        if not force_comm:
            return fx, None, (t0, n)
        comm = TorchDistComm(dist, device=device, stream=stream)
        fx.set_comm(comm.comm)
        return fx, comm, (t0, n)
    below, above = exchange_handles(dist, gf.gf_shard_export(fx.ctx))
    gf.gf_shard_attach_ipc(fx.ctx, below, above)
    comm = TorchDistComm(dist, device=device, stream=stream)
    fx.set_comm(comm.comm)
    return fx, comm, (t0, n)
