"""Host side of the t-sharded path on CPU (no GPU): the partition of N_t, the communicator callbacks as the C library
calls them (through their C function pointers), and the exchange of the opaque store handles, over world_size-2
`gloo` processes and over the threads of one process (include/gf.h "t-shards")."""
import ctypes
import os
import socket
import sys
import threading

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_of_nt():
    from paper_1212_5221_b200 import shards
    for Nt, n in ((256, 1), (256, 2), (256, 8), (64, 4), (16, 4), (10, 2), (12, 5)):
        parts = shards.partition_t(Nt, n)
        assert len(parts) == n and parts[0][0] == 0
        assert all(t0 % 2 == 0 and nl % 2 == 0 and nl >= 2 for t0, nl in parts)
        assert all(parts[k][0] + parts[k][1] == parts[k + 1][0] for k in range(n - 1))
        assert parts[-1][0] + parts[-1][1] == Nt
        assert max(nl for _, nl in parts) - min(nl for _, nl in parts) <= 2
    for Nt, n in ((7, 1), (8, 5), (4, 3)):
        with pytest.raises(ValueError):
            shards.partition_t(Nt, n)


def test_thread_comm_sums_zero_padded_slices_exactly():
    # every shard fills its own slices of a global array and zeroes the rest: the sum must return every number unchanged
    from paper_1212_5221_b200 import shards
    n_sh, Nt = 4, 16
    parts = shards.partition_t(Nt, n_sh)
    comms = shards.ThreadComm.group(n_sh)
    full = np.random.default_rng(5).standard_normal(2 * Nt)
    got = [None] * n_sh

    def work(k):
        t0, nl = parts[k]
        buf = np.zeros(2 * Nt)
        buf[t0:t0 + nl] = full[t0:t0 + nl]
        buf[Nt + t0:Nt + t0 + nl] = full[Nt + t0:Nt + t0 + nl]
        c = comms[k].comm
        c.barrier(None)
        c.allreduce_sum(None, buf.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), buf.size)
        got[k] = buf

    th = [threading.Thread(target=work, args=(k,)) for k in range(n_sh)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    for g in got:
        assert np.array_equal(g, full)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update({"RANK": str(rank), "WORLD_SIZE": str(world), "LOCAL_RANK": str(rank),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_1212_5221_b200 import gf, shards
    dist.init_process_group("gloo", rank=rank, world_size=world)
    Nt = 12
    t0, nl = shards.partition_t(Nt, world)[rank]
    comm = shards.TorchDistComm(dist)
    full = np.arange(1.0, 2 * Nt + 1.0) / 7.0
    buf = np.zeros(2 * Nt)
    buf[t0:t0 + nl] = full[t0:t0 + nl]
    buf[Nt + t0:Nt + t0 + nl] = full[Nt + t0:Nt + t0 + nl]
    comm.comm.barrier(None)                                     # as libgf.so calls them
    comm.comm.allreduce_sum(None, buf.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), buf.size)
    h = gf.gf_shard_handle()
    h.t0, h.Nt_local, h.has_transform = t0, nl, 1
    for k in range(64):
        h.links[k] = (rank * 64 + k) % 251
    below, above = shards.exchange_handles(dist, h)
    q.put((rank, bool(np.array_equal(buf, full)), (below.t0, below.Nt_local, below.links[3]),
           (above.t0, above.Nt_local, above.links[3]), dict(comm.calls)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_comm_and_handle_exchange():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, exact, below, above, calls in got:
        other = 1 - rank
        assert exact
        assert below == above == (6 * other, 6, (other * 64 + 3) % 251)     # two shards: the other one is on both sides
        assert calls == {"barrier": 1, "allreduce": 1}
