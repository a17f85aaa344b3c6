"""world_size-2 gloo test of the only multi-GPU logic the path has: batch sharding without a collective.
Each rank evaluates its shard with the fp64 oracle (CPU stand-in for its GPU); rank 0 checks that the
concatenated shards equal the whole-batch result bit for bit and that timings reduce with MAX."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2605_31481_b200 import dist as D, workloads as W


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, B, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    desc = W.config_robot(2)
    q, qd, qdd = (a.astype(np.float64) for a in W.config_states(2, B))
    lo, hi = D.shard_range(B, rank, world)
    o = oracle.Oracle(desc)
    sl = [np.ascontiguousarray(D.soa_slice(a, lo, hi)) for a in (q, qd, qdd)]
    tau = torch.from_numpy(o.rnea(*sl))
    M = torch.from_numpy(o.crba(sl[0]))
    t = D.max_over_ranks(1.0 + rank)
    D.barrier()
    if rank == 0:
        taus, Ms = [tau], [M]
        for r in range(1, world):
            l2, h2 = D.shard_range(B, r, world)
            a = torch.empty((tau.shape[0], h2 - l2), dtype=torch.float64)
            b = torch.empty((M.shape[0], M.shape[1], h2 - l2), dtype=torch.float64)
            dist.recv(a, src=r); dist.recv(b, src=r)
            taus.append(a); Ms.append(b)
        full_tau, full_M = o.rnea(q, qd, qdd), o.crba(q)
        ok = np.array_equal(torch.cat(taus, -1).numpy(), full_tau) and np.array_equal(torch.cat(Ms, -1).numpy(), full_M)
        out.put((ok, t))
    else:
        dist.send(tau.contiguous(), dst=0); dist.send(M.contiguous(), dst=0)
    dist.destroy_process_group()


def test_shard_ranges_partition_the_batch():
    for B in (1, 5, 64, 1000, 4096, 65536 + 3):
        for world in (1, 2, 3, 4, 8):
            r = [D.shard_range(B, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == B
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            assert all(lo % 4 == 0 for lo, _ in r if lo < B)


def test_two_rank_sharding_matches_whole_batch():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, 203, out)) for r in range(2)]
    for p in ps:
        p.start()
    ok, t = out.get(timeout=120)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ok
    assert t == 2.0          # MAX over ranks of (1 + rank)
