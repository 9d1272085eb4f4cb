"""world_size-2 gloo test (CPU) of bench.py's multi-process plumbing: barrier, max-over-ranks time, summed units.
The path itself does not shard ("replicas only"): each rank runs an independent replica, here the CPU oracle on a
tiny workload stands in for the per-rank work so that the aggregation is exercised end to end."""
import os
import socket

import pytest
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update({"RANK": str(rank), "WORLD_SIZE": str(world), "LOCAL_RANK": str(rank),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    from paper_2006_00561_b200 import dist
    from oracle import pa_oracle as orc
    g = dist.init_from_env(backend="gloo", device_kind="cpu")
    orc.set_threads(1)
    pa = orc.OraclePA(8, 64, seed=100 + rank)  # independent replica per rank
    dist.barrier(g)
    units = 0
    for k in range(1, 4):
        pa.step(0.1 * k, 2)
        units += 2 * 64 * pa.R
    seconds = 1.0 + rank  # synthetic per-rank time: the slowest rank must define the job time
    value, total, tmax = dist.aggregate_throughput(g, units, seconds)
    dist.barrier(g)
    q.put((rank, units, value, total, tmax, g.is_main))
    dist.shutdown(g)


def test_two_rank_aggregation_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, u0, v0, t0, m0, main0), (r1, u1, v1, t1, m1, main1) = res
    assert main0 and not main1
    assert t0 == t1 == u0 + u1 and m0 == m1 == 2.0  # max over ranks, not the mean
    assert v0 == v1 == pytest.approx((u0 + u1) / 2.0)


def test_single_process_is_identity():
    from paper_2006_00561_b200 import dist
    g = dist.Group()
    assert dist.aggregate_throughput(g, 10.0, 2.0) == (5.0, 10.0, 2.0)
    dist.barrier(g)
