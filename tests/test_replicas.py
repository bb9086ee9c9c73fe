"""The N>1 path of bench.py (independent replicas; barrier + MAX-over-ranks timing), exercised with
two gloo processes on the CPU."""
import os
import socket

import pytest
import torch
import torch.multiprocessing as mp


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2405_08470_b200 import replicas
    r, w, l = replicas.init("gloo")
    assert (r, w, l) == (rank, world, rank)
    replicas.barrier()
    ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    value, ms = replicas.aggregate_throughput(1000.0, ms_local)
    mx = replicas.max_over_ranks(float(rank))
    replicas.barrier()
    replicas.finalize()
    q.put((rank, value, ms, mx))


def test_two_replicas_aggregate_with_max_time():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, ms, mx in res:
        assert ms == 15.0                              # slowest rank's time on every rank
        assert value == pytest.approx(2 * 1000.0 / 15e-3)   # both replicas' units over that time
        assert mx == 1.0


def test_single_process_is_a_noop():
    from paper_2405_08470_b200 import replicas
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    assert replicas.env_ranks() == (0, 1, 0)
    replicas.barrier()
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.aggregate_throughput(100.0, 50.0) == (pytest.approx(2000.0), 50.0)
