"""The N > 1 path of bench.py (replicas only) on CPU: two gloo ranks
line up, shard independent propagations and combine timings as max / units as sum."""
import os
import socket

import torch
import torch.multiprocessing as mp

from paper_1706_02261_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    assert replicas.init("gloo") == world
    replicas.barrier()
    lo, hi = replicas.shard(5, rank, world)
    t = 2.0 if rank == 0 else 3.0                 # rank 1 is slower
    out = (lo, hi, replicas.max_over_ranks(t), replicas.sum_over_ranks(hi - lo),
           replicas.throughput(float(hi - lo), t))
    replicas.barrier()
    replicas.shutdown()
    q.put((rank, out))


def test_two_gloo_ranks_shard_and_combine():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert (res[0][0], res[0][1]) == (0, 2) and (res[1][0], res[1][1]) == (2, 5)
    for r in (0, 1):
        assert res[r][2] == 3.0 and res[r][3] == 5.0 and abs(res[r][4] - 5.0 / 3.0) < 1e-12


def test_single_process_is_a_no_op():
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert replicas.env_world() == (0, 0, 1)
    assert replicas.max_over_ranks(1.5) == 1.5 and replicas.sum_over_ranks(2.0) == 2.0
    assert replicas.shard(7, 0, 1) == (0, 7)
    assert replicas.throughput(10.0, 2.0) == 5.0
