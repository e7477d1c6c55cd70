"""The N > 1 path of bench.py is "independent replicas": no data-path collective, one
max-over-ranks reduction of the device time.  Covered here with world_size 2 on the gloo backend."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    base = np.zeros((8, 5))
    base[:, 3] = np.linspace(-1e-9, 0.0, 8)
    mine = bench.replica_templates(base, rank)
    # pretend rank r needed (10 + 5 r) ms for 4 steps of 1000 units each
    value, ms = bench.aggregate_ranks(10.0 + 5.0 * rank, 1000, 4, dist)
    q.put((rank, mine[:, 3].tolist(), value, ms))
    dist.destroy_process_group()


def test_two_replicas_disjoint_banks_and_max_over_ranks():
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
    (r0, f0, v0, m0), (r1, f1, v1, m1) = res
    assert set(f0).isdisjoint(f1)                                 # every rank searches its own sub-bank
    step = f0[1] - f0[0]
    assert abs((min(f0) - max(f1)) - step) < 1e-6 * abs(step)     # the banks tile the fdot axis without a hole
    assert m0 == m1 == 15.0 / 4                                   # slowest rank's time, on both ranks
    assert v0 == v1 == 2 * 1000 / (15.0 / 4 * 1e-3)               # whole-job units / that time
