"""N > 1 path of bench.py (replicas only) on CPU: world_size 2, gloo backend, rendezvous on 127.0.0.1."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1202_1350_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        base = np.arange(64, dtype=np.uint64)
        mine = replicas.replica_input(base, 1002, rank)
        dist.barrier()
        # every rank reports its own step time; the job time is the max
        got = replicas.max_over_ranks([1.5 + rank, 10.0 - rank])
        out.put((rank, mine.tolist(), got))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_max_and_distinct_inputs():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, in0, m0), (r1, in1, m1) = res
    assert (r0, r1) == (0, 1)
    assert m0 == m1 == [2.5, 10.0]                       # MAX over ranks, identical on both
    assert in0 == list(range(64))                        # rank 0 keeps the BASELINE workload
    assert sorted(in1) == in0 and in1 != in0             # rank 1: same values, another seeded arrangement
    assert replicas.whole_job_value(1000, 2, 2.5) == 1000 * 2 / 2.5e-3


def test_single_process_is_identity():
    assert replicas.max_over_ranks([3.0, 4.0]) == [3.0, 4.0]
    x = np.arange(8, dtype=np.uint64)
    assert replicas.replica_input(x, 5, 0) is x
