"""N>1 path of bench.py (replicas only) on CPU: world_size-2 gloo, max-over-ranks timing."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_07687_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert replicas.world() == (world, rank)
        replicas.barrier()
        ms = replicas.max_over_ranks(10.0 + 5.0 * rank)       # rank 1 is the slow replica
        val = replicas.ns_per_cell(ms, 1 << 20, world)
        out.put((rank, ms, val))
    finally:
        dist.destroy_process_group()


def test_two_replicas_take_the_slowest_time():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val in res:
        assert ms == 15.0                                       # MAX over ranks, on every rank
        assert abs(val - 15.0 * 1e6 / (2 * (1 << 20))) < 1e-12  # whole-job ns/cell


def test_single_process_is_a_no_op():
    assert replicas.world() == (1, 0)
    replicas.barrier()
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.ns_per_cell(2.0, 1000, 1) == 2000.0
