"""N > 1 path (replicas only) with world_size 2 over gloo on CPU: right-hand sides are
partitioned without overlap, sources differ per rank, and the aggregation is sum(work) / max(time)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    from paper_1701_07559_b200 import inputs, replicas
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cols = replicas.columns_for_rank(12, rank, world)
    src = inputs.gaussian_source((2, 2, 2, 2), 4, replicas.source_seed(5, rank))
    work, secs = replicas.aggregate(float(len(cols)), 1.0 + rank)
    gathered = [None] * world
    dist.all_gather_object(gathered, (cols, float(src.abs().sum())))
    if rank == 0:
        out.put((work, secs, gathered))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_partition_and_aggregate():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    work, secs, gathered = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert work == 12.0 and secs == 2.0                       # sum of work, max of time
    c0, c1 = gathered[0][0], gathered[1][0]
    assert sorted(c0 + c1) == list(range(12)) and not set(c0) & set(c1) and abs(len(c0) - len(c1)) <= 1
    assert gathered[0][1] != gathered[1][1]                    # distinct right-hand sides


def test_single_process_aggregate_is_identity():
    from paper_1701_07559_b200 import replicas
    assert replicas.aggregate(3.0, 0.5) == (3.0, 0.5)
    assert replicas.columns_for_rank(12, 0, 1) == list(range(12))
