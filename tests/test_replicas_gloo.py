"""Multi-GPU plumbing of bench.py ("replicas only"): max-over-ranks timing and the whole-job value,
exercised with world_size 2 on CPU over gloo (rendezvous on 127.0.0.1)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 * (rank + 1)                      # rank 1 is the slow replica
    ms = bench.reduce_max_ms(ms_local, dist, torch.device("cpu"))
    val = bench.whole_job_value(1_000_000, world, 5, ms)
    dist.barrier()
    out.put((rank, ms, val))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val in res:
        assert ms == 20.0                              # the slowest replica sets the time on every rank
        assert abs(val - 2 * 1_000_000 * 5 / 20e-3 / 1e9) < 1e-12


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_max_ms(3.5, None, None) == 3.5
    assert bench.whole_job_value(2_000_000_000, 1, 1, 1000.0) == 2.0
