"""N > 1 path of the bench on CPU: world_size-2 gloo. The draft step does not shard (replicas only), so the
multi-rank logic is the timing reduction: job time = max over ranks, job work = sum over ranks."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2412_18934_b200 import replicas


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 10.0 + 5.0 * rank          # rank 1 is the slow replica: 15 ms
        units_local = 16.0 * 50               # gamma candidates x steps, per replica
        ms, units = replicas.job_time_and_work(ms_local, units_local)
        tput = replicas.throughput(ms_local, units_local)
        dist.barrier()
        out.put((rank, ms, units, tput))
    finally:
        dist.destroy_process_group()


def test_two_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, units, tput in res:
        assert ms == 15.0                      # max over ranks
        assert units == 2 * 16.0 * 50          # sum over ranks
        assert abs(tput - units / 15e-3) < 1e-6


def test_single_process_is_identity():
    assert replicas.job_time_and_work(3.0, 7.0) == (3.0, 7.0)
    assert replicas.throughput(2.0, 8.0) == 4000.0
