"""N > 1 path (independent replicas, no data-path collective): the only exchange is the
timing reduction, covered here with two gloo ranks on CPU."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1310_1905_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 10.0 + 5.0 * rank           # rank 1 is the slow one
        units_local = 1000.0 * (rank + 1)
        ms, units = replicas.job_totals(ms_local, units_local)
        thr = replicas.job_throughput(ms_local, units_local)
        out.put((rank, ms, units, thr, replicas.replica_seed(42, rank)))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_job_totals_two_gloo_ranks():
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
    for rank, ms, units, thr, seed in res:
        assert ms == 15.0 and units == 3000.0          # max over ranks, sum over ranks: same on every rank
        assert abs(thr - 3000.0 / 15e-3) < 1e-6
        assert seed == 42 + rank                        # replicas differ by seed only


def test_single_process_is_identity():
    assert replicas.job_totals(3.0, 7.0) == (3.0, 7.0)
    assert replicas.job_throughput(2.0, 4.0) == 2000.0
