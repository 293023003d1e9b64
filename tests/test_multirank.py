"""The N>1 path of bench.py on CPU (gloo, world_size 2): MSA shards as independent replicas -- no collective on the
data path -- so what several ranks share is the timing rule: the step time is the MAX over ranks
and the reported value is the whole job's."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dist.barrier()
        ms_local = 1.0 + 0.5 * rank                      # rank 1 is the slow one
        ms = bench.dist_max(ms_local, "cpu")
        value = bench.whole_job_value(world, 0.567, ms)  # 0.567 TFLOP per step and replica
        out.put((rank, ms, value))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_two_ranks_report_the_slowest_rank_and_the_whole_job():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=90) for _ in range(world))
    for p in procs:
        p.join(timeout=30)
        assert p.exitcode == 0
    for rank, ms, value in got:
        assert ms == pytest.approx(1.5)
        assert value == pytest.approx(2 * 0.567 / 1.5e-3)


def test_single_process_values():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.whole_job_value(1, 2.0, 4.0) == pytest.approx(500.0)
    assert bench.metric_of("cfg5_short_query")[2] == "hbm" and bench.metric_of("cfg2_llama8b")[2] == "tensor"
