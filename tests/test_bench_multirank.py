"""N > 1 host logic of bench.py on CPU (gloo, world_size 2): the path does not shard -- replicas only, no data-path
collective -- so what has to be right is the timing rule (max over ranks) and the whole-job rate."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 100.0 + 50.0 * rank                      # rank 1 is the slow one
        ms = bench.max_over_ranks(ms_local, dist, "cpu")
        rate = bench.whole_job_rate(1.0e9, 3, world, ms)
        # seeds differ per rank: every replica solves its own zone
        inp, nt, _ = bench.make_workload("config1", 10, rank)
        q.put((rank, ms, rate, int(inp.seed)))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_two_ranks_max_time_and_whole_job_rate():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=90) for _ in range(2))
    for p in procs:
        p.join(timeout=30)
        assert p.exitcode == 0
    (r0, ms0, rate0, seed0), (r1, ms1, rate1, seed1) = out
    assert ms0 == ms1 == 150.0                               # the max over ranks, on both ranks
    assert rate0 == rate1 == pytest.approx(1.0e9 * 3 * 2 / 0.150)
    assert seed0 != seed1


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, None, "cpu") == 12.5
    assert bench.whole_job_rate(2.0, 5, 1, 1000.0) == pytest.approx(10.0)
