"""The N>1 leg of bench.py on CPU: two gloo ranks (the path does not shard,
so --gpus N runs N independent replicas; the only cross-rank step is the max-over-ranks of the
timed region and the whole-job aggregate)."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    my_ms = 100.0 + 25.0 * rank                    # rank 1 is the slow replica
    total = bench.max_over_ranks(my_ms, dist, "cpu")
    dist.barrier()
    if rank == 0:
        out.put((total, bench.whole_job_value(2.0e9, 5, total, world)))
    dist.destroy_process_group()


def test_two_gloo_ranks_take_the_max_and_aggregate():
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    total, value = out.get()
    assert total == 125.0                                   # max over ranks, not the mean
    assert value == pytest.approx(2 * 2.0e9 * 5 / 0.125 / 1e9)


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.whole_job_value(1e9, 2, 1000.0, 1) == pytest.approx(2.0)
    # flop model of the step: J + K1 + K2-lower
    import dfjk_inputs as gi
    cfg = gi.CONFIGS[4]
    assert bench.flops_step(cfg) == pytest.approx(4.0 * 5000 * 1280800 + 2.0 * 5000 * 1600 ** 2 * 130
                                                  + 5000.0 * 1600 * 1601 * 130)
