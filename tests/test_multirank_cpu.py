"""N > 1 host logic of bench.py on CPU: two gloo ranks (replicas only, no data-path collective).

The GPU path needs one B200 per rank; what can be checked here is the part that is not kernels: the rendezvous from
the torchrun environment, the max-over-ranks reduction of the timed region, the whole-job aggregate, and that the
`--impl reference` arm runs on rank 0 alone.
"""
import json
import os
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = 1.0 + 0.5 * rank                       # rank 1 is the slow replica
        slowest = bench.max_over_ranks(mine, dist, "cpu")
        dist.barrier()
        out[rank] = (slowest, bench.whole_job_gbs(3e9, slowest, world))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_take_the_slowest_replica():
    world, port = 2, 29517 + os.getpid() % 200
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    slowest, value = res[0]
    assert slowest == 1.5
    assert value == pytest.approx(2 * 3e9 / 1.5 / 1e6)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(2.25, None, "cpu") == 2.25
    assert bench.whole_job_gbs(1e9, 1.0, 1) == pytest.approx(1000.0)


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_step_bytes_accounting():
    sys.path.insert(0, ROOT)
    import bench
    c, shapes = bench.layer_tensors()
    sb = bench.step_bytes(shapes)
    assert sb["B"] == 436207616                       # cfg1 layer
    assert sb["total"] == (8 + len(bench.BATCHES)) * sb["B"] and sb["gemv"] == len(bench.BATCHES) * sb["B"]
    json.dumps(sb)
