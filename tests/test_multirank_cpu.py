"""The N>1 path of bench.py on CPU: world_size-2 `gloo` processes.  The hot path has no exchange step (every
(call, head) is independent): ranks run independent replicas and only the device timings are reduced
(max over ranks) after the timed region.  This test covers exactly that plumbing."""
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
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = [10.0 + 5.0 * rank, 40.0 - 7.0 * rank]          # rank 1 is slower on the first, faster on the second
        got = bench.max_over_ranks(mine, torch.device("cpu"), world)
        dist.barrier()
        if rank == 0:
            out.put(got)
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_job_throughput_world2():
    import bench
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = out.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert got == [15.0, 40.0]
    # 2 replicas of 1e12 flop per step, 4 steps, slowest rank took 16 ms in total -> 0.5 PFLOP/s = 500 TFLOP/s
    assert bench.job_throughput(1e12, 4, 2, 16.0) == pytest.approx(500.0)
    assert bench.max_over_ranks([3.0], torch.device("cpu"), 1) == [3.0]


def test_reference_arm_only_rank0_prints(monkeypatch, capsys):
    """`--impl reference` under torchrun: ranks other than 0 exit 0 without work."""
    import bench
    monkeypatch.setenv("RANK", "1")

    class A:
        config, steps, warmup, gpus, ref_heads, ref_tiles = "tiny", 1, 0, 2, 2, None
    assert bench.run_reference(A) == 0
    assert capsys.readouterr().out == ""
