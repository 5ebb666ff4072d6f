"""The N > 1 path of bench.py on CPU (world_size 2, gloo).  One evaluation does not shard ("replicas only", DESIGN.md
section 9): ranks run independent replicas, the only inter-rank traffic is the barrier and the MAX reduction of the timed
region; the job value is world x atoms / slowest rank's time.  The reference arm runs on rank 0 alone."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dist.barrier()
        mine = 100.0 + 25.0 * rank                      # ms of this rank's timed region
        slowest = bench._max_over_ranks(mine, dist, torch.device("cpu"))
        q.put((rank, slowest, bench._job_value(world, 1000, slowest * 1e-3)))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_job_value_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    for rank, slowest, value in res:
        assert slowest == 125.0                          # rank 1 is the slow one; both ranks agree
        assert value == pytest.approx(2 * 1000 / 0.125)


def test_single_rank_needs_no_process_group():
    import torch
    sys.path.insert(0, ROOT)
    import bench
    assert bench._max_over_ranks(7.5, None, torch.device("cpu")) == 7.5
    assert bench._job_value(1, 1029000, 0.148) == pytest.approx(1029000 / 0.148)


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29999")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
