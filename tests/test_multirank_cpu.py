"""N > 1 path of bench.py on CPU: world_size-2 gloo.  The hot path does not shard in this contract (BASELINE.json:
one GPU, no collectives), so N ranks are N independent replicas and the only collective is the MAX of the timings;
the reference arm runs on rank 0 alone."""
import os
import socket
import subprocess
import sys

import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    total, e2e = bench.max_over_ranks([100.0 + 50.0 * rank, 7.0 - rank], dist, "cpu")
    out[rank] = (total, e2e, bench.aggregate_value(world, 1000, 4, total))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        total, e2e, value = res[rank]
        assert total == 150.0 and e2e == 7.0                # max over ranks, seen by every rank
        assert value == 2 * 1000 * 4 / 0.150                # whole-job aggregate of the replicas


def test_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.0, 4.0]) == [3.0, 4.0]
    assert bench.aggregate_value(1, 10, 2, 1000.0) == 20.0


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
