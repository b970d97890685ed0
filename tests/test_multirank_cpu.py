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


# ---------------------------------------------------------------- x-slab halo exchange, gloo
def _slab_worker(rank, world, port, cpd, R, out):
    import numpy as np
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2110_11398_b200 import slabs
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    g = torch.Generator().manual_seed(1234)
    pos = torch.rand((6000, 3), generator=g)                     # the same global set on every rank
    sl = slabs.slab_of(pos, cpd, 1.0)
    first, cnt = slabs.slab_partition(cpd, world)[rank]
    own_mask = ((sl - first) % cpd) < cnt
    local, n_own = slabs.halo_exchange(pos[own_mask].contiguous(), cpd, 1.0, R, rank, world, dist)
    need = slabs.needed_slabs(first, cnt, cpd, R)
    halo_mask = torch.zeros(cpd, dtype=torch.bool)
    if need:
        halo_mask[torch.tensor(sorted(need))] = True
    expect_halo = pos[halo_mask[sl] & ~own_mask]
    got_halo = local[n_own:]
    key = lambda t: np.unique(t.numpy().view([("x", "f4"), ("y", "f4"), ("z", "f4")]))     # sorted distinct rows
    ok = (n_own == int(own_mask.sum()) and torch.equal(local[:n_own], pos[own_mask])
          and got_halo.shape == expect_halo.shape and np.array_equal(key(got_halo), key(expect_halo)))
    # the halo of each peer arrives in that peer's original relative order
    order_ok = True
    off = n_own
    for q in range(world):
        if q == rank:
            continue
        fq, cq = slabs.slab_partition(cpd, world)[q]
        from_q = pos[(((sl - fq) % cpd) < cq) & halo_mask[sl]]
        order_ok &= torch.equal(local[off:off + from_q.shape[0]], from_q)
        off += from_q.shape[0]
    # more columns travel with the particle (column 3 = mass): same rows, same order, payload intact
    tag = lambda t: t[:, 0] + 2 * t[:, 1] + 3 * t[:, 2]
    pos4 = torch.cat([pos, tag(pos)[:, None]], dim=1)
    local4, n_own4 = slabs.halo_exchange(pos4[own_mask].contiguous(), cpd, 1.0, R, rank, world, dist)
    order_ok &= n_own4 == n_own and torch.equal(local4[:, :3], local) and torch.equal(local4[:, 3], tag(local))
    out[rank] = (bool(ok), bool(order_ok), int(local.shape[0]))
    dist.barrier()
    dist.destroy_process_group()


def _run_slab(world, cpd, R):
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_slab_worker, args=(world, port, cpd, R, out), nprocs=world, join=True)
        return dict(out)


def test_halo_exchange_gloo_world2():
    res = _run_slab(2, 9, 2)
    assert all(res[r][0] and res[r][1] for r in range(2)), res


def test_halo_exchange_gloo_world3_small_ranges():
    """Three ranks on 7 slabs with R = 2: ranges of 3, 2, 2 slabs, so halos come from both peers and wrap."""
    res = _run_slab(3, 7, 2)
    assert all(res[r][0] and res[r][1] for r in range(3)), res


def test_slab_partition_and_needs():
    sys.path.insert(0, ROOT)
    from paper_2110_11398_b200 import slabs
    parts = slabs.slab_partition(63, 8)
    assert sum(c for _, c in parts) == 63 and parts[0] == (0, 8) and parts[-1] == (56, 7)
    assert all(parts[i][0] + parts[i][1] == parts[i + 1][0] for i in range(7))
    assert slabs.needed_slabs(0, 8, 63, 2) == {61, 62, 8, 9}
    assert slabs.needed_slabs(3, 2, 5, 2) == {0, 1, 2}                 # cpd = 2R+1: every other slab, once
    assert slabs.needed_slabs(0, 9, 9, 2) == set()
    pos = torch.tensor([[0.0, 0, 0], [0.999999, 0, 0], [1.0 / 7, 0, 0], [float.fromhex("0x1.fffffep-1"), 0, 0]])
    assert slabs.slab_of(pos, 7, 1.0).tolist() == [0, 6, 1, 6]
