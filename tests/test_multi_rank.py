"""Host-side logic of the N > 1 path: rays are sharded over ranks with no exchange
step; the only collectives are the timing reductions.  world_size 2 on gloo, CPU only."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    seed, first, rays = bench.shard_plan(world, rank, 1 << 20)
    # rank r "took" 10 + 5 r ms for its 2^20 rays
    value, t_max = bench.aggregate(10.0 + 5.0 * rank, rays, dist, world)
    q.put((rank, seed, first, rays, value, t_max))
    dist.barrier()
    dist.destroy_process_group()


def test_shard_plan_and_aggregate_world2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps: p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    (r0, s0, f0, n0, v0, t0), (r1, s1, f1, n1, v1, t1) = res
    assert s0 != s1                                  # every rank draws its own camera
    assert (f0, f1) == (0, 1 << 20) and n0 == n1 == 1 << 20      # disjoint, contiguous ray ranges
    assert t0 == t1 == 15.0                          # max over ranks
    assert v0 == v1 == (2 << 20) / 15.0 / 1e3        # whole-job Mrays/s = all rays / slowest rank


def test_aggregate_single_rank_needs_no_process_group():
    import bench
    v, t = bench.aggregate(20.0, 1 << 20, dist, 1)
    assert t == 20.0 and abs(v - (1 << 20) / 20.0 / 1e3) < 1e-9
