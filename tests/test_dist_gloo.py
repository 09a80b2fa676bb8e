"""World-size-2 gloo test (CPU) of the N > 1 host logic: unit sharding covers every pose once, the timing reduction
is the max over ranks, whole-job throughput sums the ranks' units (replicas, no data-path collective)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2512_20927_b200 import dist as qd
    units = qd.shard_units(8, rank, world)                 # config 4: 8 poses on a circle
    ms = 10.0 + 5.0 * rank                                 # rank 1 is slower
    mx = qd.max_over_ranks(ms)
    total = qd.sum_over_ranks(len(units))
    out[rank] = (units, mx, total)
    dist.barrier()
    dist.destroy_process_group()


def test_sharding_and_timing_reduction_world2():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    u0, m0, t0 = out[0]
    u1, m1, t1 = out[1]
    assert sorted(u0 + u1) == list(range(8)) and not set(u0) & set(u1)
    assert m0 == m1 == 15.0
    assert t0 == t1 == 8.0
    from paper_2512_20927_b200 import dist as qd
    assert abs(qd.job_throughput([len(u0), len(u1)], m0) - 8 / 0.015) < 1e-9


def test_single_process_identity():
    from paper_2512_20927_b200 import dist as qd
    assert qd.max_over_ranks(3.5) == 3.5
    assert qd.shard_units(5, 0, 1) == [0, 1, 2, 3, 4]
