"""N>1 path on CPU: world_size-2 gloo run of the replicas-only plumbing:
ranks own disjoint seed ranges that together cover the job, times reduce by MAX, work by SUM."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1901_01047_b200.replicas import aggregate, rank_seeds


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, B, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seeds = rank_seeds(rank, B)
    # each rank "processes" its walkers: counter = sum of its seeds, time = rank-dependent
    ms, (acc, props) = aggregate(10.0 + 5.0 * rank, [float(seeds.sum()), float(len(seeds))])
    gathered = [None] * world
    dist.all_gather_object(gathered, seeds.tolist())
    if rank == 0:
        np.save(os.path.join(out_dir, "res.npy"), np.array([ms, acc, props] + sum(gathered, []), dtype=np.float64))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_gloo(tmp_path):
    world, B = 2, 8
    mp.spawn(_worker, args=(world, _free_port(), B, str(tmp_path)), nprocs=world, join=True)
    res = np.load(tmp_path / "res.npy")
    ms, acc, props = res[:3]
    seeds = res[3:].astype(np.int64)
    assert ms == 15.0                                   # max over ranks
    assert props == world * B                           # sum over ranks
    assert sorted(seeds.tolist()) == list(range(world * B))   # disjoint, covering
    assert acc == sum(range(world * B))


def test_single_replica_needs_no_process_group():
    ms, (a,) = aggregate(3.0, [7])
    assert ms == 3.0 and a == 7.0
    assert rank_seeds(3, 4).tolist() == [12, 13, 14, 15] and rank_seeds(0, 2).dtype == np.uint64
