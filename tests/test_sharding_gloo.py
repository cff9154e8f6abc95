"""Multi-GPU host logic on CPU: world_size-2 gloo.

The path shards whole sky points -- hence whole (sky, tau, n) groups -- across ranks with no
data-path collective.  Here two gloo ranks each evaluate their shard (the oracle stands in for the
kernels, which need a GPU), gather the per-group candidates, and rank 0 checks that the assembled
result equals the unsharded one, element by element."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import paper_2507_07816_b200 as tcw
import tcw_inputs


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _workload():
    w = tcw_inputs.make_workload("cfg1")
    sky = tcw_inputs.fibonacci_cap(5, 1.0, 0.3, 10.0)            # 5 sky points: uneven split 3 + 2
    w = w.subgrid(f0=slice(0, 24), tau=[0, 2])
    w.sky = sky
    return w


def _rank_main(rank: int, world: int, port: int, out_path: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _workload()
        part = tcw.shard_groups(len(w.sky), rank, world)
        mine = w.subgrid(sky=part)
        ref = oracle.evaluate(mine)
        val, idx = oracle.best(ref.stat, len(mine.f0))
        # out_stat slices are disjoint and ordered by sky: gather them (variable length -> object gather)
        stats = [None] * world
        bests = [None] * world
        dist.all_gather_object(stats, (part.start, ref.stat))
        dist.all_gather_object(bests, (part.start, val, idx))
        # max-over-ranks timing reduction used by bench.py
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert t.item() == float(world)
        dist.barrier()
        if rank == 0:
            stats.sort(key=lambda p: p[0])
            bests.sort(key=lambda p: p[0])
            np.savez(out_path, stat=np.concatenate([p[1] for p in stats]),
                     val=np.concatenate([p[1] for p in bests]), idx=np.concatenate([p[2] for p in bests]))
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding_reassembles_the_unsharded_search(tmp_path):
    out = str(tmp_path / "gathered.npz")
    mp.spawn(_rank_main, args=(2, _free_port(), out), nprocs=2, join=True)
    got = np.load(out)
    w = _workload()
    ref = oracle.evaluate(w)
    val, idx = oracle.best(ref.stat, len(w.f0))
    assert np.array_equal(got["stat"], ref.stat)
    assert np.array_equal(got["val"], val) and np.array_equal(got["idx"], idx)


def test_shard_groups_partitions_every_rank_count():
    for n_sky in (1, 2, 5, 256, 4096):
        for world in (1, 2, 3, 8):
            parts = [tcw.shard_groups(n_sky, r, world) for r in range(world)]
            assert parts[0].start == 0 and parts[-1].stop == n_sky
            assert all(a.stop == b.start for a, b in zip(parts, parts[1:]))
