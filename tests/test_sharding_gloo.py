"""Multi-GPU host logic on CPU: world_size 2 and 3 on gloo.

The path shards the flattened (sky, tau, n) group index into contiguous ranges, whole groups per
rank, with no data-path collective.  Here gloo ranks each take their range
from `shard_groups`, decompose it into sub-grids with the library's own host routine
(`tcw_split_groups`, what `tcw_search_groups` runs on a GPU), evaluate each sub-grid -- the oracle
stands in for the kernels, which need a GPU -- and gather; rank 0 checks that the assembled
`out_stat` / `out_best` equal the unsharded oracle element by element.  The n_sky = 1 grids are the
case round 1 could not split at all."""
import os
import socket

import numpy as np
import pytest
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


def _workload(n_sky: int):
    w = tcw_inputs.make_workload("cfg1").subgrid(f0=slice(0, 24))       # 4 tau x 3 n
    if n_sky > 1:
        w.sky = tcw_inputs.fibonacci_cap(n_sky, 1.0, 0.3, 10.0)
    return w


def _rank_main(rank: int, world: int, port: int, n_sky: int, out_path: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _workload(n_sky)
        n_f0 = len(w.f0)
        lo, hi = tcw.shard_groups(w.n_groups, rank, world)
        stat, val, idx = [], [], []
        for s, a, b in tcw.split_groups(len(w.tau), len(w.brk), lo, hi):      # what tcw_search_groups runs
            sub = w.subgrid(sky=s, tau=a, brk=b)
            ref = oracle.evaluate(sub)
            v, i = oracle.best(ref.stat, n_f0)
            stat.append(ref.stat); val.append(v); idx.append(i)
        cat = lambda xs, dt: np.concatenate(xs) if xs else np.empty(0, dtype=dt)   # noqa: E731
        mine = (lo, cat(stat, np.float64), cat(val, np.float64), cat(idx, np.int64))
        assert len(mine[1]) == (hi - lo) * n_f0
        parts = [None] * world
        dist.all_gather_object(parts, mine)        # out_best gathered only because rank 0 wants the full list
        # max-over-ranks timing reduction used by bench.py
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert t.item() == float(world)
        dist.barrier()
        if rank == 0:
            parts.sort(key=lambda p: p[0])
            np.savez(out_path, stat=np.concatenate([p[1] for p in parts]),
                     val=np.concatenate([p[2] for p in parts]), idx=np.concatenate([p[3] for p in parts]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,n_sky", [(2, 1), (3, 1), (2, 5)])
def test_group_sharding_reassembles_the_unsharded_search(tmp_path, world, n_sky):
    out = str(tmp_path / "gathered.npz")
    mp.spawn(_rank_main, args=(world, _free_port(), n_sky, out), nprocs=world, join=True)
    got = np.load(out)
    w = _workload(n_sky)
    ref = oracle.evaluate(w)
    val, idx = oracle.best(ref.stat, len(w.f0))
    assert np.array_equal(got["stat"], ref.stat)
    assert np.array_equal(got["val"], val) and np.array_equal(got["idx"], idx)


def test_shard_groups_partitions_every_rank_count():
    for n_groups in (1, 2, 12, 160, 576, 20480, 98304):
        for world in (1, 2, 3, 8):
            parts = [tcw.shard_groups(n_groups, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n_groups
            assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
            assert max(hi - lo for lo, hi in parts) - min(hi - lo for lo, hi in parts) <= 1
