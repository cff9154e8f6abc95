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


def _rank_main(rank: int, world: int, port: int, n_sky: int, out_path: str, by_work: bool = False):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _workload(n_sky)
        n_f0 = len(w.f0)
        wts = tcw.group_work(tcw.Grid.of(w), w.timestamps, w.T_sft, w.f_min, w.n_bins) if by_work else None
        lo, hi = tcw.shard_groups(w.n_groups, rank, world, weights=wts)
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


@pytest.mark.parametrize("world,n_sky,by_work", [(2, 1, False), (3, 1, False), (2, 5, False), (3, 1, True)])
def test_group_sharding_reassembles_the_unsharded_search(tmp_path, world, n_sky, by_work):
    """by_work: the cut is placed by the in-band work per group (group_work) instead of the group count;
    still contiguous, still whole groups, and the reassembly is still the unsharded result."""
    out = str(tmp_path / "gathered.npz")
    mp.spawn(_rank_main, args=(world, _free_port(), n_sky, out, by_work), nprocs=world, join=True)
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


def test_shard_groups_with_more_ranks_than_groups_gives_empty_ranges():
    parts = [tcw.shard_groups(3, r, 8) for r in range(8)]
    assert parts[0][0] == 0 and parts[-1][1] == 3 and all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
    assert sum(hi == lo for lo, hi in parts) == 5 and all(0 <= lo <= hi <= 3 for lo, hi in parts)


def test_work_weighted_cut_is_a_partition_and_balances_work():
    rng = np.random.default_rng(5)
    for n_groups in (1, 7, 576, 20480):
        wt = rng.random(n_groups) ** 3 * np.linspace(0.1, 2.0, n_groups)       # skewed: late groups cost more
        for world in (1, 2, 3, 8):
            parts = [tcw.shard_groups(n_groups, r, world, weights=wt) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n_groups
            assert all(a[1] == b[0] for a, b in zip(parts, parts[1:])) and all(lo <= hi for lo, hi in parts)
            if n_groups >= 576:
                work = np.array([wt[lo:hi].sum() for lo, hi in parts])
                assert work.max() <= wt.sum() / world + wt.max()                # within one group of the ideal
                count = np.array([wt[slice(*tcw.shard_groups(n_groups, r, world))].sum() for r in range(world)])
                assert work.max() <= count.max() + 1e-9                         # never worse than the equal-count cut
    # zero and uniform weights reduce to the equal-count cut
    assert [tcw.shard_groups(12, r, 4, weights=np.zeros(12)) for r in range(4)] == [tcw.shard_groups(12, r, 4) for r in range(4)]
    assert [tcw.shard_groups(12, r, 4, weights=np.ones(12)) for r in range(4)] == [tcw.shard_groups(12, r, 4) for r in range(4)]
    with pytest.raises(ValueError):
        tcw.shard_groups(12, 0, 4, weights=np.ones(11))


def test_group_work_tracks_the_oracles_in_band_lookups():
    """group_work is an estimate (no Doppler) of what the oracle counts exactly; on cfg1 and on a cfg4-like
    grid whose small-tau tracks leave the band early, they agree to a fraction of a percent per group."""
    w = tcw_inputs.make_workload("cfg1")
    est = tcw.group_work(tcw.Grid.of(w), w.timestamps, w.T_sft, w.f_min, w.n_bins)
    ref = oracle.evaluate(w)
    exact = ref.n_inband.reshape(w.n_groups, len(w.f0)).sum(axis=1)
    assert est.shape == exact.shape
    assert np.all(np.abs(est - exact) <= 0.01 * exact.max() + len(w.f0))
    assert exact.min() < exact.max() and np.corrcoef(est, exact)[0, 1] > 0.999
