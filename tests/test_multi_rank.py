"""Host logic of the N>1 path on CPU (gloo, world_size 2): rays are independent, so ranks take
disjoint contiguous ray ranges (nif_inputs.shard_range) with no data-path collective; only the
timing reduction (max over ranks) and an optional gather of per-rank results go through
torch.distributed.  The per-rank "query" here is the CPU oracle's traversal -- this test checks
the sharding arithmetic and the rendezvous/reduction code, not a kernel."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import nif_inputs as I


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 128, 1000, 2_073_600):
        for world in (1, 2, 3, 8):
            spans = [I.shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            for (a0, a1), (b0, b1) in zip(spans, spans[1:]):
                assert a1 == b0 and a0 <= a1
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, n: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import Oracle
        cfg = I.get_config(0)
        orc = Oracle()
        occ = I.occupancy(cfg)
        pose = I.poses(cfg)[0]
        lat = orc.deform_lattice(cfg.nv, float(pose[0]), float(pose[1]))
        bvh = orc.bvh_build(cfg.nv, occ, lat)
        o, d = I.rays(cfg, 0, n=n)
        b, e = I.shard_range(n, rank, world)
        vid, ti, to = bvh.traverse(o[b:e], d[b:e])
        # what bench.py does with its device time: max over ranks
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        hits = torch.tensor([int((vid >= 0).sum())], dtype=torch.int64)
        dist.all_reduce(hits, op=dist.ReduceOp.SUM)
        gathered = [None] * world
        dist.all_gather_object(gathered, (b, e, vid))
        if rank == 0:
            full = np.concatenate([g[2] for g in sorted(gathered, key=lambda g: g[0])])
            np.save(os.path.join(out_dir, "vid.npy"), full)
            np.save(os.path.join(out_dir, "meta.npy"), np.array([t.item(), hits.item()]))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_ranks_shard_rays_without_exchange(tmp_path, oracle):
    n, world = 1001, 2                                   # odd count: ragged shards
    mp.spawn(_worker, args=(world, _free_port(), n, str(tmp_path)), nprocs=world, join=True)
    cfg = I.get_config(0)
    occ = I.occupancy(cfg)
    pose = I.poses(cfg)[0]
    lat = oracle.deform_lattice(cfg.nv, float(pose[0]), float(pose[1]))
    o, d = I.rays(cfg, 0, n=n)
    vid, _, _ = oracle.bvh_build(cfg.nv, occ, lat).traverse(o, d)
    got = np.load(tmp_path / "vid.npy")
    t_max, hits = np.load(tmp_path / "meta.npy")
    assert np.array_equal(got, vid)                      # sharded == single rank, ray for ray
    assert t_max == world and hits == int((vid >= 0).sum())


# ---- what bench.py actually does at N > 1: every rank runs the whole frame (replicas, weak scaling), the
# slowest rank's device time is taken (max over ranks) and the whole-job value is world x rays / that time ----
def _bench_worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        n_rays = 2_073_600
        my_ms = 0.9 + 0.3 * rank                        # stand-in for this rank's device-timed elapsed time
        dist.barrier()
        ms = bench.max_over_ranks(my_ms, dist)
        value = bench.whole_job_value(world, n_rays, ms)
        if rank == 0:
            np.save(os.path.join(out_dir, "bench.npy"), np.array([ms, value]))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_bench_aggregate_is_world_times_rays_over_slowest_rank(tmp_path):
    import bench
    world = 2
    mp.spawn(_bench_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    ms, value = np.load(tmp_path / "bench.npy")
    assert ms == pytest.approx(1.2)                      # the slowest of 0.9 and 1.2
    assert value == pytest.approx(2 * 2_073_600 / 1.2e-3 / 1e6)
    # single process: identity
    assert bench.max_over_ranks(3.5) == 3.5 and bench.whole_job_value(1, 1000, 1.0) == pytest.approx(1.0)


def test_bench_gpus_flag_reexecs_under_torchrun(monkeypatch):
    """`python bench.py --gpus 2` run plainly must become two ranks (torch.distributed.run), not time one GPU."""
    import subprocess, sys
    import bench
    calls = []
    monkeypatch.setattr(subprocess, "call", lambda cmd: calls.append(cmd) or 0)
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "2", "--steps", "3"])
    with pytest.raises(SystemExit) as e:
        bench.main()
    assert e.value.code == 0 and len(calls) == 1
    cmd = calls[0]
    assert "torch.distributed.run" in cmd and "--nproc-per-node=2" in cmd and "127.0.0.1" in cmd
    assert cmd[-4:] == ["--gpus", "2", "--steps", "3"]


def test_bench_reads_its_counts_from_the_committed_ncu_exports():
    """roofline counts come from profiles/*.csv (ncu --page raw --csv), not from constants in bench.py"""
    import bench
    for cfg_id in (1, 4):
        c = bench.ncu_counts(cfg_id, "compose")
        assert c is not None and c["file"].startswith("profiles/")
        for k in ("l1_wavefronts", "l2_sectors", "dram_bytes_read", "hit_rays_per_launch"):
            assert c[k] > 0, (cfg_id, k)
    assert bench.ncu_counts(0, "compose") is None       # no export for this config: bench falls back and says so
