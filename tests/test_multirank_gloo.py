"""world_size-2 coverage of bench.py's multi-rank host logic on CPU (gloo): replicas only
(multi-GPU): every rank runs its own seeded copy, the timing is the max over ranks,
value = units of all ranks / that time, rank 0 alone reports.  No GPU, no libkc call."""
import json
import os
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # replicas: each rank draws its own trajectories (seed shifted by rank), same shapes
        traj = bench.build_trajectories("cfg1", 2, seed_shift=rank)
        ps, _ = traj["walk"]
        local_ms = 10.0 * (rank + 1)                       # rank 1 is the slow one
        ms_max, units = bench.aggregate_over_ranks(local_ms, ps[0].shape[0] * 2, torch.device("cpu"))
        digest = torch.tensor([float(np.float64(ps[0]).sum())], dtype=torch.float64)
        both = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(both, digest)
        if rank == 0:
            json.dump(dict(ms_max=ms_max, units=units, digests=[float(b) for b in both],
                           shape=list(ps[0].shape)), open(out, "w"))
    finally:
        dist.barrier()
        dist.destroy_process_group()


def test_replicas_max_over_ranks_and_whole_job_units(tmp_path):
    out = str(tmp_path / "r.json")
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["ms_max"] == 20.0                               # the slowest rank sets the time
    assert r["units"] == 2 * 2 * r["shape"][0]               # whole-job units: both ranks' points
    assert r["digests"][0] != r["digests"][1]                # independently seeded copies


def test_schedule_splits_steps_over_families():
    import bench
    fams, per = bench.schedule("cfg2", 100)
    assert len(fams) == 5 and per == [20] * 5
    fams, per = bench.schedule("cfg2", 7)
    assert sum(per) == 7 and max(per) - min(per) <= 1


def test_reference_arm_other_ranks_exit_silently():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "3"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


# ---- the all-pairs pass sharded by query ----------------------------------------
def test_query_slices_partition_the_ids():
    from paper_2606_18314_b200.sharding import query_slice, slice_width
    for n, world in [(1048576, 1), (1048576, 2), (1048576, 8), (1001, 2), (10, 3), (2, 4), (0, 2), (7, 7)]:
        cuts = [query_slice(n, r, world) for r in range(world)]
        assert cuts[0][0] == 0 and cuts[-1][1] == n
        assert all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))          # contiguous, in rank order
        sizes = [b - a for a, b in cuts]
        assert max(sizes) - min(sizes) <= 1 and max(sizes) == slice_width(n, world) and sizes == sorted(sizes, reverse=True)
    import pytest
    with pytest.raises(ValueError):
        query_slice(10, 2, 2)


def _shard_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    from paper_2606_18314_b200.sharding import gather_columns, query_slice
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ok = True
        for n in (1001, 4096, 5):
            # the "certificates" of id i are a known function of i; a rank fills only its own slice
            # (the rest of its buffer holds garbage), then the ranks exchange the columns
            want = torch.stack([torch.arange(n, dtype=torch.int32) * (k + 3) + k for k in range(5)])
            buf = torch.full((5, (n + 3) // 4 * 4), -777, dtype=torch.int32)
            lo, hi = query_slice(n, rank, world)
            buf[:, lo:hi] = want[:, lo:hi]
            gather_columns(buf, n)
            ok &= bool(torch.equal(buf[:, :n], want))
            ok &= bool((buf[:, n:] == -777).all())                        # the padding is not touched
        flags = [torch.zeros(1, dtype=torch.int32) for _ in range(world)]
        dist.all_gather(flags, torch.tensor([int(ok)], dtype=torch.int32))
        if rank == 0:
            json.dump(dict(ok=[int(f) for f in flags]), open(out, "w"))
    finally:
        dist.barrier()
        dist.destroy_process_group()


def test_sharded_certificates_are_gathered_on_every_rank(tmp_path):
    for world in (2, 3):
        out = str(tmp_path / f"s{world}.json")
        port = 31500 + (os.getpid() + world) % 2000
        mp.spawn(_shard_worker, args=(world, port, out), nprocs=world, join=True)
        assert json.load(open(out))["ok"] == [1] * world


def test_gather_without_a_process_group_is_the_identity():
    from paper_2606_18314_b200.sharding import gather_columns
    buf = torch.arange(20, dtype=torch.int32).reshape(5, 4)
    assert gather_columns(buf, 4) is buf and torch.equal(buf, torch.arange(20, dtype=torch.int32).reshape(5, 4))
