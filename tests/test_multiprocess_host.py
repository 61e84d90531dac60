"""The N > 1 path of bench.py on CPU: two processes, gloo backend, 127.0.0.1.  The gridding path
shards by channel block with no data-path collective, so what has to hold is
host logic: every rank gets its own disjoint band, the whole-job figure is (units of all ranks) /
(slowest rank's device time), and only rank 0 reports."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parents[1]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, str(ROOT))
    import bench
    import synth
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        shard = bench.shard_plan(world, rank)
        assert shard["collective"] is None
        wl = synth.make_workload(1, n_time=1, band=shard["band"])
        assert abs(wl.freq[0] - (140.0e6 + rank * 32 * 40.0e3)) < 1e-3          # config 1: 32 x 40 kHz per band
        # every rank's band, gathered: disjoint and contiguous
        lo_hi = torch.tensor([wl.freq.min(), wl.freq.max()], dtype=torch.float64)
        bands = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(bands, lo_hi)
        for a, b in zip(bands[:-1], bands[1:]):
            assert a[1] < b[0] and abs((b[0] - a[1]).item() - 40.0e3) < 1e-3
        # per-rank device time and units -> whole-job aggregate (max over ranks, sum of units)
        ms = torch.tensor([10.0 + 5.0 * rank], dtype=torch.float64)
        units = torch.tensor([float(wl.n_vis * wl.support[0] ** 2)], dtype=torch.float64)
        all_ms = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        all_units = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(all_ms, ms)
        dist.all_gather(all_units, units)
        agg = bench.aggregate([float(x) for x in all_ms], [float(x) for x in all_units], steps=4)
        assert agg["ms_total"] == 10.0 + 5.0 * (world - 1)
        assert agg["ms_per_step"] == agg["ms_total"] / 4
        expect = sum(float(x) for x in all_units) * 4 / (agg["ms_total"] * 1e-3)
        assert abs(agg["value"] - expect) <= 1e-9 * expect
        dist.barrier()
        if rank == 0:
            (Path(out_dir) / "rank0.txt").write_text(repr(agg["value"]))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_channel_block_sharding(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert (tmp_path / "rank0.txt").exists()
    assert len(list(tmp_path.iterdir())) == 1          # rank 0 alone reports


def test_shard_plan_rejects_bad_rank_and_reference_arm_is_rank0_only():
    sys.path.insert(0, str(ROOT))
    import bench
    with pytest.raises(ValueError):
        bench.shard_plan(2, 2)
    assert bench.shard_plan(8, 7)["f0_hz"] == 140.0e6 + 7 * 768 * 40.0e3
    # aggregate: weak scaling -- doubling ranks at equal time doubles the value
    a1 = bench.aggregate([20.0], [1e9], steps=2)
    a2 = bench.aggregate([20.0, 20.0], [1e9, 1e9], steps=2)
    assert np.isclose(a2["value"], 2 * a1["value"])


# ---- row f4: the deterministic sum of the per-rank grids (paper_1003_5575_b200/mfs.py) ----------------
def _sum_parts_cpu(parts):
    """What gridder_sum_parts computes, written out with torch CPU ops (the tests' stand-in for the kernel)."""
    acc = torch.zeros(parts.shape[1], dtype=torch.float64)
    for p in range(parts.shape[0]):
        acc += parts[p].double()
    return acc.float()


def _mfs_worker(rank, world, port, out_dir, shape):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, str(ROOT))
    from paper_1003_5575_b200 import mfs
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        grids = [torch.from_numpy(np.random.default_rng(100 + r).standard_normal(shape).astype(np.float32) * 10.0 ** r)
                 for r in range(world)]
        mine = grids[rank].clone()
        out = mfs.reduce_grids(mine, sum_parts=_sum_parts_cpu)
        assert out is mine
        expect = torch.zeros(shape, dtype=torch.float64)
        for r in range(world):                               # rank order, double, one rounding
            expect += grids[r].double()
        assert torch.equal(mine, expect.float()), "not the fixed-order FP64 sum"
        np.save(Path(out_dir) / f"sum{rank}.npy", mine.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,shape", [(2, (4, 6, 6, 2)), (3, (4, 5, 5, 2)), (2, (1, 1, 1, 2))])
def test_reduce_grids_is_the_fixed_order_sum_on_every_rank(tmp_path, world, shape):
    mp.spawn(_mfs_worker, args=(world, _free_port(), str(tmp_path), shape), nprocs=world, join=True)
    sums = [np.load(tmp_path / f"sum{r}.npy") for r in range(world)]
    for s in sums[1:]:
        assert np.array_equal(s, sums[0])                    # the same bits on every rank


def test_slice_len_covers_and_is_float4_aligned():
    sys.path.insert(0, str(ROOT))
    from paper_1003_5575_b200 import mfs
    for numel in (1, 2, 7, 8, 288, 4 * 4096 * 4096 * 2):
        for world in (1, 2, 3, 8):
            L = mfs.slice_len(numel, world)
            assert L % 4 == 0 and world * L >= numel and world * (L - 4) < numel


def test_bench_gpus_n_starts_its_own_ranks(repo_root):
    """`python bench.py --gpus 2` with no launcher around it starts 2 ranks itself (torch.distributed.run on
    127.0.0.1); the line rank 0 prints says n_gpus = 2 and every rank got its own band."""
    import json
    import subprocess
    import sys
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, str(repo_root / "bench.py"), "--gpus", "2", "--spawn-check"], env=env,
                         capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    line = [l for l in res.stdout.splitlines() if l.startswith("{")][-1]
    out = json.loads(line)
    assert out["n_gpus"] == out["requested_gpus"] == 2
    assert out["f0_hz"] == [140.0e6, 140.0e6 + 768 * 40.0e3]
