"""The N > 1 path of bench.py on CPU: world_size 2, gloo backend (the sharding has no data-path collective,
so what is tested is the slice partition and the max-over-ranks timing reduction)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1009_2288_b200 import shard


def test_slice_partitions():
    assert list(shard.slice_range(0, 2, 64)) == list(range(64))
    assert list(shard.slice_range(1, 2, 64)) == list(range(64, 128))
    parts = shard.split_slices(10, 4)
    assert [len(p) for p in parts] == [3, 3, 2, 2]
    assert [i for p in parts for i in p] == list(range(10))
    assert shard.split_slices(0, 2) == [range(0, 0), range(0, 0)]
    with pytest.raises(ValueError):
        shard.slice_range(2, 2, 4)
    assert shard.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]      # no process group: identity


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from ctr_inputs import make_case, scaled_config
        cfg = scaled_config("c1", batch=2)
        mine = shard.slice_range(rank, world, cfg.batch)
        case = make_case(cfg, slices=mine, raster=False)
        ms = 10.0 + 5.0 * rank                                   # rank 1 is the slow one
        value, ms_max = shard.job_throughput(cfg.batch, world, ms)
        # per-rank checksum of the seeded inputs, gathered: shards must be disjoint and seed-stable
        s = torch.tensor([float(case["sino"].sum())], dtype=torch.float64)
        got = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(got, s)
        if rank == 0:
            out.put((value, ms_max, [float(g) for g in got], list(mine)))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    value, ms_max, sums, mine = out.get()
    assert ms_max == 15.0 and value == pytest.approx(2 * 2 / 15e-3)
    assert mine == [0, 1]
    from ctr_inputs import make_case, scaled_config
    cfg = scaled_config("c1", batch=2)
    want = [float(make_case(cfg, slices=range(2 * r, 2 * r + 2), raster=False)["sino"].sum()) for r in range(2)]
    assert sums == pytest.approx(want, rel=1e-12) and sums[0] != sums[1]
