"""Host logic of bench.py that needs no GPU: the max-over-ranks timing rule on a 2-rank gloo group, the replica
aggregate, the out-of-core size fallback and the clock-reason decoding."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402
import workload as W  # noqa: E402


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = [10.0 + 5.0 * rank, 3.0 - rank]                # rank 1 is slower on the first, faster on the second
        out = bench.max_over_ranks(ms, dist, "cpu")
        q.put((rank, out, bench.aggregate_value(1000.0, world, out[0])))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_two_rank_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, out, agg in res:
        assert out == [15.0, 3.0]                           # the slowest rank's time on every entry, on every rank
        assert agg == pytest.approx(2 * 1000.0 / 15.0e-3)   # replicas: units of all ranks / slowest time


def test_max_over_ranks_without_group_is_identity():
    assert bench.max_over_ranks([1.5, 2.5], None, "cpu") == [1.5, 2.5]
    assert bench.aggregate_value(10.0, 1, 2.0) == pytest.approx(5000.0)


def test_ooc_config_cuts_whole_brick_layers():
    cfg = W.get_config(5)
    same, note = bench.ooc_config(cfg, 3072)
    assert same.dims == cfg.dims and note == "full size"
    cut, note = bench.ooc_config(cfg, 700)
    assert cut.dims == (4096, 4096, 512) and cut.brick == 256 and "cut" in note
    assert cut.recipe.n_sources == cfg.recipe.n_sources * 512 // 3072
    assert cut.n_views == cfg.n_views and cut.width == cfg.width and cut.out_of_core


def test_config_block_names_the_workload():
    b = bench.config_block(W.get_config(2))
    assert "512x512x1024" in b["workload"] and b["cube_bytes"] == 1 << 30 and "model" not in b
