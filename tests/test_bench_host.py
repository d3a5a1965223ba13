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


# ---------------------------------------------------------------------------------- the whole flow, emulated
class _NoClocks:
    def start(self):
        pass

    def finish(self):
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["emulated"]}


class SimtRig:
    """bench.TorchCudaRig's interface on the host emulation of the library (tests/simt): buffers are guarded host
    allocations, "events" are host clock readings (the emulated runtime is synchronous)."""
    name = "simt"
    stream_arg = 0

    def __init__(self):
        sys.path.insert(0, os.path.join(ROOT, "tests", "simt"))
        import simt_lib
        self.lib = simt_lib

    def host_empty(self, shape, dtype=np.float32, pinned=True):
        return self.lib.Buffer(shape, dtype, device=False)

    def dev_empty(self, shape, dtype=np.float32):
        return self.lib.Buffer(shape, dtype, device=True)

    def to_device(self, host):
        return self.lib.Buffer.of(host.array, device=True)

    def as_numpy(self, host):
        return host.array

    def read(self, t):
        return np.array(t.array, copy=True)

    def event(self):
        return [0.0]

    def record(self, e):
        import time
        e[0] = time.perf_counter()

    def elapsed_ms(self, a, b):
        return (b[0] - a[0]) * 1e3

    def synchronize(self):
        pass

    stream_synchronize = empty_cache = synchronize

    def copy_h2d(self, d, h):
        d.array[...] = h.array

    def clock_sampler(self):
        return _NoClocks()


def _args(**kw):
    import argparse
    d = dict(gpus=1, steps=1, warmup=1, impl="ours", config=2, no_cpu=False, no_e2e=False, cpu_seconds=0.3, ooc_nz=0,
             ooc_resident_frac=0.25, path=0, lag=-1, no_zcopy=False, row_loads=-1, views=2)
    d.update(kw)
    return argparse.Namespace(**d)


@pytest.mark.parametrize("number,scale", [(2, 1 / 16), (3, 1 / 32), (4, 1 / 64), (5, 1 / 32)])
def test_bench_flow_and_json_line_in_emulation(number, scale, capsys):
    """bench.py's own measurement flow — warm-up, timed steps, per-render events, cold cameras, the end-to-end leg with
    host buffers, roofline arithmetic, cpu_baseline — executed on a scaled config against the emulated library: the
    line the driver parses is assembled without an exception and carries every key of the contract."""
    import json
    rig = SimtRig()
    cfg = W.get_config(number, scale=scale)
    if number == 5:                                     # 48 bricks instead of cfg5's 3072: one emulated launch per brick
        from dataclasses import replace
        cfg = replace(cfg, brick=32, recipe=replace(cfg.recipe, nx=128, ny=128, nz=96), name="cfg5-test")
    with rig.lib.emulated():
        line = bench.run_ours(_args(config=number), rig=rig, cfg=cfg)
    printed = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert printed["metric"] == line["metric"] == "voxel_samples_per_s" and printed["unit"] == "samples/s"
    for key in ("value", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline", "dtype",
                "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert key in printed, key
    assert printed["value"] > 0 and printed["gpu_launches"] > 0 and printed["dtype"] == "f32" and printed["vs_baseline"] is None
    assert "workload" in printed["config"] and "model" not in printed["config"]
    r = printed["roofline"]
    assert r["bound"] in ("hbm", "alu", "host_link") and r["achieved"] > 0 and r["peak"] > 0 and "traffic" in r
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    e = printed["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] >= 4 * np.prod(cfg.dims) and e["d2h_bytes_per_step"] > 0
    c = printed["cpu_baseline"]
    assert c["kind"] == "oracle" and c["value"] > 0 and c["cores"] >= 1 and "sample" in c
    if number != 5:
        assert printed["data_passes"]["summary_ms"] > 0 and printed["data_passes"]["statistics_gbs"] > 0
        assert printed["render_ms_cold"] is not None or cfg.sort_last
        assert len(printed["render_ms_by_view"]) == 2 * len(cfg.modes)


def test_reference_arm_line(capsys):
    """--impl reference: the oracle on the host cores, same metric / unit / config block, the keys the contract adds."""
    import json
    line = bench.run_reference(_args(impl="reference", steps=2, warmup=1), cfg=W.get_config(4, scale=1 / 64))
    printed = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert printed == json.loads(json.dumps(line))
    assert printed["impl"] == "reference" and printed["metric"] == "voxel_samples_per_s" and printed["value"] > 0
    assert printed["cpu_baseline"]["kind"] == "oracle" and printed["cpu_baseline"]["value"] == printed["value"]
    assert printed["e2e"] == {"value": printed["value"], "unit": "samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
