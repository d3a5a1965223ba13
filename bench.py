#!/usr/bin/env python
"""bench.py — throughput of the hot path on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A *step* is one pass of the whole hot path over one synthetic cube: the data-summary pass
(vr_minmax_histogram: min/max, then the 256-bin histogram over [min,max]), vr_set_transfer_function
with that range, and vr_render of every orbit view of the config.  Default workload: cfg4, the largest
single-GPU config of BASELINE.json (2048x2048x4096 = 64 GiB resident in HBM, 64 perspective orbit views
3840x2160, step 1, emission-absorption with early ray termination at alpha 0.99); --config 2|3|5 select
the others.

value  = nominal voxel samples of all rendered views / step time, cube resident in HBM when the
         timed region starts (CUDA events on the launching stream, max over ranks).
e2e    = the same metric through the C ABI with HOST buffers: every step creates the handle on the
         pinned host cube (the whole cube host->device inside the timed region), runs the same calls with
         pinned host outputs (summary and images copied device->host) and destroys the handle.
Multi-GPU: the path does not shard (north_star: one GPU, no collectives) => N independent replicas,
"scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

ALU_SLOTS_PER_EA_SAMPLE = 64      # issue slots of one EA sample
ALU_SLOTS_PER_MIP_SAMPLE = 45
N_SM, LANES_PER_SM = 148, 128     # B200 (B200_PROFILING.md): 148 SMs, 4 x 32 fp32/int lanes each


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


def ncu_traffic(cfg_number: int):
    """DRAM bytes (read + write) per launch of the ray-march kernel from the committed ncu --set full summary
    (profiles/ncu_traffic.csv: config,kernel,dram_read_bytes,dram_write_bytes,source), or None."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(p):
        return None
    best = None
    with open(p) as f:
        for ln in f:
            c = [x.strip() for x in ln.split(",")]
            if len(c) >= 4 and c[0] == f"cfg{cfg_number}" and c[1].startswith("k_rows"):
                try:
                    best = float(c[2]) + float(c[3])
                except ValueError:
                    pass
    return best


# ---------------------------------------------------------------------------------- clocks
_REASONS = {0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x10: "sync_boost",
            0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown"}


class ClockSampler(threading.Thread):
    """Polls NVML for SM clock and clock-event reasons while the timed region runs."""

    def __init__(self, index: int, period: float = 0.1):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._halt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    bits = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    bits = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for b, name in _REASONS.items():
                    if bits & b:
                        self.reasons.add(name)
            except Exception:
                pass
            self._halt.wait(self.period)

    def finish(self) -> dict:
        self._halt.set()
        if self.is_alive():
            self.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml_unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def physical_gpu_index(local: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except Exception:
            return local
    return local


def max_over_ranks(values, dist, device):
    """Element-wise MAX of a list of floats over all ranks (identity without a process group): the timing rule
    of the contract — every multi-rank number is the slowest rank's."""
    if dist is None:
        return [float(v) for v in values]
    import torch
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def aggregate_value(units_per_rank: float, world: int, ms_step: float) -> float:
    """Whole-job throughput of N independent replicas (weak scaling): units all ranks processed / slowest time."""
    return world * units_per_rank / (ms_step * 1e-3)


# ---------------------------------------------------------------------------------- device rig
_NP2TORCH = {"float32": "float32", "uint8": "uint8"}


class TorchCudaRig:
    """Everything bench.py needs from the device side — buffers, events on the launching stream, synchronisation —
    behind one small object, so that tests/test_bench_host.py can execute the whole measurement flow (and the JSON
    line it assembles) against the host emulation of the library with a rig of the same interface."""
    name = "cuda"

    def __init__(self, local: int):
        import torch
        if not torch.cuda.is_available():
            raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
        torch.cuda.set_device(local)
        self.torch, self.local = torch, local
        self.stream = torch.cuda.current_stream()
        self.stream_arg = self.stream                       # what the binding's `stream=` takes

    def _dt(self, dtype):
        return getattr(self.torch, _NP2TORCH[np.dtype(dtype).name])

    def host_empty(self, shape, dtype=np.float32, pinned=True):
        return self.torch.empty(tuple(shape), dtype=self._dt(dtype), pin_memory=pinned)

    def dev_empty(self, shape, dtype=np.float32):
        return self.torch.empty(tuple(shape), dtype=self._dt(dtype), device="cuda")

    def to_device(self, host):
        return host.cuda()

    def as_numpy(self, host):
        return host.numpy()

    def read(self, t):
        """Synchronise and return the bytes of a device or pinned-host buffer as a numpy array."""
        self.torch.cuda.synchronize()
        return (t.cpu() if t.is_cuda else t).numpy()

    def event(self):
        return self.torch.cuda.Event(enable_timing=True)

    def record(self, e):
        e.record(self.stream)

    def elapsed_ms(self, a, b) -> float:
        return float(a.elapsed_time(b))

    def synchronize(self):
        self.torch.cuda.synchronize()

    def stream_synchronize(self):
        self.stream.synchronize()

    def empty_cache(self):
        self.torch.cuda.empty_cache()

    def copy_h2d(self, d, h):
        d.copy_(h, non_blocking=True)

    def clock_sampler(self):
        return ClockSampler(physical_gpu_index(self.local))


def read_summary(rig, buf, nbins: int = 256):
    import paper_1111_6661_b200 as vr
    raw = np.ascontiguousarray(rig.read(buf)).tobytes()[: 32 + 8 * nbins]
    return np.frombuffer(raw, dtype=vr.summary_dtype(nbins))[0]


# ---------------------------------------------------------------------------------- workload
def make_host_cube(cfg, rig=None, pinned=True):
    """The config's seeded cube in (pinned) host memory, filled in z-slabs by the shared generator."""
    import workload as W
    nx, ny, nz = cfg.dims
    if rig is None:
        import torch
        t = torch.empty((nz, ny, nx), dtype=torch.float32, pin_memory=pinned)
    else:
        t = rig.host_empty((nz, ny, nx), np.float32, pinned)
    gen = W.CubeGenerator(cfg.recipe)
    slab = max(1, (1 << 28) // (nx * ny))
    for z0 in range(0, nz, slab):
        z1 = min(nz, z0 + slab)
        gen.fill_ptr(t.data_ptr() + 4 * z0 * ny * nx, z0, z1)
    return t


def modes_of(cfg):
    import paper_1111_6661_b200 as vr
    return [vr.VR_EA if m == "ea" else vr.VR_MIP for m in cfg.modes]


# ---------------------------------------------------------------------------------- reference arm
def cpu_oracle_rate(cfg, host_np, tf, vmin, vmax, budget_s=15.0, view=0):
    """Times the oracle as it stands (f32-canonical, OpenMP on all host cores) on a pixel lattice of
    one view of the workload; returns samples/s and what the sample was."""
    import oracle as O
    cam = cfg.camera(view)
    H, Wd = cam.height, cam.width
    mode = O.EA if "ea" in cfg.modes else O.MIP

    def run(stride):
        mask = np.zeros((H, Wd), dtype=np.uint8)
        mask[stride // 2::stride, stride // 2::stride] = 1
        t0 = time.perf_counter()
        r = O.render(host_np, cam, mode, tf, vmin, vmax, mask=mask)
        dt = time.perf_counter() - t0
        n = r.n_ert if mode == O.EA else r.n_nominal
        return r.n_nominal, n, dt

    n_nom, n_done, dt = run(16)                       # calibration pass
    rate = max(n_nom / max(dt, 1e-6), 1.0)
    total = n_nom * 256.0
    stride = int(np.clip(np.ceil(np.sqrt(total / (rate * budget_s))), 1, 16))
    if stride < 16:
        n_nom, n_done, dt = run(stride)
    return {"value": n_nom / dt, "unit": "samples/s", "cores": O.num_threads(), "kind": "oracle",
            "sample": f"{cfg.name} view {view}, every {stride}th pixel in x and y ({n_nom} nominal samples, "
                      f"{n_done} evaluated before ERT, {dt:.2f} s), f32-canonical oracle, OpenMP",
            "seconds": dt, "n_samples": int(n_nom)}


def run_reference(args, cfg=None):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return None
    import workload as W
    import oracle as O
    if cfg is None:
        cfg = W.get_config(args.config)
        if cfg.out_of_core:                      # the linear cube of cfg5 does not fit the host: same cut as our arm
            cfg, _ = ooc_config(cfg, args.ooc_nz)
    host = make_host_cube(cfg, None, pinned=False).numpy()
    s = O.minmax_hist(host[: max(2, min(host.shape[0], (1 << 27) // (host.shape[1] * host.shape[2])))])
    tf = W.tf_haze(cfg.dims, cfg.step)
    budget = 45.0 / max(args.steps + args.warmup, 1)
    times, n = [], 0
    for it in range(args.warmup + args.steps):
        r = cpu_oracle_rate(cfg, host, tf, float(s.vmin), float(s.vmax), budget_s=min(budget, 15.0),
                            view=it % cfg.n_views)
        if it >= args.warmup:
            times.append(r["seconds"]); n += r["n_samples"]
    value = n / sum(times)
    line = {"impl": "reference", "metric": "voxel_samples_per_s", "value": value, "unit": "samples/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * sum(times) / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": config_block(cfg, "bounded sample per step: one orbit view on a pixel lattice"),
            "cpu_baseline": {"value": value, "unit": "samples/s", "cores": O.num_threads(), "kind": "oracle",
                             "sample": r["sample"]},
            "e2e": {"value": value, "unit": "samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return line


def config_block(cfg, note=""):
    nx, ny, nz = cfg.dims
    return {"workload": f"{cfg.name}: {nx}x{ny}x{nz} float32 noise+{cfg.recipe.n_sources} sources, "
                        f"{cfg.n_views} orbit views {cfg.width}x{cfg.height}, step {cfg.step}, "
                        f"modes {'+'.join(cfg.modes)}, ERT {cfg.ert_alpha}, TF_HAZE, + min/max & 256-bin histogram",
            "cube_bytes": 4 * nx * ny * nz, "brick": cfg.brick, "views": cfg.n_views,
            "image": [cfg.width, cfg.height], "l2": "inputs larger than L2 (cube >= 1 GiB, orbit views evict each other)",
            "parallelism": "replicas", "note": note}


# ---------------------------------------------------------------------------------- our arm
def run_ours(args, rig=None, cfg=None):
    """`rig` / `cfg`: the emulated rig and a scaled config of tests/test_bench_host.py; None = B200 and --config."""
    import paper_1111_6661_b200 as vr
    import workload as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if rig is None:
        rig = TorchCudaRig(local)
    dist = None
    if world > 1:
        import torch
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    if cfg is None:
        cfg = W.get_config(args.config)
    if cfg.out_of_core:
        if dist is not None:
            dist.destroy_process_group()
        return run_ours_ooc(args, cfg, rig)
    nx, ny, nz = cfg.dims
    n_vox = nx * ny * nz
    host = make_host_cube(cfg, rig, pinned=True)
    dev = rig.to_device(host)
    modes = modes_of(cfg)
    view_ids = list(range(cfg.n_views))
    if args.views > 0:
        view_ids = view_ids[:: max(1, cfg.n_views // args.views)][: args.views]      # spread over the orbit
    cams = [cfg.camera(v) for v in view_ids]
    cam_structs = [vr.make_camera(c) for c in cams]
    samples_view = [W.nominal_samples(c, cfg.dims) for c in cams]
    samples_step = sum(samples_view) * len(modes)
    frames_step = len(cams) * len(modes)

    vol = vr.Volume(dev, cfg.dims, brick=cfg.brick)
    if args.path:
        vol.set_option(vr.VR_OPT_RENDER_PATH, args.path)
    if args.lag >= 0:
        vol.set_option(vr.VR_OPT_LANE_LAG, args.lag)
    if args.no_zcopy:
        vol.set_option(vr.VR_OPT_ZFAST_COPY, 0)
    if args.row_loads >= 0:
        vol.set_option(vr.VR_OPT_ROW_LOADS, args.row_loads)
    sbuf = rig.dev_empty((32 + 8 * 256,), np.uint8)
    vol.minmax_histogram(256, out=sbuf, stream=rig.stream_arg)
    s = read_summary(rig, sbuf)
    vmin, vmax = float(s["vmin"]), float(s["vmax"])
    tf = W.tf_haze(cfg.dims, cfg.step)
    images = {m: rig.dev_empty((cfg.height, cfg.width, 4) if m == vr.VR_EA else (cfg.height, cfg.width)) for m in modes}

    ev_pairs = []                                    # (start, end) around every vr_render of the timed region
    quad_launches = []                               # per timed render: launches that used 16-byte row loads

    def step(record=False):
        vol.minmax_histogram(256, out=sbuf, stream=rig.stream_arg)
        vol.set_transfer_function(tf, vmin, vmax)
        n = 0
        for m in modes:
            for c in cam_structs:
                if record:
                    a, b = rig.event(), rig.event()
                    rig.record(a)
                vol.render(c, m, out=images[m], stream=rig.stream_arg)
                if record:
                    rig.record(b); ev_pairs.append((a, b))
                st = vol.stats()
                n += st["kernel_launches"]
                if record:
                    quad_launches.append(st["quad_launches"])
        return n

    def barrier():
        rig.synchronize()
        if dist is not None:
            dist.barrier()
            rig.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    clocks = rig.clock_sampler()
    clocks.start()
    launches0 = vol.stats()["total_kernel_launches"]
    e0, e1 = rig.event(), rig.event()
    rig.record(e0)
    for _ in range(args.steps):
        step(record=True)
    rig.record(e1)
    barrier()
    clk = clocks.finish()
    ms_total = rig.elapsed_ms(e0, e1)
    launches = vol.stats()["total_kernel_launches"] - launches0
    render_ms = [rig.elapsed_ms(a, b) for a, b in ev_pairs]
    path = vol.stats()["path"]
    zfast = vol.stats()["zfast_copy"]
    # cold cameras: one orbit at azimuths none of the steps above has seen (an interactively moving camera);
    # the per-frame host work of vr_render is O(1) (no per-camera plan, no cache), so this must equal render_ms
    cold_ms = []
    if not cfg.sort_last:
        for v_i in view_ids:
            c = vr.make_camera(W.orbit_camera(cfg.dims, v_i + 0.37, cfg.n_views, cfg.width, cfg.height, step=cfg.step,
                                              ert_alpha=cfg.ert_alpha))
            a, b = rig.event(), rig.event()
            rig.record(a); vol.render(c, modes[0], out=images[modes[0]], stream=rig.stream_arg); rig.record(b)
            cold_ms.append((a, b))
        rig.synchronize()
        cold_ms = [rig.elapsed_ms(a, b) for a, b in cold_ms]
    # the data passes on their own (outside the timed region): summary = min/max pass + histogram pass (8 B/voxel),
    # statistics = five passes (20 B/voxel); HBM-bound streams, reported against the same measured copy peak
    pass_ms = {}
    stbuf = rig.dev_empty((40,), np.uint8)
    for name, call in (("summary", lambda: vol.minmax_histogram(256, out=sbuf, stream=rig.stream_arg)),
                       ("statistics", lambda: vol.statistics(out=stbuf, stream=rig.stream_arg))):
        call(); rig.synchronize()
        a, b = rig.event(), rig.event()
        rig.record(a); call(); rig.record(b); rig.synchronize()
        pass_ms[name] = rig.elapsed_ms(a, b)
    ms_total = max_over_ranks([ms_total], dist, "cuda")[0]
    ms_step = ms_total / args.steps
    value = aggregate_value(samples_step, world, ms_step)

    # ---- end to end through the C ABI with host buffers (every step uploads the cube)
    h_sum = rig.host_empty((32 + 8 * 256,), np.uint8)
    h_img = {m: rig.host_empty(tuple(images[m].shape)) for m in modes}

    def e2e_step():
        with vr.Volume(host, cfg.dims, brick=cfg.brick, n_copy_streams=4) as hv:
            hv.minmax_histogram(256, out=h_sum, stream=rig.stream_arg)
            h2d = hv.stats()["h2d_bytes"]
            rig.stream_synchronize()
            hs = read_summary(rig, h_sum)
            hv.set_transfer_function(tf, float(hs["vmin"]), float(hs["vmax"]))
            d2h = 32 + 8 * 256
            for m in modes:
                for c in cam_structs:
                    hv.render(c, m, out=h_img[m], stream=rig.stream_arg)
                    d2h += hv.stats()["d2h_bytes"]
            rig.stream_synchronize()
        return h2d, d2h

    vol.close()
    del dev
    rig.empty_cache()
    e2e_steps = max(1, min(args.steps, 3))
    h2d = d2h = 0
    e2e_ms = float("nan")
    if not args.no_e2e:
        e2e_step()
        barrier()
        a, b = rig.event(), rig.event()
        rig.record(a)
        for _ in range(e2e_steps):
            h2d, d2h = e2e_step()
        rig.record(b)
        barrier()
        e2e_ms = rig.elapsed_ms(a, b)
    e2e_ms = max_over_ranks([e2e_ms], dist, "cuda")[0]
    e2e_value = aggregate_value(samples_step, world, e2e_ms / e2e_steps)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the ray-march kernel: one or two launches per vr_render)
    hbm_peak, sm_max_mhz, peak_src = measured_peaks()
    k_ms = float(np.mean(render_ms))
    ea_frac = sum(1 for m in modes if m == vr.VR_EA) / len(modes)
    slots = ALU_SLOTS_PER_EA_SAMPLE * ea_frac + ALU_SLOTS_PER_MIP_SAMPLE * (1 - ea_frac)
    samples_launch = float(np.mean(samples_view))
    bytes_launch = 4.0 * n_vox + 4.0 * cfg.width * cfg.height * (4 * ea_frac + (1 - ea_frac))
    alu_peak = N_SM * LANES_PER_SM * sm_max_mhz * 1e6              # lane-instructions / s
    hbm_floor_ms = bytes_launch / (hbm_peak * 1e9) * 1e3
    alu_floor_ms = slots * samples_launch / alu_peak * 1e3
    hbm_roof = {"bound": "hbm", "achieved": bytes_launch / (k_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "traffic": ncu_traffic(cfg.number), "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_src})",
                "algorithmic_bytes_per_launch": bytes_launch, "floor_ms": hbm_floor_ms}
    hbm_roof["frac"] = hbm_roof["achieved"] / hbm_peak
    alu_roof = {"bound": "alu", "achieved": slots * samples_launch / (k_ms * 1e-3) / 1e12, "peak": alu_peak / 1e12,
                "unit": "Tlane-instr/s", "traffic": None,
                "peak_source": f"{N_SM} SMs x {LANES_PER_SM} lanes x {sm_max_mhz:.0f} MHz (DESIGN.md §6)",
                "algorithmic_slots_per_sample": slots, "floor_ms": alu_floor_ms}
    alu_roof["frac"] = alu_roof["achieved"] / alu_roof["peak"]
    primary, other = (alu_roof, hbm_roof) if alu_floor_ms > hbm_floor_ms else (hbm_roof, alu_roof)
    kname = {1: "k_march_full (ray-major tiles)",
             2: "k_rows<PART> + k_composite (sort-last: one lane-mapped march per frame writes the per-brick fragments)",
             7: "k_rows (lane-mapped rows; one or two launches per vr_render)"}.get(path, f"vr_render path {path}")
    primary = dict(primary, kernel=kname, kernel_ms=k_ms, launches_timed=len(render_ms), zfast_copy=int(zfast))

    line = {"metric": "voxel_samples_per_s", "value": value, "unit": "samples/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": config_block(cfg, "" if len(view_ids) == cfg.n_views else f"ONLY views {view_ids} (profiling run)"),
            "clocks": clk,
            "e2e": {"value": e2e_value, "unit": "samples/s", "h2d_bytes_per_step": int(h2d),
                    "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps},
            "gpu_launches": int(launches),
            "roofline": primary, "roofline_other": other,
            "frames_per_s": world * frames_step / (ms_step * 1e-3),
            "render_ms": {"min": float(np.min(render_ms)), "median": float(np.median(render_ms)),
                          "mean": k_ms, "max": float(np.max(render_ms))},
            "render_ms_by_view": [round(float(np.mean(render_ms[v::frames_step])), 4) for v in range(frames_step)],
            "render_share_of_step": float(np.sum(render_ms)) / ms_total,
            "quad_launches_by_view": [int(q) for q in quad_launches[:frames_step]],
            "render_ms_cold": ({"mean": float(np.mean(cold_ms)), "max": float(np.max(cold_ms)),
                                "note": "one orbit at unseen azimuths, outside the timed region"} if cold_ms else None),
            "effective_hbm_gbs_per_frame": 4.0 * n_vox / (k_ms * 1e-3) / 1e9,
            "data_passes": {"summary_ms": pass_ms["summary"], "summary_gbs": 8.0 * n_vox / (max(pass_ms["summary"], 1e-9) * 1e-3) / 1e9,
                            "statistics_ms": pass_ms["statistics"],
                            "statistics_gbs": 20.0 * n_vox / (max(pass_ms["statistics"], 1e-9) * 1e-3) / 1e9,
                            "hbm_peak_gbs": hbm_peak, "note": "vr_minmax_histogram (2 passes) and vr_statistics (5 passes), "
                            "algorithmic bytes / device time, outside the timed region"},
            "samples_per_step": int(samples_step)}
    if world == 1 and not args.no_cpu:
        line["cpu_baseline"] = cpu_oracle_rate(cfg, rig.as_numpy(host), tf, vmin, vmax, budget_s=args.cpu_seconds)
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return line


# ---------------------------------------------------------------------------------- out-of-core arm (cfg5)
def host_mem_available() -> int:
    try:
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable:"):
                    return int(line.split()[1]) * 1024
    except Exception:
        pass
    return 64 << 30


def ooc_config(cfg, nz_arg: int):
    """cfg5 needs 4096x4096x3072 in pinned host memory as 256^3(+1) bricks = 209 GB.  When the box cannot pin
    that (SURVEY H7 fallback b) the spectral axis is cut to whole brick layers that fit a third of the available
    host memory; everything else (brick size, image, views, step, streams) is cfg5's."""
    from dataclasses import replace
    import workload as W
    nx, ny, nz = cfg.dims
    B = cfg.brick
    layer_bytes = 4 * W.bricked_halo_elems((nx, ny, B), B)
    if nz_arg <= 0:
        fit = int(host_mem_available() / 3 // layer_bytes)
        nz_arg = min(nz, max(1, fit) * B)
    if nz_arg >= nz:
        return cfg, "full size"
    nz_arg = max(B, nz_arg // B * B)
    rec = replace(cfg.recipe, nz=nz_arg, n_sources=max(1, cfg.recipe.n_sources * nz_arg // nz))
    return replace(cfg, recipe=rec, name=f"{cfg.name}@nz{nz_arg}"), f"spectral axis cut from {nz} to {nz_arg} channels: the box cannot pin the full 209 GB"


def measure_h2d_peak(rig, nbytes: int = 1 << 30) -> float:
    """Host-link peak as SURVEY 8(d) defines it: pinned 1 GiB cudaMemcpyAsync, best of 10, GB/s."""
    h = rig.host_empty((nbytes,), np.uint8)
    d = rig.dev_empty((nbytes,), np.uint8)
    best = 0.0
    for _ in range(10):
        a, b = rig.event(), rig.event()
        rig.record(a); rig.copy_h2d(d, h); rig.record(b); rig.synchronize()
        best = max(best, nbytes / (max(rig.elapsed_ms(a, b), 1e-6) * 1e-3) / 1e9)
    del h, d
    rig.empty_cache()
    return best


def run_ours_ooc(args, cfg, rig):
    """cfg5: the cube lives in pinned host memory as brick-major 256^3(+1 halo) bricks; a fixed part of the brick
    pool stays resident, the rest is streamed per frame in view order on 4 copy streams (A5).  `value` times steps
    on one handle (resident part already loaded); `e2e` creates the handle inside every step."""
    import paper_1111_6661_b200 as vr
    import workload as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if cfg.number == 5 and cfg.name == "cfg5":
        cfg, size_note = ooc_config(cfg, args.ooc_nz)
    else:
        size_note = "scaled test config"
    nx, ny, nz = cfg.dims
    B = cfg.brick
    n_el = W.bricked_halo_elems(cfg.dims, B)
    host = rig.host_empty((n_el,), np.float32, pinned=True)
    W.fill_bricked_halo_ptr(cfg.recipe, B, host.data_ptr())
    cube_bytes = 4 * n_el
    resident = int(args.ooc_resident_frac * cube_bytes)
    link_peak = measure_h2d_peak(rig, min(1 << 30, max(1 << 20, cube_bytes)))
    cams = [cfg.camera(v) for v in range(cfg.n_views)]
    cam_structs = [vr.make_camera(c) for c in cams]
    samples_step = sum(W.nominal_samples(c, cfg.dims) for c in cams)
    tf = W.tf_haze(cfg.dims, cfg.step)
    img = rig.dev_empty((cfg.height, cfg.width, 4))
    h_img = rig.host_empty((cfg.height, cfg.width, 4))
    h_sum = rig.host_empty((32 + 8 * 256,), np.uint8)
    frame_ms, frame_h2d, sum_ms, sum_h2d = [], [], [], []
    last_range = [0.0, 1.0]

    def step(vol, out_img, record):
        ev = [rig.event() for _ in range(2 + len(cam_structs))]
        rig.record(ev[0])
        vol.minmax_histogram(256, out=h_sum, stream=rig.stream_arg)
        h2d_s = vol.stats()["h2d_bytes"]
        rig.record(ev[1])
        rig.stream_synchronize()
        hs = read_summary(rig, h_sum)
        last_range[0], last_range[1] = float(hs["vmin"]), float(hs["vmax"])
        vol.set_transfer_function(tf, last_range[0], last_range[1])
        h2d_f = []
        for k, c in enumerate(cam_structs):
            vol.render(c, vr.VR_EA, out=out_img, stream=rig.stream_arg)
            h2d_f.append(vol.stats()["h2d_bytes"])
            rig.record(ev[2 + k])
        rig.stream_synchronize()
        if record:
            sum_ms.append(rig.elapsed_ms(ev[0], ev[1])); sum_h2d.append(h2d_s)
            for k in range(len(cam_structs)):
                frame_ms.append(rig.elapsed_ms(ev[1 + k], ev[2 + k])); frame_h2d.append(h2d_f[k])
        return h2d_s + sum(h2d_f)

    vol = vr.Volume(host, cfg.dims, brick=B, layout=vr.VR_BRICKED_HALO1, resident_bytes=resident,
                    n_copy_streams=cfg.n_copy_streams)
    for _ in range(args.warmup):
        step(vol, img, False)
    rig.synchronize()
    clocks = rig.clock_sampler(); clocks.start()
    launches0 = vol.stats()["total_kernel_launches"]
    e0, e1 = rig.event(), rig.event()
    rig.record(e0)
    h2d_step = 0
    for _ in range(args.steps):
        h2d_step = step(vol, img, True)
    rig.record(e1); rig.synchronize()
    clk = clocks.finish()
    ms_step = rig.elapsed_ms(e0, e1) / args.steps
    launches = vol.stats()["total_kernel_launches"] - launches0
    vol.close()

    e2e_steps = max(1, min(args.steps, 2))
    a, b = rig.event(), rig.event()
    rig.record(a)
    e2e_h2d = 0
    for _ in range(e2e_steps):
        with vr.Volume(host, cfg.dims, brick=B, layout=vr.VR_BRICKED_HALO1, resident_bytes=resident,
                       n_copy_streams=cfg.n_copy_streams) as hv:
            e2e_h2d = step(hv, h_img, False)
    rig.record(b); rig.synchronize()
    e2e_ms = rig.elapsed_ms(a, b) / e2e_steps
    ms_step, e2e_ms = max_over_ranks([ms_step, e2e_ms], dist, "cuda")
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return None
    k_ms = float(np.mean(frame_ms))
    gbs = float(np.sum(frame_h2d)) / (float(np.sum(frame_ms)) * 1e-3) / 1e9
    sum_gbs = float(np.sum(sum_h2d)) / (float(np.sum(sum_ms)) * 1e-3) / 1e9
    block = config_block(cfg, f"out of core: {size_note}; cube {cube_bytes / 1e9:.1f} GB pinned host, brick-major "
                              f"{B}^3(+1 halo), resident cap {resident / 1e9:.1f} GB, {cfg.n_copy_streams} copy streams")
    block["cube_bytes"] = cube_bytes
    line = {"metric": "voxel_samples_per_s", "value": world * samples_step / (ms_step * 1e-3), "unit": "samples/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": block, "clocks": clk,
            "e2e": {"value": world * samples_step / (e2e_ms * 1e-3), "unit": "samples/s",
                    "h2d_bytes_per_step": int(e2e_h2d),
                    "d2h_bytes_per_step": int(len(cams) * cfg.height * cfg.width * 16 + 32 + 8 * 256),
                    "ms_per_step": e2e_ms, "steps": e2e_steps},
            "gpu_launches": int(launches),
            "roofline": {"bound": "host_link", "achieved": gbs, "peak": link_peak, "unit": "GB/s", "frac": gbs / link_peak,
                         "traffic": None, "kernel": "vr_render, out-of-core brick chain (cudaMemcpyAsync on the copy streams "
                         "+ k_chain_brick per brick)", "kernel_ms": k_ms, "launches_timed": len(frame_ms),
                         "peak_source": "pinned 1 GiB cudaMemcpyAsync, best of 10, measured in this run",
                         "algorithmic_bytes_per_launch": float(np.mean(frame_h2d))},
            "summary_pass": {"h2d_gbs": sum_gbs, "frac_of_link": sum_gbs / link_peak, "ms": float(np.mean(sum_ms)),
                             "h2d_bytes": int(np.mean(sum_h2d))},
            "frames_per_s": world * len(cams) / (ms_step * 1e-3),
            "render_ms": {"min": float(np.min(frame_ms)), "median": float(np.median(frame_ms)), "mean": k_ms,
                          "max": float(np.max(frame_ms))},
            "h2d_bytes_per_step": int(h2d_step), "samples_per_step": int(samples_step), "cpu_baseline": None}
    if world == 1 and not args.no_cpu:
        import oracle as O
        cam = cfg.camera(0)
        mask = np.zeros((cam.height, cam.width), dtype=np.uint8)
        mask[4::8, 4::8] = 1
        hn = rig.as_numpy(host).reshape(-1, B + 1, B + 1, B + 1)
        t0 = time.perf_counter()
        r = O.render(hn, cam, O.EA, tf, last_range[0], last_range[1], mask=mask, layout=O.BRICKED_HALO1,
                     layout_brick=B, dims=cfg.dims)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": r.n_nominal / dt, "unit": "samples/s", "cores": O.num_threads(), "kind": "oracle",
                                "sample": f"{cfg.name} view 0, every 8th pixel in x and y ({r.n_nominal} nominal samples, "
                                          f"{dt:.2f} s), f32-canonical oracle on the brick-major cube, OpenMP"}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4,
                    help="BASELINE.json config number (default 4: the largest single-GPU config; the metric is 'per cube size')")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg (profiling runs)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--ooc-nz", type=int, default=0, help="cfg5: spectral channels to use (0 = as many brick layers as fit host memory)")
    ap.add_argument("--ooc-resident-frac", type=float, default=0.25, help="cfg5: device brick pool as a fraction of the cube")
    ap.add_argument("--path", type=int, default=0, help="VR_OPT_RENDER_PATH for ablations (0 = auto, the product default)")
    ap.add_argument("--lag", type=int, default=-1, help="VR_OPT_LANE_LAG for ablations (-1 = library default)")
    ap.add_argument("--no-zcopy", action="store_true", help="VR_OPT_ZFAST_COPY = 0 (ablation)")
    ap.add_argument("--row-loads", type=int, default=-1, help="VR_OPT_ROW_LOADS for ablations: 0 scalar, 1 16-byte quads, 2 auto (-1 = library default, auto)")
    ap.add_argument("--views", type=int, default=0, help="render only the first N views of the orbit (profiling runs)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
