#!/usr/bin/env python
"""bench.py -- particles/s of the Splotch per-frame rendering path on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--mode additive|ordered]
                  [--impl ours|reference] [--no-per-config] [--frames-only] [--tile T]

A step is one whole frame (count -> scan -> scatter -> splat -> large -> compose) with the particles already
resident in HBM.  BASELINE.json's metric names no config, so the default line is on the largest single-GPU
configuration, configs[3] (400M particles, camera inside the densest halo, 4096 x 4096, additive mode); the same
JSON line carries, under `per_config`, frame time, particles/s, per-stage roofline fractions and the fraction of the
frame roofline for all five configs and for the ordered mode on the 120-frame orbit (cfg4).
`e2e` is the same frame through splotch_render_host: pinned HOST particle arrays in, HOST image out, copies inside
the timed region (chunked, copy / compute overlapped on two streams).
N > 1 runs N independent replicas (the path does not shard: north_star fixes one GPU), so
scaling is weak and no collective is on the data path.
`--impl reference` times the CPU oracle (oracle/, test infrastructure) on the host cores instead.
"""
from __future__ import annotations

import argparse
import gc
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_1309_1114_b200 import workloads as wl  # noqa: E402

KERNELS_ADDITIVE = 7         # k_count, k_scan, k_layout, k_scatter, k_splat, k_large, k_compose (+ memset nodes)
L2_FLUSH_BYTES = 256 << 20   # written between frames when a config's inputs fit in the 126 MB L2
DEFAULT_CONFIG = 3           # the largest single-GPU configuration of BASELINE.json


TILE_OVERRIDE = 0


def tile_for(cfg: int, mode: str = "additive") -> int:
    """Tile side the configuration is timed with (a parameter of the library; its default is 16).  32 px for the frames of 1e8
    particles and more in additive mode: a quarter of the bins makes k_scatter's stores land better (cfg2: 1.98 -> 1.49 ms) for a
    little more k_splat time (2.38 -> 2.59 ms); the ordered mode and the small frames are faster with 16 px."""
    if TILE_OVERRIDE:
        return TILE_OVERRIDE
    return 32 if (cfg == 3 or (cfg in (2, 4) and mode == "additive")) else 16


def ordered_kernels_per_frame(n_tiles: int) -> int:
    tile_bytes = 1
    while tile_bytes < 4 and (n_tiles - 1) >> (8 * tile_bytes):
        tile_bytes += 1
    return 3 + 5 * (4 + tile_bytes) + 3   # count, scan, pairs; 5 launches per radix pass; bounds, render, combine


FLOP_PER_FRAGMENT = 8        # 2 FMA (d^2) + compare + scale + exp2 + 3 FMA, FMA counted once
FLOP_PER_FRAGMENT_ORDERED = 26   # + optical depth, 1 - exp(-x) (7-term series, exp2, selects), 3 x (sub, FMA), transmission product


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs (as fast as NVML answers, so
    that even a region of a few milliseconds holds several samples)."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max_mhz = index, False, [], set(), None
        self.t_begin = self.t_end = None          # the timed region (perf_counter); samples outside it are dropped
        self.stamps, self.flags = [], []
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def sample(self):
        if self.nv is None:
            return
        nv = self.nv
        t = time.perf_counter()
        mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
        try:
            r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        self.stamps.append(0.5 * (t + time.perf_counter()))
        self.sm.append(mhz)
        self.flags.append(r)

    def run(self):
        # started BEFORE the timed region so that the first NVML call (slow) is not inside it; begin() / end() mark it
        while not self.stop_flag:
            self.sample()
            time.sleep(0.0002 if len(self.sm) < 256 else 0.01)

    def begin(self):
        self.t_begin = time.perf_counter()

    def end(self):
        self.t_end = time.perf_counter()
        self.stop_flag = True

    def result(self):
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake", 0x2: "applications_clocks_setting"}
        inside = [i for i, t in enumerate(self.stamps)
                  if self.t_begin is not None and self.t_end is not None and self.t_begin <= t <= self.t_end]
        sm = [self.sm[i] for i in inside]
        reasons = set()
        for i in inside:
            for bit, name in names.items():
                if self.flags[i] & bit:
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(reasons), "samples": len(sm)}


def ncu_traffic(kernel: str, workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed ncu --set full capture
    (profiles/dram_traffic.csv: kernel,workload,bytes), or None."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    best, src = None, None
    if os.path.exists(path):
        for line in open(path).read().splitlines()[1:]:
            parts = line.split(",")
            if len(parts) >= 4 and parts[0] == kernel and parts[1] == workload:
                # the newest capture (last source file) counts; a kernel launched several times per frame (radix passes, some of
                # which return at once) has several rows there: the largest is the full launch
                if parts[3] != src:
                    best, src = None, parts[3]
                best = float(parts[2]) if best is None else max(best, float(parts[2]))
    return best


def max_over_ranks(ms: float, dist, device) -> float:
    """The slowest rank's time: every multi-GPU number is the max over ranks of a device-side timing."""
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, n: int, ms_step: float) -> float:
    """particles/s of the whole job: N replicas (weak scaling) render world * n particles per step."""
    return world * n / (ms_step * 1e-3)


def check_world(gpus: int, world: int) -> None:
    """--gpus N must agree with the launch (torchrun sets WORLD_SIZE); a silent 1-GPU run under --gpus 8 is refused."""
    if gpus != world:
        raise SystemExit(f"bench.py: --gpus {gpus} but WORLD_SIZE is {world}: launch with "
                         f"`python -m torch.distributed.run --nproc-per-node {gpus} bench.py --gpus {gpus} ...`")


def visible_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


ROUTE_RADIUS = 32.0          # csrc kRouteRadius: with 32-px tiles k_large also renders the MEDIUM discs wider than this


def fragments_estimate(r, fields, species, kw, chunk=1 << 26):
    """Algorithmic fragments of a frame: 1 per SMALL particle, pixel centres inside the clip disc otherwise
    (pi r^2, at most the on-screen pixel box); second value: the fragments k_large renders (LARGE discs and, with
    32-px tiles, MEDIUM discs wider than ROUTE_RADIUS).  Computed once, outside the timed region, in chunks."""
    n = fields["x"].numel()
    total = large = 0.0
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        sub = {k: v[a:b] for k, v in fields.items()}
        d = r.debug_geometry(sub, [wl.Species(0, b - a)], **dict(kw, additive=True))
        cls, rp, box = d["cls"], d["rp"].double(), d["pbox"].double()
        area = (box[:, 1] - box[:, 0] + 1) * (box[:, 3] - box[:, 2] + 1)
        disc = torch.minimum(torch.pi * rp * rp, area)
        total += float((cls == 1).sum() + disc[cls >= 2].sum())
        by_large = (cls == 3) | ((cls == 2) & (rp > ROUTE_RADIUS)) if kw.get("tile") == 32 and kw.get("additive", True) else (cls == 3)
        large += float(disc[by_large].sum())
        del d, cls, rp, box, area, disc
    return total, large


def stage_bytes(additive: bool, w, st, passes: int):
    """Algorithmic HBM bytes per stage and frame."""
    pairs = st["pairs"] + st["large_pairs"]
    active = st["n"] - st["count"][0]
    if additive:
        rec_bytes = 32.0 * pairs - 16.0 * st["count"][1]          # a SMALL particle has one pair, a 16-byte record; the others 32 bytes
        tile_rec_bytes = 32.0 * st["pairs"] - 16.0 * st["count"][1]
        return {
            "count": 16.0 * w.n,                                   # x y z h read once
            "scatter": 24.0 * w.n + rec_bytes,                     # six fields read, one record written per pair
            "splat": tile_rec_bytes,                               # records read once
            "large": rec_bytes - tile_rec_bytes,                   # super-tile records read once (the blocks of a super-tile share them in L2)
            "compose": (24.0 + 12.0) * w.width * w.height,         # fixed-point sums read, image written once
        }, ("count", "scatter"), ("splat", "large", "compose")
    return {
        "count": 16.0 * w.n,
        "pairs": 24.0 * w.n + 32.0 * active + 12.0 * pairs,        # fields read, one record per particle, key + value per pair
        "sort": passes * (8.0 + 12.0 + 12.0) * pairs,              # per pass: keys read (histogram), key + value read and written
        "bounds": 8.0 * pairs,
        "render": (4.0 + 32.0) * pairs,                            # value + gathered record per pair
        "combine": 12.0 * w.width * w.height,
    }, ("count", "pairs", "sort"), ("render", "combine")


class Run:
    """One configuration resident on the device: renderer, fields, parameters."""

    def __init__(self, cfg: int, mode: str, local: int, fields=None, workload=None):
        from paper_1309_1114_b200 import binding
        self.cfg, self.mode, self.local = cfg, mode, local
        self.additive = mode == "additive"
        self.w = workload if workload is not None else wl.make_config(cfg, device=f"cuda:{local}")
        w = self.w
        self.tile = tile_for(cfg, mode)
        self.lut = wl.palette()
        self.fields = fields if fields is not None else {k: v.contiguous() for k, v in w.fields.items()}
        w.fields = self.fields
        self.r = binding.Renderer(w.width, w.height, w.n, device=local)
        self.r.set_camera(w.camera)
        for s, sp in enumerate(w.species):
            if sp.use_colormap:
                self.r.set_colormap(s, self.lut)
        self.kw = dict(chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=self.tile,
                       additive=self.additive, apply_transfer=False)
        self.image = torch.empty((w.height, w.width, 3), dtype=torch.float32, device=f"cuda:{local}")
        self.orbit = cfg == 4                    # fly-through: the camera moves 3 degrees per frame
        self.flush = 24 * w.n < (126 << 20)      # inputs fit in L2: flush it between frames
        self.fbuf = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=f"cuda:{local}") if self.flush else None

    def frame(self, i: int):
        if self.orbit:
            self.r.set_camera(wl.orbit_camera(i % 120))
        self.r.render(self.fields, self.w.species, image=self.image, **self.kw)

    def timed(self, steps: int, warmup: int, barrier, sampler=None):
        """(ms per step on this rank, sorted per-frame times, stats with per-stage means)."""
        stream = torch.cuda.current_stream()
        for i in range(max(warmup, 3)):
            self.frame(i)
        torch.cuda.synchronize()
        assert self.r.stats()["overflow"] == 0, "pair capacity overflow"
        self.r.set_profiling(True)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        if sampler is not None:
            sampler.start()
            time.sleep(0.05)
        barrier()
        if sampler is not None:
            sampler.begin()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(steps):
            if self.flush:
                self.fbuf.fill_(i & 255)
            ev[i][0].record(stream)
            self.frame(i)
            ev[i][1].record(stream)
        e1.record(stream)
        barrier()
        if sampler is not None:
            sampler.end()
        per_frame = sorted(a.elapsed_time(b) for a, b in ev)
        # with an L2 flush between frames the step time is the sum of the frames' own event pairs
        ms_total = sum(per_frame) if self.flush else e0.elapsed_time(e1)
        st = self.r.stats()
        self.r.set_profiling(False)
        return ms_total / steps, per_frame, st

    def timed_graph(self, steps: int):
        """ms per frame when the frame is captured once into a CUDA graph and replayed (the library only enqueues kernels and memsets
        on the caller's stream, so a frame can be captured): what a launch-bound frame costs without the launch gaps."""
        self.r.set_profiling(False)
        side = torch.cuda.Stream()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            self.frame(0)
            torch.cuda.synchronize()
            with torch.cuda.graph(graph, stream=side):
                self.frame(0)
        torch.cuda.synchronize()
        stream = torch.cuda.current_stream()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for i in range(3):
            graph.replay()
        for i in range(steps):
            if self.flush:
                self.fbuf.fill_(i & 255)
            ev[i][0].record(stream)
            graph.replay()
            ev[i][1].record(stream)
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in ev) / steps

    def summary(self, ms_step: float, per_frame, st, hbm_gbs: float, fma_peak: float, frags=None):
        """Per-stage roofline fractions and the frame lower bound (sum over stages)."""
        w = self.w
        if self.orbit:
            self.r.set_camera(wl.orbit_camera((len(per_frame) - 1) % 120))   # the camera of the frame the statistics belong to
        if frags is None:
            frags = fragments_estimate(self.r, self.fields, w.species, self.kw)
        passes = -(-st["sort_key_bits"] // 8) if not self.additive else 0      # radix passes that really ran
        bytes_by_stage, hbm_stages, alu_stages = stage_bytes(self.additive, w, st, passes)
        stage = st["stage_ms"]
        flop = FLOP_PER_FRAGMENT if self.additive else FLOP_PER_FRAGMENT_ORDERED
        stage_roof = {}
        for k in stage:
            stage_roof[k] = {"ms": stage[k]}
            if k in hbm_stages and stage[k] > 0:
                gbs = bytes_by_stage[k] / (stage[k] * 1e-3) / 1e9
                stage_roof[k].update({"GB/s": gbs, "frac_hbm": gbs / hbm_gbs})
        frag_stage = {"splat": frags[0] - frags[1], "large": frags[1]} if self.additive else {"render": frags[0]}
        for k, f in frag_stage.items():
            if k in stage and stage[k] > 0 and f > 0:
                stage_roof[k]["Gfragments/s"] = f / (stage[k] * 1e-3) / 1e9
                stage_roof[k]["frac_fma"] = f * flop / (stage[k] * 1e-3) / fma_peak
        t_min_ms = sum(bytes_by_stage.values()) / (hbm_gbs * 1e9) * 1e3 + frags[0] * flop / fma_peak * 1e3
        dist_ms = {"min": per_frame[0], "median": per_frame[len(per_frame) // 2],
                   "p95": per_frame[min(len(per_frame) - 1, int(0.95 * len(per_frame)))], "max": per_frame[-1]}
        return {"workload": w.name, "mode": self.mode, "tile": self.tile, "ms_per_frame": ms_step,
                "particles_per_s": w.n / (ms_step * 1e-3), "frame_ms": dist_ms, "stages": stage_roof,
                "frame_lower_bound_ms": t_min_ms, "frac_of_frame_roofline": t_min_ms / ms_step,
                "classes": dict(zip(("culled", "small", "medium", "large"), st["count"])),
                "pairs": st["pairs"] + st["large_pairs"], "fragments_estimate": frags[0], "fragments_large": frags[1],
                "l2": "256 MB written between frames" if self.flush else "inputs exceed L2, no flush"}, bytes_by_stage, frags

    def close(self):
        self.r.close()
        self.fields = self.image = self.fbuf = None
        self.w.fields = None


def run_ours(args):
    from paper_1309_1114_b200 import binding
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    check_world(args.gpus, world)
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    run = Run(args.config, args.mode, local)
    w, additive = run.w, run.additive
    # ---- device-resident timing -------------------------------------------------------------------------------
    sampler = ClockSampler(visible_index(local))
    ms_local, per_frame, st = run.timed(args.steps, args.warmup, barrier, sampler)
    sampler.join(timeout=1.0)
    ms_step = max_over_ranks(ms_local, dist, f"cuda:{local}")

    if args.frames_only:          # profiling runs (ncu): the timed frames only, no end-to-end leg, no CPU baseline
        if rank == 0:
            print(json.dumps({"frames_only": True, "workload": w.name, "mode": args.mode, "tile": run.tile, "ms_per_step": ms_step,
                              "stages": st["stage_ms"]}))
        if dist is not None:
            dist.destroy_process_group()
        return
    # ---- end to end through the C ABI with HOST buffers ---------------------------------------------------------
    host = {k: v.cpu().pin_memory() for k, v in run.fields.items()}
    himg = torch.empty((w.height, w.width, 3), dtype=torch.float32).pin_memory()
    e2e_steps = max(3, min(args.steps, 20 if w.n <= 20_000_000 else 3))
    if run.orbit:
        run.r.set_camera(wl.orbit_camera(0))
    run.r.render_host(host, w.species, himg, **run.kw)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        run.r.render_host(host, w.species, himg, **run.kw)          # synchronises the stream before returning
    t1 = time.perf_counter()
    e2e_ms = max_over_ranks((t1 - t0) * 1e3 / e2e_steps, dist, f"cuda:{local}")
    del host, himg

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    # ---- peaks: measured HBM copy rate (driver) and FP32 FMA / MUFU.EX2 rates measured here by the library ----------
    hbm_gbs, sm_max_mhz, peak_src = measured_peaks()
    pk = run.r.measure_peaks()
    fma_peak = pk["fma_lane_ops_per_s"]
    # ---- roofline of the dominant kernel ------------------------------------------------------------------------
    summ, bytes_by_stage, frags = run.summary(ms_step, per_frame, st, hbm_gbs, fma_peak)
    stage = st["stage_ms"]
    dom = max(stage, key=stage.get)
    flop = FLOP_PER_FRAGMENT if additive else FLOP_PER_FRAGMENT_ORDERED
    n_tiles = (-(-w.width // run.tile)) * (-(-w.height // run.tile))
    # kernel of the dominant stage, and its DRAM traffic per launch from the committed ncu capture (profiles/dram_traffic.csv)
    ordered_kernel = {"count": "k_ocount", "pairs": "k_opairs", "sort": "k_rs_scatter", "bounds": "k_obounds", "render": "k_orender", "combine": "k_ocombine"}
    dom_kernel = "k_" + dom if additive else ordered_kernel.get(dom, "k_" + dom)
    traffic = ncu_traffic(dom_kernel, w.name if additive else w.name + "_ordered")
    bytes_by_stage.setdefault(dom, 0.0)
    t_hbm = bytes_by_stage[dom] / (hbm_gbs * 1e9)
    dom_frags = ({"splat": frags[0] - frags[1], "large": frags[1]} if additive else {"render": frags[0]}).get(dom, 0.0)
    t_alu = dom_frags * flop / fma_peak
    # the roofline that bounds the stage is the larger of its two lower bounds ("report both, take the larger")
    if t_hbm >= t_alu:
        ach = bytes_by_stage[dom] / (stage[dom] * 1e-3) / 1e9
        roof = {"kernel": dom_kernel, "bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s",
                "frac": ach / hbm_gbs, "traffic": traffic, "peak_source": peak_src + " copy bandwidth (MEASURED_PEAKS.json)",
                "other_bound": {"bound": "alu", "lower_bound_ms": t_alu * 1e3}}
    else:
        ach = dom_frags * flop / (stage[dom] * 1e-3) / 1e12
        roof = {"kernel": dom_kernel, "bound": "alu", "achieved": ach, "peak": fma_peak / 1e12, "unit": "TFLOP/s",
                "frac": ach * 1e12 / fma_peak, "traffic": traffic,
                "peak_source": "FP32 FMA lane-ops/s measured by splotch_measure_peaks on this GPU (FMA = 1 op; nominal "
                               "148 SM x 128 lanes x %.0f MHz = %.1f T)" % (sm_max_mhz, 148 * 128 * sm_max_mhz * 1e-6),
                "algorithmic": "%d lane-ops x %.4g fragments per launch (DESIGN.md section 7)" % (flop, dom_frags),
                "other_bound": {"bound": "hbm", "lower_bound_ms": t_hbm * 1e3}}

    # ---- CPU baseline: the oracle as it stands, one thread, and the same code through the all-cores row-band driver ----
    cpu1 = cpu_baseline_frame(args.config, args.cpu_sample, run.tile, additive, threads=1)
    cpu_all = cpu_baseline_frame(args.config, args.cpu_sample, run.tile, additive, threads=0)

    out = {
        "metric": "particles/s rendered end-to-end per frame",
        "value": whole_job_value(world, w.n, ms_step), "unit": "particles/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "particles": w.n, "image": [w.width, w.height], "mode": args.mode,
                   "tile": run.tile, "chi": w.chi, "r_large": w.r_large, "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": ("256 MB written between frames (inputs fit in L2); step time = sum of per-frame event pairs" if run.flush else
                          "inputs (%.0f MB) and records (%.0f MB) exceed the 126 MB L2, no flush" % (24e-6 * w.n, 32e-6 * summ["pairs"])),
                   "camera": "orbit, 3 deg/frame" if run.orbit else "fixed",
                   "classes": summ["classes"], "pairs": summ["pairs"],
                   "active": st["n"] - st["count"][0], "fragments_estimate": frags[0], "fragments_large": frags[1]},
        "clocks": sampler.result(),
        "e2e": {"value": whole_job_value(world, w.n, e2e_ms), "unit": "particles/s", "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": 24 * w.n, "d2h_bytes_per_step": 12 * w.width * w.height, "steps": e2e_steps,
                "api": "splotch_render_host (pinned host arrays in, host image out; chunked, copies overlap the kernels)"},
        "gpu_launches": (KERNELS_ADDITIVE if additive else ordered_kernels_per_frame(n_tiles)) * args.steps,
        "frame_ms": summ["frame_ms"],
        "roofline": roof,
        "stages": summ["stages"],
        "frame_lower_bound_ms": summ["frame_lower_bound_ms"], "frac_of_frame_roofline": summ["frac_of_frame_roofline"],
        "peaks": {"hbm_GBps": hbm_gbs, "hbm_source": peak_src, "fma_lane_Tops": fma_peak / 1e12,
                  "mufu_ex2_Tops": pk["mufu_ex2_per_s"] / 1e12, "source": "splotch_measure_peaks (this run, this GPU)"},
        "cpu_baseline": cpu1,
        "cpu_baseline_all_cores": cpu_all,
        "host_cores": cpu_all["host_cores"],
    }
    # ---- all five configs and the ordered orbit, same run -----------------------------------------------------------
    if world == 1 and not args.no_per_config:
        per = {f"cfg{args.config}_{args.mode}": summ}
        run.close()
        del run
        gc.collect()
        torch.cuda.empty_cache()
        shared = None
        for cfg, mode, steps in ((0, "additive", 20), (1, "additive", 20), (2, "additive", 10), (3, "additive", 5),
                                 (4, "additive", 120), (4, "ordered", 120)):
            key = f"cfg{cfg}_{mode}"
            if key in per:
                continue
            if cfg == 4 and shared is not None:
                r2 = Run(cfg, mode, local, fields=shared[0], workload=shared[1])
                r2.w.camera = wl.orbit_camera(0)
            else:
                r2 = Run(cfg, mode, local)
            ms2, pf2, st2 = r2.timed(steps, 3, barrier)
            per[key] = r2.summary(ms2, pf2, st2, hbm_gbs, fma_peak)[0]
            if r2.flush and not r2.orbit:           # small frames are launch bound: the same frame replayed from a CUDA graph
                per[key]["ms_per_frame_cuda_graph"] = r2.timed_graph(steps)
            keep = cfg == 4 and mode == "additive"
            if keep:
                shared = (r2.fields, r2.w)
                r2.r.close()
            else:
                if cfg == 4:
                    shared = None
                r2.close()
            del r2
            gc.collect()
            torch.cuda.empty_cache()
        # the memory-coherent variant of the recipe: cfg1's particles contiguous by halo
        r3 = Run(1, "additive", local)
        perm = wl.halo_order(1, r3.w.n, f"cuda:{local}")
        r3.fields = {k: v[perm].contiguous() for k, v in r3.fields.items()}
        r3.w.fields = r3.fields
        ms3, pf3, st3 = r3.timed(20, 3, barrier)
        per["cfg1_additive_by_halo"] = r3.summary(ms3, pf3, st3, hbm_gbs, fma_peak)[0]
        per["cfg1_additive_by_halo"]["workload"] += " (particles contiguous by halo)"
        r3.close()
        del r3, perm
        out["per_config"] = per
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def cpu_baseline_frame(cfg: int, sample_n: int, tile: int = 16, additive: bool = True, threads: int = 1):
    """Time the oracle on a bounded sample of the workload: the first sample_n particles of the full-size recipe
    (same densities, smoothing lengths and camera; the generator is counter based), one full frame.
    threads = 1: the single-threaded definition; threads = 0: the row-band driver on all host cores."""
    from oracle import splotch_oracle as so
    w = wl.make_config(cfg, device="cpu", count=sample_n)
    lut = wl.palette()
    f = {k: v.numpy() for k, v in w.fields.items()}
    luts = [lut.numpy() if s.use_colormap else None for s in w.species]
    so.lib()
    nthreads = so.host_cores() if threads <= 0 else threads
    t0 = time.perf_counter()
    so.render(f, w.species, luts, w.camera, w.width, w.height, chi=w.chi, r_small=w.r_small, r_large=w.r_large,
              z_near=w.z_near, tile=tile, additive=additive, threads=nthreads)
    dt = time.perf_counter() - t0
    full_n = w.meta.get("full_n", w.n)
    return {"value": w.n / dt, "unit": "particles/s", "cores": nthreads, "host_cores": so.host_cores(), "kind": "oracle",
            "seconds": dt,
            "sample": "first %d of %d particles of %s, one full frame, %s" %
                      (w.n, full_n, w.name, "single thread" if nthreads == 1 else "row-band driver, %d threads" % nthreads)}


def default_cpu_sample(cfg: int) -> int:
    """About 10-30 s of single-thread oracle time (cfg3 costs ~35 us per particle: ~2400 fragments each)."""
    return {0: 100_000, 1: 10_000_000, 2: 10_000_000, 3: 500_000, 4: 10_000_000}[cfg]


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    tile, additive = tile_for(args.config, args.mode), args.mode == "additive"
    # bounded sample: the whole --steps / --warmup run stays near two minutes
    sample_n = max(20_000, min(args.ref_sample, int(6 * default_cpu_sample(args.config) / (args.steps + args.warmup))))
    times = []
    base = None
    for i in range(args.warmup + args.steps):
        base = cpu_baseline_frame(args.config, sample_n, tile, additive, threads=1)
        if i >= args.warmup:
            times.append(base["seconds"])
    w = wl.make_config(args.config, device="cpu", count=1)
    ms = 1e3 * sum(times) / len(times)
    val = sample_n / (ms * 1e-3)
    out = {"impl": "reference", "metric": "particles/s rendered end-to-end per frame", "value": val,
           "unit": "particles/s", "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": w.name, "particles": w.meta.get("full_n", w.n), "image": [w.width, w.height], "mode": args.mode,
                      "tile": tile, "chi": w.chi, "r_large": w.r_large},
           "cpu_baseline": {"value": val, "unit": "particles/s", "cores": 1, "host_cores": base["host_cores"], "kind": "oracle",
                            "sample": "each step: " + base["sample"]},
           "e2e": {"value": val, "unit": "particles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG)
    ap.add_argument("--mode", default="additive", choices=["additive", "ordered"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-sample", type=int, default=None)
    ap.add_argument("--ref-sample", type=int, default=10_000_000)
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config sweep over the other configs")
    ap.add_argument("--frames-only", action="store_true", help="time the frames and stop (for runs under ncu)")
    ap.add_argument("--tile", type=int, default=0, help="tile side in px (default: tile_for(config, mode))")
    args = ap.parse_args()
    if args.cpu_sample is None:
        args.cpu_sample = default_cpu_sample(args.config)
    global TILE_OVERRIDE
    TILE_OVERRIDE = args.tile
    if args.impl == "reference":
        args.steps = 3 if args.steps is None else args.steps
        run_reference(args)
    else:
        args.steps = 20 if args.steps is None else args.steps
        run_ours(args)


if __name__ == "__main__":
    main()
