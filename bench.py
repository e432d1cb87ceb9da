#!/usr/bin/env python
"""bench.py -- particles/s of the Splotch per-frame rendering path on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--mode additive|ordered] [--impl ours|reference]

A step is one whole frame (count -> scan -> scatter -> splat -> large -> compose) of BASELINE configs[1]
(10M particles, 50 Plummer halos + 20 % background, 800 x 800, additive mode) with the particles
already resident in HBM.  One JSON line is printed by rank 0.  `e2e` is the same frame through
splotch_render_host: pinned HOST particle arrays in, HOST image out, copies inside the timed region.
N > 1 runs N independent replicas (the path does not shard: north_star fixes one GPU, DESIGN.md
"Multi-GPU"), so scaling is weak and no collective is on the data path.
`--impl reference` times the CPU oracle (oracle/, test infrastructure) on the host cores instead.
"""
from __future__ import annotations

import argparse
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

KERNELS_ADDITIVE = 6         # k_count, k_scan, k_scatter, k_splat, k_large, k_compose (+ one memset node)
L2_FLUSH_BYTES = 256 << 20   # written between frames when a config's inputs fit in the 126 MB L2


def tile_for(cfg: int) -> int:
    return 32 if cfg == 3 else 16       # 4096^2 at 16 px would need a 65,536-bin per-block histogram


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
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max_mhz = index, False, [], set(), None
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
        self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
        try:
            r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake", 0x2: "applications_clocks_setting"}
        for bit, name in names.items():
            if r & bit:
                self.reasons.add(name)

    def run(self):
        while not self.stop_flag:
            self.sample()
            time.sleep(0.01)

    def result(self):
        if not self.sm:
            self.sample()
        return {"sm_mhz": statistics.median(self.sm) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.sm)}


def ncu_traffic(kernel: str, workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed ncu --set full capture
    (profiles/dram_traffic.csv: kernel,workload,bytes), or None."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if os.path.exists(path):
        for line in open(path).read().splitlines()[1:]:
            k, wk, b = line.split(",")[:3]
            if k == kernel and wk == workload:
                return float(b)
    return None


def max_over_ranks(ms: float, dist, device) -> float:
    """The slowest rank's time: every multi-GPU number is the max over ranks of a device-side timing."""
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, n: int, ms_step: float) -> float:
    """particles/s of the whole job: N replicas (weak scaling) render world * n particles per step."""
    return world * n / (ms_step * 1e-3)


def visible_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


def fragments_estimate(r, fields, species, kw) -> float:
    """Algorithmic fragments of a frame: 1 per SMALL particle, pixel centres inside the clip disc otherwise
    (pi r^2, at most the on-screen pixel box).  Computed once, outside the timed region."""
    d = r.debug_geometry(fields, species, **kw)
    cls, rp, box = d["cls"], d["rp"].double(), d["pbox"].double()
    area = (box[:, 1] - box[:, 0] + 1) * (box[:, 3] - box[:, 2] + 1)
    disc = torch.minimum(torch.pi * rp * rp, area)
    return float((cls == 1).sum() + disc[cls >= 2].sum()), float(disc[cls == 3].sum())


def run_ours(args):
    from paper_1309_1114_b200 import binding
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    w = wl.make_config(args.config, device=f"cuda:{local}")
    TILE = tile_for(args.config)
    additive = args.mode == "additive"
    lut = wl.palette()
    fields = {k: v.contiguous() for k, v in w.fields.items()}
    r = binding.Renderer(w.width, w.height, w.n, device=local)
    r.set_camera(w.camera)
    for s, sp in enumerate(w.species):
        if sp.use_colormap:
            r.set_colormap(s, lut)
    kw = dict(chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=TILE, additive=additive,
              apply_transfer=False)
    image = torch.empty((w.height, w.width, 3), dtype=torch.float32, device=f"cuda:{local}")
    stream = torch.cuda.current_stream()
    orbit = args.config == 4                 # fly-through: the camera moves 3 degrees per frame
    flush = 24 * w.n < (126 << 20)           # inputs fit in L2: flush it between frames
    fbuf = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=f"cuda:{local}") if flush else None

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def frame(i):
        if orbit:
            r.set_camera(wl.orbit_camera(i % 120))
        r.render(fields, w.species, image=image, **kw)

    # ---- device-resident timing -------------------------------------------------------------------------------
    for i in range(max(args.warmup, 3)):
        frame(i)
    torch.cuda.synchronize()
    st0 = r.stats()
    assert st0["overflow"] == 0, "pair capacity overflow"
    r.set_profiling(True)
    sampler = ClockSampler(visible_index(local))
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(args.steps):
        if flush:
            fbuf.fill_(i & 255)
        ev[i][0].record(stream)
        frame(i)
        ev[i][1].record(stream)
    e1.record(stream)
    barrier()
    sampler.stop_flag = True
    per_frame = sorted(a.elapsed_time(b) for a, b in ev)
    # with an L2 flush between frames the step time is the sum of the frames' own event pairs
    ms_total = sum(per_frame) if flush else e0.elapsed_time(e1)
    st = r.stats()
    r.set_profiling(False)
    sampler.join(timeout=1.0)
    ms_step = max_over_ranks(ms_total, dist, f"cuda:{local}") / args.steps
    dist_ms = {"min": per_frame[0], "median": per_frame[len(per_frame) // 2],
               "p95": per_frame[min(len(per_frame) - 1, int(0.95 * len(per_frame)))], "max": per_frame[-1]}

    # ---- end to end through the C ABI with HOST buffers ---------------------------------------------------------
    host = {k: v.cpu().pin_memory() for k, v in fields.items()}
    himg = torch.empty((w.height, w.width, 3), dtype=torch.float32).pin_memory()
    e2e_steps = max(3, min(args.steps, 20 if w.n <= 20_000_000 else 3))
    if orbit:
        r.set_camera(wl.orbit_camera(0))
    r.render_host(host, w.species, himg, **kw)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        r.render_host(host, w.species, himg, **kw)          # synchronises the stream before returning
    t1 = time.perf_counter()
    e2e_ms = max_over_ranks((t1 - t0) * 1e3 / e2e_steps, dist, f"cuda:{local}")

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    # ---- roofline of the dominant kernel ------------------------------------------------------------------------
    hbm_gbs, sm_max_mhz, peak_src = measured_peaks()
    stage = st["stage_ms"]
    dom = max(stage, key=stage.get)
    pairs = st["pairs"] + st["large_pairs"]
    active = st["n"] - st["count"][0]
    if orbit:
        r.set_camera(wl.orbit_camera((args.steps - 1) % 120))     # the camera of the frame the statistics belong to
    frags, frags_large = fragments_estimate(r, fields, w.species, kw)
    n_tiles = (-(-w.width // TILE)) * (-(-w.height // TILE))
    passes = -(-st["sort_key_bits"] // 8) if not additive else 0      # radix passes that really ran
    # algorithmic bytes per stage and frame
    if additive:
        bytes_by_stage = {
            "count": 16.0 * w.n,                                   # x y z h read once
            "scatter": 24.0 * w.n + 32.0 * pairs,                  # six fields read, one 32-B record written per pair
            "splat": 32.0 * st["pairs"],                           # records read once
            "large": 32.0 * st["large_pairs"],                     # super-tile records read once (64 tiles share them in L2)
            "compose": (24.0 + 12.0) * w.width * w.height,         # fixed-point sums read, image written once
        }
        hbm_stages, alu_stages = ("count", "scatter"), ("splat", "large", "compose")
    else:
        bytes_by_stage = {
            "count": 16.0 * w.n,
            "pairs": 24.0 * w.n + 32.0 * active + 12.0 * pairs,    # fields read, one record per particle, key + value per pair
            "sort": passes * (8.0 + 12.0 + 12.0) * pairs,          # per pass: keys read (histogram), key + value read and written
            "bounds": 8.0 * pairs,
            "render": (4.0 + 32.0) * pairs,                        # value + gathered record per pair
            "combine": 12.0 * w.width * w.height,
        }
        hbm_stages, alu_stages = ("count", "pairs", "sort"), ("render", "combine")
    traffic = ncu_traffic("k_" + dom, w.name)
    flop = FLOP_PER_FRAGMENT if additive else FLOP_PER_FRAGMENT_ORDERED
    peak_tf = 148 * 128 * sm_max_mhz * 1e6 / 1e12              # FP32 lanes x clock, one op per lane per cycle
    bytes_by_stage.setdefault(dom, 0.0)
    t_hbm = bytes_by_stage[dom] / (hbm_gbs * 1e9)
    dom_frags = {"splat": frags - frags_large, "large": frags_large, "render": frags}.get(dom, 0.0) if additive or dom == "render" else 0.0
    t_alu = dom_frags * flop / (peak_tf * 1e12)
    # the roofline that bounds the stage is the larger of its two lower bounds ("report both, take the larger")
    if t_hbm >= t_alu:
        ach = bytes_by_stage[dom] / (stage[dom] * 1e-3) / 1e9
        roof = {"kernel": "k_" + dom, "bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s",
                "frac": ach / hbm_gbs, "traffic": traffic, "peak_source": peak_src + " copy bandwidth",
                "other_bound": {"bound": "alu", "lower_bound_ms": t_alu * 1e3}}
    else:
        ach = dom_frags * flop / (stage[dom] * 1e-3) / 1e12
        roof = {"kernel": "k_" + dom, "bound": "alu", "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": ach / peak_tf, "traffic": traffic,
                "peak_source": "148 SM x 128 FP32 lanes x %.0f MHz, FMA = 1 op (DESIGN.md)" % sm_max_mhz,
                "other_bound": {"bound": "hbm", "lower_bound_ms": t_hbm * 1e3}}
    stage_roof = {}
    for k in stage:
        stage_roof[k] = {"ms": stage[k]}
        if k in hbm_stages:
            gbs = bytes_by_stage[k] / (stage[k] * 1e-3) / 1e9
            stage_roof[k].update({"GB/s": gbs, "frac_hbm": gbs / hbm_gbs})
    rk = "splat" if additive else "render"
    stage_roof[rk]["Gfragments/s"] = frags / (stage[rk] * 1e-3) / 1e9
    # sum of per-stage lower bounds: HBM terms + ALU term
    flop = FLOP_PER_FRAGMENT if additive else FLOP_PER_FRAGMENT_ORDERED
    t_min_ms = sum(bytes_by_stage.values()) / (hbm_gbs * 1e9) * 1e3 + frags * flop / (148 * 128 * sm_max_mhz * 1e6) * 1e3

    # ---- CPU baseline: the oracle as it stands, one thread ---------------------------------------------------------
    cpu = cpu_baseline_frame(w, lut, min(w.n, args.cpu_sample), TILE, additive)

    out = {
        "metric": "particles/s rendered end-to-end per frame",
        "value": whole_job_value(world, w.n, ms_step), "unit": "particles/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "particles": w.n, "image": [w.width, w.height], "mode": args.mode,
                   "tile": TILE, "chi": w.chi, "r_large": w.r_large, "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": ("256 MB written between frames (inputs fit in L2); step time = sum of per-frame event pairs" if flush else
                          "inputs (%.0f MB) and records (%.0f MB) exceed the 126 MB L2, no flush" % (24e-6 * w.n, 32e-6 * pairs)),
                   "camera": "orbit, 3 deg/frame" if orbit else "fixed",
                   "classes": dict(zip(("culled", "small", "medium", "large"), st["count"])), "pairs": pairs,
                   "active": active, "fragments_estimate": frags, "fragments_large": frags_large},
        "clocks": sampler.result(),
        "e2e": {"value": whole_job_value(world, w.n, e2e_ms), "unit": "particles/s", "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": 24 * w.n, "d2h_bytes_per_step": 12 * w.width * w.height, "steps": e2e_steps,
                "api": "splotch_render_host (pinned host arrays in, host image out)"},
        "gpu_launches": (KERNELS_ADDITIVE if additive else ordered_kernels_per_frame(n_tiles)) * args.steps,
        "frame_ms": dist_ms,
        "roofline": roof,
        "stages": stage_roof,
        "frame_lower_bound_ms": t_min_ms, "frac_of_frame_roofline": t_min_ms / ms_step,
        "cpu_baseline": cpu,
    }
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def cpu_baseline_frame(w, lut, sample_n: int, tile: int = 16, additive: bool = True):
    """Time the oracle (single thread, as it stands) on the first sample_n particles of the workload."""
    from oracle import splotch_oracle as so
    f = {k: v[:sample_n].cpu().numpy() for k, v in w.fields.items()}
    import copy
    species = []
    for sp in w.species:
        s2 = copy.copy(sp)
        s2.begin, s2.end = min(sp.begin, sample_n), min(sp.end, sample_n)
        species.append(s2)
    luts = [lut.numpy() if s.use_colormap else None for s in species]
    so.lib()
    t0 = time.perf_counter()
    so.render(f, species, luts, w.camera, w.width, w.height, chi=w.chi, r_small=w.r_small, r_large=w.r_large,
              z_near=w.z_near, tile=tile, additive=additive)
    dt = time.perf_counter() - t0
    return {"value": sample_n / dt, "unit": "particles/s", "cores": 1, "kind": "oracle", "seconds": dt,
            "sample": "first %d of %d particles of %s, one full frame, single thread" % (sample_n, w.n, w.name)}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = wl.make_config(args.config, device="cpu")
    lut = wl.palette()
    # bounded sample: about 0.75 us of oracle time per particle, whole run kept near two minutes
    sample_n = min(w.n, args.ref_sample, max(100_000, int(1.6e8 / (args.steps + args.warmup))))
    times = []
    for _ in range(args.warmup):
        cpu_baseline_frame(w, lut, sample_n, tile_for(args.config), args.mode == "additive")
    for _ in range(args.steps):
        times.append(cpu_baseline_frame(w, lut, sample_n, tile_for(args.config), args.mode == "additive")["seconds"])
    ms = 1e3 * sum(times) / len(times)
    val = sample_n / (ms * 1e-3)
    out = {"impl": "reference", "metric": "particles/s rendered end-to-end per frame", "value": val,
           "unit": "particles/s", "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": w.name, "particles": w.n, "image": [w.width, w.height], "mode": args.mode,
                      "tile": tile_for(args.config), "chi": w.chi, "r_large": w.r_large},
           "cpu_baseline": {"value": val, "unit": "particles/s", "cores": 1, "kind": "oracle",
                            "sample": "each step: one frame of the first %d of %d particles, single thread" % (sample_n, w.n)},
           "e2e": {"value": val, "unit": "particles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--mode", default="additive", choices=["additive", "ordered"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-sample", type=int, default=10_000_000)
    ap.add_argument("--ref-sample", type=int, default=10_000_000)
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 3 if args.steps is None else args.steps
        run_reference(args)
    else:
        args.steps = 100 if args.steps is None else args.steps
        run_ours(args)


if __name__ == "__main__":
    main()
