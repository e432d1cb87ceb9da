"""Seeded synthetic particle sets, cameras and palettes for the five BASELINE.json configs.

This module is the ONLY code shared by the oracle side (tests, bench cpu_baseline) and the CUDA
side.  It holds none of the rendering method's arithmetic: it only draws particle fields
(x, y, z, h, I, scalar as float32 SoA), names camera poses and builds an analytic palette.
The recipe is stated in DESIGN.md ("Input recipe") and stands in for the paper's Gadget
snapshot (§5 — 200M dark matter + 200M gas + 10M stars), which is not available.

Random numbers come from a stateless counter-based generator: uniform(seed, particle index,
draw number).  It uses only 32-bit integer arithmetic carried in int64 tensors, so the same
code gives the same bits with torch on the CPU and on a CUDA device (large configs are drawn
directly in HBM).  Transcendental steps (pow, log, cos) run in float64 and may differ in the
last ulp between devices; whichever device drew the particles, both sides consume the SAME
float32 arrays, so this never enters a parity comparison.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import torch

_M32 = 0xFFFFFFFF


# ----------------------------------------------------------------------------------------------
# counter-based uniform generator
# ----------------------------------------------------------------------------------------------
def _mul32(x: torch.Tensor, c: int) -> torch.Tensor:
    """(x * c) mod 2^32 for x holding a uint32 in an int64 tensor; no int64 overflow."""
    lo = x & 0xFFFF
    hi = x >> 16
    return (lo * c + (((hi * c) & 0xFFFF) << 16)) & _M32


def _mix32(x: torch.Tensor) -> torch.Tensor:
    x = x ^ (x >> 16)
    x = _mul32(x, 0x85EBCA6B)
    x = x ^ (x >> 13)
    x = _mul32(x, 0xC2B2AE35)
    x = x ^ (x >> 16)
    return x


def _mix32_scalar(x: int) -> int:
    x &= _M32
    x ^= x >> 16
    x = (x * 0x85EBCA6B) & _M32
    x ^= x >> 13
    x = (x * 0xC2B2AE35) & _M32
    x ^= x >> 16
    return x


def uniform(seed: int, idx: torch.Tensor, draw: int) -> torch.Tensor:
    """float64 uniform in (0, 1), a pure function of (seed, idx, draw). idx: int64 tensor < 2^32."""
    k1 = _mix32_scalar(seed * 0x9E3779B1 + draw * 0x7F4A7C15 + 0x165667B1)
    k2 = _mix32_scalar(k1 + 0x27D4EB2F)
    a = _mix32(idx ^ k1)
    b = _mix32(((a + 0x9E3779B9) & _M32) ^ k2)
    hi = (a >> 5).to(torch.float64)          # 27 bits
    lo = (b >> 6).to(torch.float64)          # 26 bits
    return (hi * 67108864.0 + lo + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed: int, idx: torch.Tensor, draw: int) -> torch.Tensor:
    """Standard normal by Box-Muller from draws (draw, draw+1)."""
    u1 = uniform(seed, idx, draw)
    u2 = uniform(seed, idx, draw + 1)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)


# ----------------------------------------------------------------------------------------------
# data classes
# ----------------------------------------------------------------------------------------------
@dataclass
class Camera:
    eye: Tuple[float, float, float]
    lookat: Tuple[float, float, float]
    up: Tuple[float, float, float]
    fov_deg: float                      # horizontal, full angle


@dataclass
class Species:
    begin: int
    end: int
    brightness: float = 1.0
    absorb: float = 1.0                 # kappa_s, ordered mode only
    use_colormap: bool = True
    fixed_rgb: Tuple[float, float, float] = (1.0, 1.0, 1.0)
    scalar_min: float = 0.0
    scalar_max: float = 1.0
    scalar_log10: bool = False
    auto_range: bool = False            # normalisation range found from the data instead of scalar_min / scalar_max
    vector_colour: bool = False         # colour from the vector fields cr, cg, cb


@dataclass
class Workload:
    name: str
    n: int
    width: int
    height: int
    fields: Dict[str, torch.Tensor]     # x y z h I scalar, float32, length n
    species: List[Species]
    camera: Camera
    chi: float = 3.0
    r_small: float = 0.5
    r_large: float = 64.0
    z_near: float = 1e-6
    additive: bool = True
    apply_transfer: bool = False
    meta: Dict[str, object] = field(default_factory=dict)


FIELD_NAMES = ("x", "y", "z", "h", "I", "scalar")


def palette(n_entries: int = 256) -> torch.Tensor:
    """Analytic colour ramp (black-red-yellow-white with a 0.05 floor), float32 [n_entries, 3]."""
    t = torch.arange(n_entries, dtype=torch.float64) / (n_entries - 1)
    r = torch.clamp(3.0 * t, 0.0, 1.0)
    g = torch.clamp(3.0 * t - 1.0, 0.0, 1.0)
    b = torch.clamp(3.0 * t - 2.0, 0.0, 1.0)
    rgb = 0.05 + 0.95 * torch.stack([r, g, b], dim=1)
    return rgb.to(torch.float32).contiguous()


# ----------------------------------------------------------------------------------------------
# generators
# ----------------------------------------------------------------------------------------------
_PLUMMER_TRUNC = 1000.0 / 101.0 ** 1.5      # mass fraction inside r = 10 a


def _plummer_offset(seed: int, idx: torch.Tensor, draw0: int, a) -> Tuple[torch.Tensor, ...]:
    """Offset from the halo centre: Plummer radius truncated at 10 a, isotropic direction."""
    u = uniform(seed, idx, draw0) * _PLUMMER_TRUNC
    r = a / torch.sqrt(torch.pow(u, -2.0 / 3.0) - 1.0)
    ct = 1.0 - 2.0 * uniform(seed, idx, draw0 + 1)
    st = torch.sqrt(torch.clamp(1.0 - ct * ct, min=0.0))
    ph = 2.0 * math.pi * uniform(seed, idx, draw0 + 2)
    return r * st * torch.cos(ph), r * st * torch.sin(ph), r * ct, r


def _chunks(n: int, step: int):
    for s in range(0, n, step):
        yield s, min(n, s + step)


def halo_table(seed: int, n_halos: int = 50):
    """Masses (dN/dM ~ M^-1.9 on [1, 1000]), scales a_k and centres of the halo set (float64, CPU)."""
    k = torch.arange(n_halos, dtype=torch.int64)
    hs = seed ^ 0x5EED
    u = uniform(hs, k, 0)
    mass = torch.pow(1.0 - u * (1.0 - 1000.0 ** -0.9), -1.0 / 0.9)
    scale = torch.clamp(0.005 * torch.pow(mass, 1.0 / 3.0), 0.005, 0.05)
    centre = torch.stack([0.1 + 0.8 * uniform(hs, k, 1 + d) for d in range(3)], dim=1)
    return mass, scale, centre


def _single_plummer(seed: int, n: int, device, count: Optional[int] = None) -> Dict[str, torch.Tensor]:
    count = n if count is None else min(count, n)
    out = {f: torch.empty(count, dtype=torch.float32, device=device) for f in FIELD_NAMES}
    for s, e in _chunks(count, 1 << 22):
        idx = torch.arange(s, e, dtype=torch.int64, device=device)
        dx, dy, dz, _ = _plummer_offset(seed, idx, 0, 0.1)
        out["x"][s:e] = (0.5 + dx).to(torch.float32)
        out["y"][s:e] = (0.5 + dy).to(torch.float32)
        out["z"][s:e] = (0.5 + dz).to(torch.float32)
        out["h"][s:e] = torch.exp(math.log(0.005) + 0.5 * normal(seed, idx, 3)).to(torch.float32)
        out["scalar"][s:e] = torch.exp(normal(seed, idx, 5)).to(torch.float32)
        out["I"][s:e] = (0.5 + uniform(seed, idx, 7)).to(torch.float32)
    return out


def _halo_set(seed: int, n: int, eta: float, device, star_begin: Optional[int] = None, count: Optional[int] = None):
    """50 Plummer halos + 20 % uniform background; h from the analytic local number density.

    `count` draws only particles [0, count) of the n-particle set (the generator is counter based, so these are the
    same particles the full set starts with; densities and smoothing lengths are those of the full set).  The
    scalar range is then the analytic one of the full set: [log10(0.2 n), log10 of the densest halo centre]."""
    mass, scale, centre = halo_table(seed)
    msum = float(mass.sum())
    cum = (torch.cumsum(mass, 0) / msum).to(device)
    cum[-1] = 1.0
    mass_d, scale_d, centre_d = mass.to(device), scale.to(device), centre.to(device)
    n_bg = 0.2 * n
    partial = count is not None and count < n
    count = n if count is None else min(count, n)
    out = {f: torch.empty(count, dtype=torch.float32, device=device) for f in FIELD_NAMES}
    dmin, dmax = math.inf, -math.inf
    for s, e in _chunks(count, 1 << 22):
        idx = torch.arange(s, e, dtype=torch.int64, device=device)
        is_bg = uniform(seed, idx, 0) < 0.2
        hk = torch.clamp(torch.searchsorted(cum, uniform(seed, idx, 1)), max=mass.numel() - 1)
        a = scale_d[hk]
        dx, dy, dz, r = _plummer_offset(seed, idx, 2, a)
        px = torch.where(is_bg, uniform(seed, idx, 5), centre_d[hk, 0] + dx)
        py = torch.where(is_bg, uniform(seed, idx, 6), centre_d[hk, 1] + dy)
        pz = torch.where(is_bg, uniform(seed, idx, 7), centre_d[hk, 2] + dz)
        n_k = 0.8 * n * mass_d[hk] / msum
        dens_halo = 3.0 * n_k / (4.0 * math.pi * a ** 3) * torch.pow(1.0 + (r / a) ** 2, -2.5)
        dens = n_bg + torch.where(is_bg, torch.zeros_like(dens_halo), dens_halo)
        h = torch.clamp(eta * torch.pow(dens, -1.0 / 3.0), 1e-4, 0.05)
        sc = torch.log10(dens)
        out["x"][s:e] = px.to(torch.float32)
        out["y"][s:e] = py.to(torch.float32)
        out["z"][s:e] = pz.to(torch.float32)
        out["h"][s:e] = h.to(torch.float32)
        out["scalar"][s:e] = sc.to(torch.float32)
        inten = torch.ones_like(h)
        if star_begin is not None:
            stars = idx >= star_begin
            inten = torch.where(stars, torch.exp(normal(seed, idx, 8)), inten)
        out["I"][s:e] = inten.to(torch.float32)
        dmin = min(dmin, float(sc.min()))
        dmax = max(dmax, float(sc.max()))
    if partial:      # the prefix does not see the extremes of the full set: use the analytic bounds of the recipe
        dmin = math.log10(n_bg)
        dmax = math.log10(n_bg + float((3.0 * (0.8 * n * mass / msum) / (4.0 * math.pi * scale ** 3)).max()))
    info = {"scalar_min": dmin, "scalar_max": dmax, "halo_mass": mass, "halo_scale": scale,
            "halo_centre": centre}
    return out, info


def halo_order(cfg: int, n: int, device) -> torch.Tensor:
    """Permutation that makes the halo set of configs[cfg] contiguous by halo (background particles last): the memory-coherent
    variant of the recipe (the default interleaves the halos' particles, the hard case for the binning stages)."""
    seed = 1002 if cfg == 4 else 1000 + cfg
    mass, _, _ = halo_table(seed)
    cum = (torch.cumsum(mass, 0) / float(mass.sum())).to(device)
    cum[-1] = 1.0
    key = torch.empty(n, dtype=torch.int16, device=device)
    for s, e in _chunks(n, 1 << 22):
        idx = torch.arange(s, e, dtype=torch.int64, device=device)
        hk = torch.clamp(torch.searchsorted(cum, uniform(seed, idx, 1)), max=mass.numel() - 1)
        key[s:e] = torch.where(uniform(seed, idx, 0) < 0.2, torch.full_like(hk, mass.numel()), hk).to(torch.int16)
    return torch.sort(key, stable=True).indices


def orbit_camera(frame: int, fov_deg: float = 45.0) -> Camera:
    """cfg4 fly-through: eye on a radius-2 circle around the box centre, 3 degrees per frame."""
    ang = math.radians(3.0 * frame)
    return Camera((0.5 + 2.0 * math.sin(ang), 0.5, 0.5 + 2.0 * math.cos(ang)), (0.5, 0.5, 0.5),
                  (0.0, 1.0, 0.0), fov_deg)


def make_config(cfg: int, n: Optional[int] = None, device="cpu", size: Optional[Tuple[int, int]] = None,
                eta: Optional[float] = None, count: Optional[int] = None) -> Workload:
    """Workload for BASELINE.json configs[cfg] (0-based). `n` / `size` shrink it for oracle-sized tests.
    `count` keeps the n-particle recipe (densities, smoothing lengths, camera) but draws only its first `count`
    particles: a bounded sample of the same workload for the timed CPU baseline."""
    w = _make_config(cfg, n, device, size, eta, count)
    if count is not None and count < w.n:
        w.meta["full_n"] = w.n
        w.n = count
        for sp in w.species:
            sp.begin, sp.end = min(sp.begin, count), min(sp.end, count)
    return w


def _make_config(cfg, n, device, size, eta, count) -> Workload:
    seed = 1000 + cfg
    centre = (0.5, 0.5, 0.5)
    front = Camera((0.5, 0.5, 2.5), centre, (0.0, 1.0, 0.0), 45.0)
    if cfg == 0:
        n = 100_000 if n is None else n
        w, h = size or (256, 256)
        f = _single_plummer(seed, n, device, count)
        sp = [Species(0, n, brightness=1.0, scalar_min=-2.0, scalar_max=2.0, scalar_log10=True)]
        return Workload("cfg0_plummer_100k", n, w, h, f, sp, front)
    if cfg == 1:
        n = 10_000_000 if n is None else n
        w, h = size or (800, 800)
        f, info = _halo_set(seed, n, 0.25 if eta is None else eta, device, count=count)
        sp = [Species(0, n, brightness=1.0, scalar_min=info["scalar_min"], scalar_max=info["scalar_max"])]
        return Workload("cfg1_halos_10M", n, w, h, f, sp, front, meta=info)
    if cfg in (2, 4):
        n = 100_000_000 if n is None else n
        w, h = size or (1920, 1080)
        n_gas = (6 * n) // 10
        f, info = _halo_set(seed if cfg == 2 else 1002, n, 0.25 if eta is None else eta, device,
                            star_begin=n_gas, count=count)
        sp = [Species(0, n_gas, brightness=1.0, absorb=0.5, scalar_min=info["scalar_min"],
                      scalar_max=info["scalar_max"]),
              Species(n_gas, n, brightness=0.3, absorb=2.0, use_colormap=False,
                      fixed_rgb=(1.0, 0.9, 0.6))]
        if cfg == 2:
            d = (1.0, 0.5, 0.8)
            nrm = math.sqrt(sum(c * c for c in d))
            cam = Camera(tuple(0.5 + 2.0 * c / nrm for c in d), centre, (0.0, 1.0, 0.0), 45.0)
            return Workload("cfg2_two_species_100M", n, w, h, f, sp, cam, meta=info)
        return Workload("cfg4_orbit_100M", n, w, h, f, sp, orbit_camera(0), meta=info)
    if cfg == 3:
        n = 400_000_000 if n is None else n
        w, h = size or (4096, 4096)
        f, info = _halo_set(seed, n, 1.5 if eta is None else eta, device, count=count)
        k = int(torch.argmax(info["halo_mass"]))
        c = info["halo_centre"][k]
        a = float(info["halo_scale"][k])
        eye = (float(c[0]) + 0.5 * a * 0.6, float(c[1]), float(c[2]) + 0.5 * a * 0.8)
        sp = [Species(0, n, brightness=1.0, scalar_min=info["scalar_min"], scalar_max=info["scalar_max"])]
        return Workload("cfg3_inside_halo_400M", n, w, h, f, sp, Camera(eye, centre, (0.0, 1.0, 0.0), 45.0),
                        r_large=64.0, meta=info)
    raise ValueError(f"unknown config {cfg}")
