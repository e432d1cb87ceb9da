"""Additive-mode particle sharding over several GPUs (the paper's MPI scheme: "distributes
chunks of particles among different processors, each ... producing a partial rendering, the root processor composing
final renderings"; multi-GPU is its stated future work, :356).

With E_p = A_p the frame is S = sum_p E_p tau_p: a sum over particles, so rank r renders the particles of
its contiguous index range into a partial image with the single-GPU path and the partial images are added with ONE
collective, a sum all-reduce of the 12 W H-byte float32 image over NCCL (NVLink 5 / NVSwitch).  The transfer
1 - exp(-S) is not linear and is applied after the sum (splotch_apply_transfer).  The ordered mode does not shard by
particles (its composition is not a sum) and is refused here.

Only argument marshalling and the collective live in this module; every step of the path runs in the library's kernels.
`partial_render` is injectable so that the rank logic can be exercised on CPU ranks (gloo) in the tests.
"""
from __future__ import annotations

import copy
from typing import Callable, Dict, List, Optional, Sequence, Tuple

import torch


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous index range of `rank`: equal shares rounded up to a multiple of 4 particles (aligned vector loads)."""
    per = -(-n // world)
    per = -(-per // 4) * 4
    lo = min(n, rank * per)
    return lo, min(n, lo + per)


def shard_species(species: Sequence, lo: int, hi: int) -> List:
    """The species ranges of the set [0, n) cut to [lo, hi) and re-based to the shard."""
    out = []
    for sp in species:
        s2 = copy.copy(sp)
        s2.begin = min(max(sp.begin, lo), hi) - lo
        s2.end = min(max(sp.end, lo), hi) - lo
        out.append(s2)
    return out


def shard_fields(fields: Dict[str, torch.Tensor], lo: int, hi: int) -> Dict[str, torch.Tensor]:
    return {k: v[lo:hi].contiguous() for k, v in fields.items()}


def global_ranges(fields: Dict[str, torch.Tensor], species: Sequence, dist=None) -> List:
    """Species with auto_range need the extrema over ALL ranks: resolve them with two tiny all-reduces (min, max) and hand
    every rank the same explicit range.  Finite values only, log10 first where the species asks for it."""
    if not any(getattr(sp, "auto_range", False) for sp in species):
        return list(species)
    out = []
    for sp in species:
        s2 = copy.copy(sp)
        if getattr(sp, "auto_range", False):
            keys = ("cr", "cg", "cb") if getattr(sp, "vector_colour", False) else ("scalar",)
            lo_v = torch.tensor(float("inf"), dtype=torch.float32, device=fields["x"].device)
            hi_v = torch.tensor(float("-inf"), dtype=torch.float32, device=fields["x"].device)
            for k in keys:
                v = fields[k][sp.begin:sp.end]
                if sp.scalar_log10 and not getattr(sp, "vector_colour", False):
                    v = torch.log10(v.double()).to(torch.float32)
                v = v[torch.isfinite(v)]
                if v.numel():
                    lo_v, hi_v = torch.minimum(lo_v, v.min()), torch.maximum(hi_v, v.max())
            if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
                dist.all_reduce(lo_v, op=dist.ReduceOp.MIN)
                dist.all_reduce(hi_v, op=dist.ReduceOp.MAX)
            if not bool(lo_v <= hi_v):
                lo_v, hi_v = torch.tensor(0.0), torch.tensor(1.0)
            s2.scalar_min, s2.scalar_max, s2.auto_range = float(lo_v), float(hi_v), False
        out.append(s2)
    return out


def sharded_frame(partial_render: Callable[[Dict[str, torch.Tensor], List, Dict], torch.Tensor],
                  fields: Dict[str, torch.Tensor], species: Sequence, params: Dict, dist=None,
                  apply_transfer_fn: Optional[Callable[[torch.Tensor], torch.Tensor]] = None) -> torch.Tensor:
    """One frame from THIS rank's shard (`fields`, `species` already cut with shard_fields / shard_species):
    partial image -> sum all-reduce -> optional transfer.  Every rank returns the full image."""
    if not params.get("additive", True):
        raise ValueError("particle sharding is valid in the additive (E = A) mode only: the ordered composition is not a sum")
    want_transfer = bool(params.get("apply_transfer", False))
    species = global_ranges(fields, species, dist)
    image = partial_render(fields, species, dict(params, additive=True, apply_transfer=False))
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(image, op=dist.ReduceOp.SUM)              # the one collective of the data path
    if want_transfer:
        image = apply_transfer_fn(image) if apply_transfer_fn is not None else -torch.expm1(-image)
    return image


class ShardedRenderer:
    """One process per GPU: owns a single-GPU Renderer and the rank's shard; NCCL through torch.distributed."""

    def __init__(self, width: int, height: int, n_total: int, device: int, dist=None):
        from . import binding
        self.dist = dist
        self.rank = dist.get_rank() if dist is not None and dist.is_initialized() else 0
        self.world = dist.get_world_size() if dist is not None and dist.is_initialized() else 1
        self.lo, self.hi = shard_range(n_total, self.rank, self.world)
        self.r = binding.Renderer(width, height, max(self.hi - self.lo, 1), device=device)

    def set_camera(self, cam) -> None:
        self.r.set_camera(cam)

    def set_colormap(self, species: int, rgb) -> None:
        self.r.set_colormap(species, rgb)

    def render(self, shard_fields_dev: Dict[str, torch.Tensor], shard_species_: Sequence, **params) -> torch.Tensor:
        def partial(f, sp, prm):
            return self.r.render(f, sp, **prm)
        return sharded_frame(partial, shard_fields_dev, shard_species_, params, self.dist, self.r.apply_transfer)

    def close(self) -> None:
        self.r.close()
