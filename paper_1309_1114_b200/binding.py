"""Thin ctypes binding of the C ABI in include/splotch.h -- argument marshalling only.

Module-level functions carry the C names (splotch_create, splotch_set_camera, splotch_set_colormap,
splotch_render, splotch_destroy, ...) and take raw pointers / ctypes structs.  `Renderer` is a small
convenience wrapper that owns a context, allocates the workspace and the image with torch and passes
`tensor.data_ptr()` and the current CUDA stream.  Every step of the path runs inside the library's CUDA
kernels; there is no CPU fallback: a missing library raises, it is never replaced.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Sequence, Tuple

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsplotch_b200.so")

SPLOTCH_OK, SPLOTCH_EINVAL, SPLOTCH_ENOMEM, SPLOTCH_ECUDA, SPLOTCH_EDEVICE, SPLOTCH_ESTATE = 0, -1, -2, -3, -4, -5
CULLED, SMALL, MEDIUM, LARGE = 0, 1, 2, 3
MAX_SPECIES = 8

EXPORTS = (
    "splotch_create", "splotch_destroy", "splotch_set_camera", "splotch_get_camera_constants",
    "splotch_set_colormap", "splotch_set_profiling", "splotch_workspace_bytes", "splotch_render",
    "splotch_render_host", "splotch_get_stats", "splotch_stage_name", "splotch_debug_geometry",
    "splotch_debug_tile_counts", "splotch_last_error", "splotch_version", "splotch_measure_peaks", "splotch_set_host_chunk", "splotch_apply_transfer",
    "splotch_count_static", "splotch_compose_shards",
)


class SplotchParticles(C.Structure):
    _fields_ = [("x", C.c_void_p), ("y", C.c_void_p), ("z", C.c_void_p), ("h", C.c_void_p), ("I", C.c_void_p),
                ("scalar", C.c_void_p), ("species_offsets", C.POINTER(C.c_uint64)), ("n_species", C.c_int),
                ("cr", C.c_void_p), ("cg", C.c_void_p), ("cb", C.c_void_p)]


class SplotchSpeciesParams(C.Structure):
    _fields_ = [("brightness", C.c_float), ("absorb", C.c_float), ("use_colormap", C.c_int),
                ("fixed_rgb", C.c_float * 3), ("scalar_min", C.c_float), ("scalar_max", C.c_float),
                ("scalar_log10", C.c_int), ("auto_range", C.c_int), ("vector_colour", C.c_int)]


class SplotchParams(C.Structure):
    _fields_ = [("chi", C.c_float), ("r_small", C.c_float), ("r_large", C.c_float), ("z_near", C.c_float),
                ("tile", C.c_int), ("additive", C.c_int), ("apply_transfer", C.c_int),
                ("species", C.POINTER(SplotchSpeciesParams)), ("renderer", C.c_int), ("btile_np", C.c_int)]


class SplotchStats(C.Structure):
    _fields_ = [("n", C.c_uint64), ("count", C.c_uint64 * 4), ("pairs", C.c_uint64), ("large_pairs", C.c_uint64),
                ("chunks", C.c_uint64), ("pair_capacity", C.c_uint64), ("overflow", C.c_int32),
                ("n_stages", C.c_int32), ("stage_ms", C.c_float * 8), ("sort_key_bits", C.c_int32),
                ("reserved", C.c_int32)]


class SplotchError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"splotch error {code}: {msg}")
        self.code = code


_lib = None


def load() -> C.CDLL:
    """Load the C-ABI library.  Raises if it has not been built (python -m paper_1309_1114_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1309_1114_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, u64, i32, f32p = C.c_void_p, C.c_uint64, C.c_int, C.POINTER(C.c_float)
    lib.splotch_create.argtypes = [C.POINTER(vp), i32, i32, i32, u64]
    lib.splotch_destroy.argtypes = [vp]
    lib.splotch_set_camera.argtypes = [vp, f32p, f32p, f32p, C.c_float]
    lib.splotch_get_camera_constants.argtypes = [vp, f32p]
    lib.splotch_set_colormap.argtypes = [vp, i32, f32p, i32]
    lib.splotch_set_profiling.argtypes = [vp, i32]
    lib.splotch_workspace_bytes.argtypes = [vp, u64, i32, u64, i32]
    lib.splotch_workspace_bytes.restype = C.c_size_t
    lib.splotch_render.argtypes = [vp, C.POINTER(SplotchParticles), u64, C.POINTER(SplotchParams), vp, vp, C.c_size_t, vp]
    lib.splotch_render_host.argtypes = lib.splotch_render.argtypes
    lib.splotch_get_stats.argtypes = [vp, C.POINTER(SplotchStats)]
    lib.splotch_stage_name.argtypes = [i32, i32]
    lib.splotch_stage_name.restype = C.c_char_p
    lib.splotch_debug_geometry.argtypes = [vp, C.POINTER(SplotchParticles), u64, C.POINTER(SplotchParams)] + [vp] * 10
    lib.splotch_debug_tile_counts.argtypes = [vp, vp, vp]
    lib.splotch_compose_shards.argtypes = [vp, C.POINTER(vp), i32, i32, i32, i32, i32, vp, vp]
    lib.splotch_count_static.argtypes = [vp, C.POINTER(SplotchParticles), u64, C.POINTER(SplotchParams), vp, vp, vp]
    lib.splotch_measure_peaks.argtypes = [vp, C.POINTER(C.c_double), vp]
    lib.splotch_set_host_chunk.argtypes = [vp, u64]
    lib.splotch_apply_transfer.argtypes = [vp, vp, vp]
    lib.splotch_last_error.argtypes = [vp]
    lib.splotch_last_error.restype = C.c_char_p
    lib.splotch_version.restype = C.c_char_p
    for name in EXPORTS:
        if getattr(lib, name).restype is C.c_int:
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


# ---- C names, raw marshalling ------------------------------------------------------------------------------------
def _f3(v):
    return (C.c_float * 3)(*[float(t) for t in v])


def splotch_create(device: int, width: int, height: int, max_particles: int) -> C.c_void_p:
    ctx = C.c_void_p()
    rc = load().splotch_create(C.byref(ctx), device, width, height, max_particles)
    if rc != SPLOTCH_OK:
        raise SplotchError(rc, "splotch_create: " + load().splotch_last_error(None).decode())
    return ctx


def _check(ctx, rc):
    if rc != SPLOTCH_OK:
        raise SplotchError(rc, load().splotch_last_error(ctx).decode())


def splotch_destroy(ctx) -> None:
    load().splotch_destroy(ctx)


def splotch_set_camera(ctx, eye, lookat, up, fov_deg: float) -> None:
    _check(ctx, load().splotch_set_camera(ctx, _f3(eye), _f3(lookat), _f3(up), float(fov_deg)))


def splotch_get_camera_constants(ctx):
    out = (C.c_float * 16)()
    _check(ctx, load().splotch_get_camera_constants(ctx, out))
    return list(out)


def splotch_set_colormap(ctx, species: int, rgb) -> None:
    t = torch.as_tensor(rgb, dtype=torch.float32, device="cpu").contiguous().reshape(-1, 3)
    _check(ctx, load().splotch_set_colormap(ctx, species, C.cast(t.data_ptr(), C.POINTER(C.c_float)), t.shape[0]))


def splotch_workspace_bytes(ctx, n: int, tile: int, pair_capacity: int = 0, with_host_staging: bool = False) -> int:
    return int(load().splotch_workspace_bytes(ctx, n, tile, pair_capacity, int(with_host_staging)))


def make_params(species: Sequence, chi=3.0, r_small=0.5, r_large=64.0, z_near=1e-6, tile=16, additive=True,
                apply_transfer=False, renderer=0, btile_np=0):
    """(SplotchParams, keep-alive array) from objects with the attributes of workloads.Species."""
    arr = (SplotchSpeciesParams * len(species))()
    for k, s in enumerate(species):
        arr[k].brightness = s.brightness
        arr[k].absorb = s.absorb
        arr[k].use_colormap = int(s.use_colormap)
        arr[k].fixed_rgb = _f3(s.fixed_rgb)
        arr[k].scalar_min = s.scalar_min
        arr[k].scalar_max = s.scalar_max
        arr[k].scalar_log10 = int(s.scalar_log10)
        arr[k].auto_range = int(getattr(s, "auto_range", False))
        arr[k].vector_colour = int(getattr(s, "vector_colour", False))
    p = SplotchParams(chi, r_small, r_large, z_near, tile, int(additive), int(apply_transfer),
                      C.cast(arr, C.POINTER(SplotchSpeciesParams)), int(renderer), int(btile_np))
    return p, arr


def make_particles(fields: Dict[str, torch.Tensor], species: Sequence):
    """(SplotchParticles, keep-alive) from float32 tensors x y z h I scalar (device or host)."""
    n = fields["x"].numel()
    ptrs = {}
    for k in ("x", "y", "z", "h", "I", "scalar"):
        t = fields[k]
        if t.dtype != torch.float32 or not t.is_contiguous() or t.numel() != n:
            raise ValueError(f"field {k} must be a contiguous float32 tensor of length {n}")
        ptrs[k] = t.data_ptr()
    offs = (C.c_uint64 * (len(species) + 1))(*([s.begin for s in species] + [species[-1].end]))
    vec = []
    for k in ("cr", "cg", "cb"):
        t = fields.get(k)
        if t is not None and (t.dtype != torch.float32 or not t.is_contiguous() or t.numel() != n):
            raise ValueError(f"field {k} must be a contiguous float32 tensor of length {n}")
        vec.append(t.data_ptr() if t is not None else None)
    p = SplotchParticles(ptrs["x"], ptrs["y"], ptrs["z"], ptrs["h"], ptrs["I"], ptrs["scalar"],
                         C.cast(offs, C.POINTER(C.c_uint64)), len(species), *vec)
    return p, offs


class Renderer:
    """Owns a splotch_ctx; allocates image and workspace with torch; marshals arguments. Nothing else."""

    def __init__(self, width: int, height: int, max_particles: int, device: int = 0):
        self.lib = load()
        self.width, self.height, self.device = width, height, device
        self.ctx = splotch_create(device, width, height, max_particles)
        self._ws: Optional[torch.Tensor] = None

    def close(self):
        if self.ctx is not None:
            splotch_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_camera(self, cam) -> None:
        splotch_set_camera(self.ctx, cam.eye, cam.lookat, cam.up, cam.fov_deg)

    def set_colormap(self, species: int, rgb) -> None:
        splotch_set_colormap(self.ctx, species, rgb)

    def set_profiling(self, on: bool) -> None:
        _check(self.ctx, self.lib.splotch_set_profiling(self.ctx, int(on)))

    def set_host_chunk(self, particles_per_chunk: int) -> None:
        _check(self.ctx, self.lib.splotch_set_host_chunk(self.ctx, particles_per_chunk))
        self._ws = None

    def apply_transfer(self, image: torch.Tensor) -> torch.Tensor:
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(self.ctx, self.lib.splotch_apply_transfer(self.ctx, image.data_ptr(), stream))
        return image

    def measure_peaks(self) -> Dict[str, float]:
        out = (C.c_double * 2)()
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(self.ctx, self.lib.splotch_measure_peaks(self.ctx, out, stream))
        return {"fma_lane_ops_per_s": out[0], "mufu_ex2_per_s": out[1]}

    def camera_constants(self):
        return splotch_get_camera_constants(self.ctx)

    def workspace(self, n: int, tile: int, pair_capacity: int = 0, host_staging: bool = False) -> torch.Tensor:
        need = splotch_workspace_bytes(self.ctx, n, tile, pair_capacity, host_staging)
        if need == 0:
            raise SplotchError(SPLOTCH_EINVAL, "splotch_workspace_bytes rejected (n, tile, pair_capacity)")
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = torch.empty(need, dtype=torch.uint8, device=f"cuda:{self.device}")
        return self._ws

    def render(self, fields: Dict[str, torch.Tensor], species: Sequence, image: Optional[torch.Tensor] = None,
               pair_capacity: int = 0, **params) -> torch.Tensor:
        n = fields["x"].numel()
        prm, keep1 = make_params(species, **params)
        prt, keep2 = make_particles(fields, species)
        ws = self.workspace(n, prm.tile, pair_capacity)
        if image is None:
            image = torch.empty((self.height, self.width, 3), dtype=torch.float32, device=f"cuda:{self.device}")
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(self.ctx, self.lib.splotch_render(self.ctx, C.byref(prt), n, C.byref(prm), image.data_ptr(),
                                                 ws.data_ptr(), ws.numel(), stream))
        return image

    def render_host(self, fields: Dict[str, torch.Tensor], species: Sequence, image: torch.Tensor,
                    pair_capacity: int = 0, **params) -> torch.Tensor:
        """fields and image are HOST tensors (pinned for asynchronous copies); synchronises before returning."""
        n = fields["x"].numel()
        prm, keep1 = make_params(species, **params)
        prt, keep2 = make_particles(fields, species)
        ws = self.workspace(n, prm.tile, pair_capacity, host_staging=True)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(self.ctx, self.lib.splotch_render_host(self.ctx, C.byref(prt), n, C.byref(prm), image.data_ptr(),
                                                      ws.data_ptr(), ws.numel(), stream))
        return image

    def stats(self) -> Dict[str, object]:
        st = SplotchStats()
        _check(self.ctx, self.lib.splotch_get_stats(self.ctx, C.byref(st)))
        d = {"n": st.n, "count": list(st.count), "pairs": st.pairs, "large_pairs": st.large_pairs,
             "chunks": st.chunks, "pair_capacity": st.pair_capacity, "overflow": st.overflow,
             "sort_key_bits": st.sort_key_bits,
             "stage_ms": {self.lib.splotch_stage_name(int(st.n_stages < 7), i).decode(): st.stage_ms[i]
                          for i in range(st.n_stages)}}
        return d

    def debug_geometry(self, fields: Dict[str, torch.Tensor], species: Sequence, **params) -> Dict[str, torch.Tensor]:
        n = fields["x"].numel()
        dev = fields["x"].device
        prm, keep1 = make_params(species, **params)
        prt, keep2 = make_particles(fields, species)
        out = {"cls": torch.empty(n, dtype=torch.int8, device=dev)}
        for k in ("px", "py", "sp", "rp", "zc"):
            out[k] = torch.empty(n, dtype=torch.float32, device=dev)
        out["pbox"] = torch.empty((n, 4), dtype=torch.int32, device=dev)
        out["tbox"] = torch.empty((n, 4), dtype=torch.int32, device=dev)
        out["ilabel"] = torch.empty(n, dtype=torch.int32, device=dev)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(self.ctx, self.lib.splotch_debug_geometry(
            self.ctx, C.byref(prt), n, C.byref(prm), *[out[k].data_ptr() for k in
                                                      ("cls", "px", "py", "sp", "rp", "zc", "pbox", "tbox", "ilabel")],
            stream))
        return out

    def compose_shards(self, workspaces: Sequence[torch.Tensor], tile: int, image: Optional[torch.Tensor] = None,
                       tile_range: Tuple[int, int] = (0, -1), apply_transfer: bool = False) -> torch.Tensor:
        """splotch_compose_shards: the image of a particle-sharded frame from the shards' workspaces (exact sum of their
        fixed-point tile sums), tiles tile_range of it."""
        if image is None:
            image = torch.zeros((self.height, self.width, 3), dtype=torch.float32, device=f"cuda:{self.device}")
        ptrs = (C.c_void_p * len(workspaces))(*[w.data_ptr() for w in workspaces])
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(self.ctx, self.lib.splotch_compose_shards(self.ctx, ptrs, len(workspaces), tile, tile_range[0], tile_range[1],
                                                         1 if apply_transfer else 0, image.data_ptr(), stream))
        return image

    @property
    def last_workspace(self) -> Optional[torch.Tensor]:
        """The workspace of the last frame (holds the tiles' fixed-point sums until the next frame)."""
        return self._ws

    def count_static(self, fields: Dict[str, torch.Tensor], species: Sequence, tile_counts: torch.Tensor,
                     class_counts: torch.Tensor, **params) -> None:
        """splotch_count_static: classes and per-tile pair counts into the caller's DEVICE tensors (nty x ntx int32 and
        int64[4]); the library call allocates nothing (its scratch is a static device array)."""
        n = fields["x"].numel()
        prm, keep1 = make_params(species, **params)
        prt, keep2 = make_particles(fields, species)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(self.ctx, self.lib.splotch_count_static(self.ctx, C.byref(prt), n, C.byref(prm), tile_counts.data_ptr(),
                                                       class_counts.data_ptr(), stream))

    def debug_tile_counts(self, tile: int) -> torch.Tensor:
        ntx, nty = -(-self.width // tile), -(-self.height // tile)
        out = torch.empty((nty, ntx), dtype=torch.int32, device=f"cuda:{self.device}")
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(self.ctx, self.lib.splotch_debug_tile_counts(self.ctx, out.data_ptr(), stream))
        return out
