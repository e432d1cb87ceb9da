"""ctypes front end of the CPU oracle (oracle/splotch_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package; inputs are plain numpy arrays and
duck-typed parameter objects (anything with the attributes named in `_species_arrays`).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "splotch_oracle.c")
_SRC_MT = os.path.join(_HERE, "splotch_oracle_mt.c")          # OpenMP drivers around the same functions
_LIB = os.path.join(_HERE, "libsplotch_oracle.so")
_lib = None

CULLED, SMALL, MEDIUM, LARGE = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fast-math, no contraction) if the .so is missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_MT)):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c99", "-fopenmp", "-shared", "-fPIC",
               "-o", _LIB + ".tmp", _SRC, _SRC_MT, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(_LIB + ".tmp", _LIB)
    return _LIB


def _p(a: np.ndarray, t):
    return a.ctypes.data_as(C.POINTER(t))


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_camera.restype = C.c_int
        _lib.orc_depth_order.restype = C.c_int64
        _lib.orc_mt_threads.restype = C.c_int
    return _lib


def host_cores() -> int:
    """Cores this process may run on (the all-cores drivers use that many threads)."""
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def _threads(threads: int) -> int:
    """threads <= 0 means all cores of the host; 1 means the single-threaded definition."""
    return host_cores() if threads <= 0 else threads


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def camera_constants(eye, lookat, up, fov_deg: float, W: int, H: int) -> np.ndarray:
    cam = np.zeros(16, np.float32)
    e, l, u = _f32(eye), _f32(lookat), _f32(up)
    rc = lib().orc_camera(_p(e, C.c_float), _p(l, C.c_float), _p(u, C.c_float), C.c_float(fov_deg),
                          C.c_int(W), C.c_int(H), _p(cam, C.c_float))
    if rc != 0:
        raise ValueError("degenerate camera")
    return cam


def geometry(x, y, z, h, cam: np.ndarray, chi: float, r_small: float, r_large: float,
             z_near: float, W: int, H: int, T: int, threads: int = 1) -> Dict[str, np.ndarray]:
    x, y, z, h = _f32(x), _f32(y), _f32(z), _f32(h)
    n = x.shape[0]
    g = {
        "cls": np.zeros(n, np.int8), "px": np.zeros(n, np.float32), "py": np.zeros(n, np.float32),
        "sp": np.zeros(n, np.float32), "rp": np.zeros(n, np.float32), "zc": np.zeros(n, np.float32),
        "pbox": np.zeros((n, 4), np.int32), "tbox": np.zeros((n, 4), np.int32),
        "ilabel": np.zeros(n, np.int32),
    }
    cam = _f32(cam)
    fn, lead = (lib().orc_geometry, []) if threads == 1 else (lib().orc_geometry_mt, [C.c_int(_threads(threads))])
    fn(*lead, C.c_int64(n), _p(x, C.c_float), _p(y, C.c_float), _p(z, C.c_float),
       _p(h, C.c_float), _p(cam, C.c_float), C.c_float(chi), C.c_float(r_small),
       C.c_float(r_large), C.c_float(z_near), C.c_int(W), C.c_int(H), C.c_int(T),
       _p(g["cls"], C.c_int8), _p(g["px"], C.c_float), _p(g["py"], C.c_float),
       _p(g["sp"], C.c_float), _p(g["rp"], C.c_float), _p(g["zc"], C.c_float),
       _p(g["pbox"], C.c_int32), _p(g["tbox"], C.c_int32), _p(g["ilabel"], C.c_int32))
    return g


def tile_counts(g: Dict[str, np.ndarray], W: int, H: int, T: int, count_large: bool = False) -> np.ndarray:
    ntx, nty = (W + T - 1) // T, (H + T - 1) // T
    counts = np.zeros(ntx * nty, np.uint32)
    n = g["cls"].shape[0]
    lib().orc_tile_counts(C.c_int64(n), _p(g["cls"], C.c_int8), _p(g["tbox"], C.c_int32),
                          C.c_int(ntx), C.c_int(nty), C.c_int(int(count_large)), _p(counts, C.c_uint32))
    return counts.reshape(nty, ntx)


def _species_arrays(n: int, species: Sequence, luts: Sequence[Optional[np.ndarray]]):
    ns = len(species)
    species_of = np.zeros(n, np.int32)
    bright = np.zeros(ns)
    kappa = np.zeros(ns)
    use_cm = np.zeros(ns, np.int32)
    fixed = np.zeros((ns, 3))
    smin = np.zeros(ns)
    smax = np.ones(ns)
    use_log = np.zeros(ns, np.int32)
    lut_off = np.zeros(ns, np.int32)
    lut_n = np.zeros(ns, np.int32)
    tables = []
    off = 0
    for s, sp in enumerate(species):
        species_of[sp.begin:sp.end] = s
        # parameters are float32 at the C ABI; the oracle sees those same float32 values
        bright[s] = np.float32(sp.brightness)
        kappa[s] = np.float32(sp.absorb)
        use_cm[s] = int(sp.use_colormap) if not getattr(sp, "vector_colour", False) else 0
        fixed[s] = np.asarray(sp.fixed_rgb, np.float32)
        smin[s] = np.float32(sp.scalar_min)
        smax[s] = np.float32(sp.scalar_max)
        use_log[s] = int(sp.scalar_log10)
        if use_cm[s]:
            t = np.asarray(luts[s], np.float32).astype(np.float64).reshape(-1, 3)
            lut_off[s], lut_n[s] = off, t.shape[0]
            tables.append(t)
            off += t.shape[0]
    lut = np.ascontiguousarray(np.concatenate(tables, 0)) if tables else np.zeros((2, 3))
    return species_of, bright, kappa, use_cm, np.ascontiguousarray(fixed), smin, smax, use_log, lut, lut_off, lut_n


def scalar_range(scalar, species: Sequence, vec=None) -> List[Tuple[float, float]]:
    """Per species (min, max) of the colour quantity over all its finite values: the scalar (after log10 if the species
    asks for it), or the three vector components together for a vector-colour species."""
    scalar = _f32(scalar)
    n = scalar.shape[0]
    ns = len(species)
    species_of = np.zeros(n, np.int32)
    use_log = np.zeros(ns, np.int32)
    for s, sp in enumerate(species):
        species_of[sp.begin:sp.end] = s
        use_log[s] = int(sp.scalar_log10) if not getattr(sp, "vector_colour", False) else 0
    out = []
    vmin, vmax = np.zeros(ns, np.float32), np.zeros(ns, np.float32)
    lib().orc_scalar_range(C.c_int64(n), _p(scalar, C.c_float), _p(species_of, C.c_int32), C.c_int(ns),
                           _p(use_log, C.c_int32), _p(vmin, C.c_float), _p(vmax, C.c_float))
    comp = []
    if vec is not None:
        for v in vec:
            a, b = np.zeros(ns, np.float32), np.zeros(ns, np.float32)
            v = _f32(v)
            lib().orc_scalar_range(C.c_int64(n), _p(v, C.c_float), _p(species_of, C.c_int32), C.c_int(ns),
                                   _p(np.zeros(ns, np.int32), C.c_int32), _p(a, C.c_float), _p(b, C.c_float))
            comp.append((a, b))
    for s, sp in enumerate(species):
        if getattr(sp, "vector_colour", False) and comp:
            # a component without a finite value reports (0, 1): leave it out unless all three are empty
            have = [(a[s], b[s]) for k, (a, b) in enumerate(comp) if np.isfinite(_f32(vec[k])[sp.begin:sp.end]).any()]
            out.append((float(min(a for a, _ in have)), float(max(b for _, b in have))) if have else (0.0, 1.0))
        else:
            out.append((float(vmin[s]), float(vmax[s])))
    return out


def resolve_ranges(fields: Dict[str, np.ndarray], species: Sequence):
    """Species parameters with the automatic ranges filled in (copies; the callers' objects stay untouched)."""
    import copy
    if not any(getattr(sp, "auto_range", False) for sp in species):
        return list(species)
    vec = [fields[k] for k in ("cr", "cg", "cb")] if "cr" in fields else None
    rng = scalar_range(fields["scalar"], species, vec)
    out = []
    for sp, (a, b) in zip(species, rng):
        sp2 = copy.copy(sp)
        if getattr(sp, "auto_range", False):
            sp2.scalar_min, sp2.scalar_max = a, b
        out.append(sp2)
    return out


def amplitude(I, scalar, h, species: Sequence, luts: Sequence, threads: int = 1, vec=None) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """E[n,3] = brightness * colour, col[n] = sqrt(pi) h I, kappa[n] (species' absorption).  vec = (cr, cg, cb) feeds
    the species in vector-colour mode."""
    I, scalar, h = _f32(I), _f32(scalar), _f32(h)
    n = I.shape[0]
    (species_of, bright, kappa, use_cm, fixed, smin, smax, use_log, lut, lut_off, lut_n) = \
        _species_arrays(n, species, luts)
    E = np.zeros((n, 3))
    col = np.zeros(n)
    fn, lead = (lib().orc_amplitude, []) if threads == 1 else (lib().orc_amplitude_mt, [C.c_int(_threads(threads))])
    fn(*lead, C.c_int64(n), _p(I, C.c_float), _p(scalar, C.c_float), _p(h, C.c_float),
       _p(species_of, C.c_int32), C.c_int(len(species)), _p(bright, C.c_double),
       _p(use_cm, C.c_int32), _p(fixed, C.c_double), _p(smin, C.c_double),
       _p(smax, C.c_double), _p(use_log, C.c_int32), _p(lut, C.c_double),
       _p(lut_off, C.c_int32), _p(lut_n, C.c_int32), _p(E, C.c_double), _p(col, C.c_double))
    vmode = np.array([int(getattr(sp, "vector_colour", False)) for sp in species], np.int32)
    if vmode.any():
        if vec is None:
            raise ValueError("a species is in vector-colour mode but no vector fields were given")
        vr, vg, vb = (_f32(v) for v in vec)
        lib().orc_amplitude_vector(C.c_int64(n), _p(vr, C.c_float), _p(vg, C.c_float), _p(vb, C.c_float),
                                   _p(species_of, C.c_int32), _p(vmode, C.c_int32), _p(bright, C.c_double),
                                   _p(smin, C.c_double), _p(smax, C.c_double), _p(E, C.c_double))
    return E, col, kappa[species_of]


def _bands(threads: int) -> int:
    return 4 * _threads(threads)          # several bands per thread: rows through a halo core cost more


def render_additive(g, E, col, chi: float, W: int, H: int, window=None, apply_transfer=False,
                    p_range=None, image: Optional[np.ndarray] = None, threads: int = 1) -> np.ndarray:
    n = g["cls"].shape[0]
    if image is None:
        image = np.zeros((H, W, 3))
    wx0, wx1, wy0, wy1 = window if window is not None else (0, W - 1, 0, H - 1)
    pb, pe = p_range if p_range is not None else (0, n)
    fn, lead = ((lib().orc_render_additive, []) if threads == 1 else
                (lib().orc_render_additive_mt, [C.c_int(_threads(threads)), C.c_int(_bands(threads))]))
    fn(*lead, C.c_int64(pb), C.c_int64(pe), _p(g["cls"], C.c_int8), _p(g["px"], C.c_float),
       _p(g["py"], C.c_float), _p(g["sp"], C.c_float), _p(g["rp"], C.c_float),
       _p(g["pbox"], C.c_int32), _p(E, C.c_double), _p(col, C.c_double),
       C.c_float(chi), C.c_int(W), C.c_int(H), C.c_int(wx0), C.c_int(wx1),
       C.c_int(wy0), C.c_int(wy1), C.c_int(int(apply_transfer)), _p(image, C.c_double))
    return image


def depth_order(g) -> np.ndarray:
    n = g["cls"].shape[0]
    order = np.zeros(max(n, 1), np.int64)
    m = lib().orc_depth_order(C.c_int64(n), _p(g["cls"], C.c_int8), _p(g["zc"], C.c_float), _p(order, C.c_int64))
    if m < 0:
        raise MemoryError
    return order[:m].copy()


def render_ordered(g, E, col, kappa, chi: float, W: int, H: int, window=None, order=None, threads: int = 1) -> np.ndarray:
    image = np.zeros((H, W, 3))
    if order is None:
        order = depth_order(g)
    order = np.ascontiguousarray(order, np.int64)
    kappa = np.ascontiguousarray(kappa, np.float64)
    wx0, wx1, wy0, wy1 = window if window is not None else (0, W - 1, 0, H - 1)
    fn, lead = ((lib().orc_render_ordered, []) if threads == 1 else
                (lib().orc_render_ordered_mt, [C.c_int(_threads(threads)), C.c_int(_threads(threads))]))
    fn(*lead, C.c_int64(order.shape[0]), _p(order, C.c_int64), _p(g["cls"], C.c_int8),
       _p(g["px"], C.c_float), _p(g["py"], C.c_float), _p(g["sp"], C.c_float),
       _p(g["rp"], C.c_float), _p(g["pbox"], C.c_int32), _p(E, C.c_double),
       _p(col, C.c_double), _p(kappa, C.c_double), C.c_float(chi), C.c_int(W),
       C.c_int(H), C.c_int(wx0), C.c_int(wx1), C.c_int(wy0), C.c_int(wy1),
       _p(image, C.c_double))
    return image


def render(fields: Dict[str, np.ndarray], species: Sequence, luts: Sequence, camera, W: int, H: int,
           chi: float = 3.0, r_small: float = 0.5, r_large: float = 64.0, z_near: float = 1e-6,
           tile: int = 16, additive: bool = True, apply_transfer: bool = False, window=None,
           return_geometry: bool = False, threads: int = 1):
    """Whole path on numpy float32 fields {x,y,z,h,I,scalar}: camera -> C1 -> C2 -> image (float64 HxWx3).

    threads = 1 is the definition (single thread, index order); threads = 0 (all cores) or > 1 runs the same
    functions through the row-band drivers of splotch_oracle_mt.c, bit-identical by construction."""
    cam = camera_constants(camera.eye, camera.lookat, camera.up, camera.fov_deg, W, H)
    g = geometry(fields["x"], fields["y"], fields["z"], fields["h"], cam, chi, r_small, r_large, z_near, W, H, tile,
                 threads=threads)
    species = resolve_ranges(fields, species)
    vec = [fields[k] for k in ("cr", "cg", "cb")] if "cr" in fields else None
    E, col, kappa = amplitude(fields["I"], fields["scalar"], fields["h"], species, luts, threads=threads, vec=vec)
    if additive:
        img = render_additive(g, E, col, chi, W, H, window=window, apply_transfer=apply_transfer, threads=threads)
    else:
        img = render_ordered(g, E, col, kappa, chi, W, H, window=window, threads=threads)
    return (img, g, cam) if return_geometry else img
