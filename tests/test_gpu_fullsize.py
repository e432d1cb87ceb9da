"""GPU parity at BASELINE.json's full sizes (configs 2, 3, 4), in the launch configuration the library uses for them.

The oracle cannot render 1e8 .. 4e8 particles in seconds, so at full size
  * the integer work is compared exhaustively: the oracle's C1 geometry runs over ALL particles in chunks and its
    class counts and per-tile pair counts must equal the library's bit for bit; on a strided sample of chunks the
    per-particle float32 geometry, boxes and labels are compared bit for bit as well;
  * the image is compared on sampled windows: for each window the particles that can touch it are selected from the
    RAW inputs by a conservative float64 projection written here (plain torch, neither oracle nor CUDA path; two
    pixels of margin), the oracle renders exactly that subset (a particle outside the selection contributes nothing
    to the window, and the subset keeps index order, so the oracle's sum and its depth order are those of the full
    set), and the library's image must match it inside the window to the north_star tolerance.
"""
import math

import numpy as np
import pytest
import torch

from oracle import splotch_oracle as so
from paper_1309_1114_b200 import workloads as wl

pytestmark = pytest.mark.gpu

REL_L2 = 1e-5
MAX_ABS = 1e-4
CHUNK = 1 << 24


def _binding():
    from paper_1309_1114_b200 import binding
    return binding


def camera_basis64(cam, W):
    """float64 pin-hole basis (test-side prefilter only)."""
    eye = np.asarray(cam.eye, np.float64)
    f = np.asarray(cam.lookat, np.float64) - eye
    f /= np.linalg.norm(f)
    r = np.cross(f, np.asarray(cam.up, np.float64))
    r /= np.linalg.norm(r)
    u = np.cross(r, f)
    s = 0.5 * W / math.tan(0.5 * math.radians(cam.fov_deg))
    return eye, r, u, f, s


def select_for_window(fields, cam, W, H, chi, window, margin=2.0):
    """Indices (ascending) of particles whose clip disc, grown by `margin` px, may touch the window."""
    wx0, wx1, wy0, wy1 = window
    eye, r, u, f, s = camera_basis64(cam, W)
    dev = fields["x"].device
    out = []
    n = fields["x"].numel()
    for a in range(0, n, CHUNK):
        b = min(n, a + CHUNK)
        d = [fields[k][a:b].double() - float(eye[i]) for i, k in enumerate("xyz")]
        zc = sum(float(f[i]) * d[i] for i in range(3))
        xc = sum(float(r[i]) * d[i] for i in range(3))
        yc = sum(float(u[i]) * d[i] for i in range(3))
        k = s / zc
        px, py = 0.5 * W + xc * k, 0.5 * H - yc * k
        rad = chi * fields["h"][a:b].double() * k + margin
        keep = (zc > 0) & (px + rad >= wx0) & (px - rad <= wx1 + 1) & (py + rad >= wy0) & (py - rad <= wy1 + 1)
        out.append(torch.nonzero(keep).squeeze(1) + a)
    return torch.cat(out).to(dev)


def subset_species(species, idx):
    import copy
    res, pos = [], 0
    idx_cpu = idx.cpu()
    for sp in species:
        cnt = int(((idx_cpu >= sp.begin) & (idx_cpu < sp.end)).sum())
        s2 = copy.copy(sp)
        s2.begin, s2.end = pos, pos + cnt
        pos += cnt
        res.append(s2)
    return res


def make_renderer(w, lut):
    b = _binding()
    r = b.Renderer(w.width, w.height, w.n)
    r.set_camera(w.camera)
    for s, sp in enumerate(w.species):
        if sp.use_colormap:
            r.set_colormap(s, lut)
    return r


def check_integer_work(r, w, kw, tile, geometry_every=8, count_large=False):
    """Oracle C1 over all particles in chunks: class counts, per-tile counts; sampled chunks bit-exact per particle."""
    cam = so.camera_constants(w.camera.eye, w.camera.lookat, w.camera.up, w.camera.fov_deg, w.width, w.height)
    assert np.array_equal(np.asarray(r.camera_constants(), np.float32), cam)
    ntx, nty = -(-w.width // tile), -(-w.height // tile)
    counts = np.zeros(4, np.int64)
    tiles = np.zeros((nty, ntx), np.int64)
    for ci, a in enumerate(range(0, w.n, CHUNK)):
        b = min(w.n, a + CHUNK)
        fc = {k: w.fields[k][a:b] for k in ("x", "y", "z", "h")}
        g = so.geometry(*[fc[k].cpu().numpy() for k in ("x", "y", "z", "h")], cam, w.chi, w.r_small, w.r_large,
                        w.z_near, w.width, w.height, tile)
        counts += np.bincount(g["cls"], minlength=4)
        tiles += so.tile_counts(g, w.width, w.height, tile, count_large=count_large)
        if ci % geometry_every == 0:
            sub = {k: w.fields[k][a:b] for k in wl.FIELD_NAMES}
            sp1 = [wl.Species(0, b - a)]
            d = r.debug_geometry(sub, sp1, **dict(kw, additive=True))
            for k in ("cls", "pbox", "tbox", "ilabel"):
                assert np.array_equal(d[k].cpu().numpy(), g[k]), (k, ci)
            act = g["cls"] != so.CULLED
            for k in ("px", "py", "sp", "rp"):
                assert np.array_equal(d[k].cpu().numpy()[act].view(np.uint32), g[k][act].view(np.uint32)), (k, ci)
            assert np.array_equal(d["zc"].cpu().numpy().view(np.uint32), g["zc"].view(np.uint32)), ("zc", ci)
    return counts, tiles


def check_windows(img, w, lut, kw, windows, additive=True):
    lutn = lut.numpy()
    num = den = 0.0
    worst, vmax = 0.0, 0.0
    for win in windows:
        idx = select_for_window(w.fields, w.camera, w.width, w.height, w.chi, win)
        sub = {k: w.fields[k][idx].cpu().numpy() for k in wl.FIELD_NAMES}
        sps = subset_species(w.species, idx)
        ref = so.render(sub, sps, [lutn if s.use_colormap else None for s in sps], w.camera, w.width, w.height,
                        chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=kw["tile"],
                        additive=additive, apply_transfer=False, window=win)
        wx0, wx1, wy0, wy1 = win
        a = ref[wy0:wy1 + 1, wx0:wx1 + 1]
        g = img[wy0:wy1 + 1, wx0:wx1 + 1].double().cpu().numpy()
        assert np.isfinite(g).all()
        num += float(((g - a) ** 2).sum())
        den += float((a ** 2).sum())
        worst = max(worst, float(np.abs(g - a).max()))
        vmax = max(vmax, float(a.max()))
    assert den > 0, "windows are empty"
    rel = math.sqrt(num / den)
    # scale: the largest oracle value inside the sampled windows (<= the image maximum, so this is the stricter bound)
    assert rel <= REL_L2, f"{w.name}: relative L2 over windows {rel:.3e}"
    assert worst <= MAX_ABS * vmax, f"{w.name}: max abs {worst:.3e} vs {MAX_ABS * vmax:.3e}"
    return rel, worst / vmax


def windows_for(img, size, n_random, seed):
    """The window around the brightest pixel, one at the image centre, one at the ragged bottom-right corner and
    n_random seeded ones.  (The library's image only chooses WHERE to look; expected values come from the oracle.)"""
    H, W = img.shape[:2]
    lum = img.sum(dim=2)
    j, i = divmod(int(torch.argmax(lum)), W)
    rng = np.random.default_rng(seed)
    cs = [(i, j), (W // 2, H // 2), (W - size // 2, H - size // 2)]
    cs += [(int(rng.integers(0, W)), int(rng.integers(0, H))) for _ in range(n_random)]
    out = []
    for cx, cy in cs:
        x0 = min(max(cx - size // 2, 0), W - size)
        y0 = min(max(cy - size // 2, 0), H - size)
        out.append((x0, x0 + size - 1, y0, y0 + size - 1))
    return out


def run_fullsize(cfg, tile, n_random=3, win=32, modes=(True,), camera=None, w=None):
    lut = wl.palette()
    if w is None:
        w = wl.make_config(cfg, device="cuda")
        w.fields = {k: v.contiguous() for k, v in w.fields.items()}
    if camera is not None:
        w.camera = camera
    r = make_renderer(w, lut)
    res = {}
    for additive in modes:
        kw = dict(chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=tile, additive=additive,
                  apply_transfer=False)
        img = r.render(w.fields, w.species, **kw)
        torch.cuda.synchronize()
        st = r.stats()
        assert st["overflow"] == 0
        if True:
            counts, tiles = check_integer_work(r, w, kw, tile, count_large=not additive)
            assert st["count"] == [int(c) for c in counts]
            gc = r.debug_tile_counts(tile).cpu().numpy().astype(np.int64)
            assert np.array_equal(gc, tiles)
            assert st["pairs"] == int(tiles.sum())
        res[additive] = (st, check_windows(img, w, lut, kw, windows_for(img, win, n_random, 7 + cfg), additive=additive))
    r.close()
    return w, res


def test_cfg2_full_size_two_species_100M():
    w, res = run_fullsize(2, 16)
    st, (rel, mab) = res[True]
    assert st["count"][1] > 30_000_000 and st["count"][2] > 10_000_000


def test_cfg3_full_size_inside_halo_400M():
    """4096 x 4096, camera inside the densest halo, a few per cent LARGE particles (tile 32: the per-block histogram
    of 65,536 16-px tiles would not fit in shared memory)."""
    w, res = run_fullsize(3, 32, n_random=2, win=24)
    st, (rel, mab) = res[True]
    assert st["count"][3] > 0.02 * w.n, st["count"]          # the large-particle stress BASELINE.json asks for


def test_cfg4_orbit_frames_100M_additive_and_ordered():
    """Frames {0, 30, 60, 90, 119} of the 120-frame orbit at full size, first in additive mode, then in the ordered
    E != A mode (kappa_gas = 0.5, kappa_star = 2.0; intensities scaled so that optical depths reach order one)."""
    w = None
    for frame in (0, 30, 60, 90, 119):
        w, res = run_fullsize(4, 16, n_random=1, camera=wl.orbit_camera(frame), w=w)
    w.fields["I"] = w.fields["I"] * 50.0
    for frame in (0, 30, 60, 90, 119):
        w, res = run_fullsize(4, 16, n_random=1, camera=wl.orbit_camera(frame), w=w, modes=(False,))
