"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA code).

Each test names the passage of PAPER.md it rests on.  None of them re-types the oracle's own
formula: the radiative-transfer tests integrate Eq. 1 through the 3-D Gaussians of Eq. 2 along
true pin-hole rays with an ODE solver; the others are invariants, reductions to library routines
or hand-worked scenarios.
"""
import json
import math
import os
from types import SimpleNamespace as NS

import numpy as np
import pytest
from scipy.integrate import solve_ivp

from oracle import splotch_oracle as so

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def species(n, **kw):
    d = dict(begin=0, end=n, brightness=1.0, absorb=1.0, use_colormap=False, fixed_rgb=(1.0, 1.0, 1.0),
             scalar_min=0.0, scalar_max=1.0, scalar_log10=False)
    d.update(kw)
    return NS(**d)


def camera(eye, lookat=(0, 0, 0), up=(0, 1, 0), fov=45.0):
    return NS(eye=eye, lookat=lookat, up=up, fov_deg=fov)


def fields(x, y, z, h, I=None, scalar=None):
    n = len(x)
    f = dict(x=x, y=y, z=z, h=h, I=np.ones(n) if I is None else I,
             scalar=np.zeros(n) if scalar is None else scalar)
    return {k: np.asarray(v, np.float32) for k, v in f.items()}


# ------------------------------------------------------------------------------------------------
# brute-force line of sight: integrate Eq. 1 with rho_p of Eq. 2 along the
# true ray of every pixel; a particle acts on a ray only if the ray passes within chi*sigma
# ------------------------------------------------------------------------------------------------
def _ray_dirs(cam, W, H):
    ex, lk, up = (np.asarray(v, float) for v in (cam.eye, cam.lookat, cam.up))
    f = (lk - ex) / np.linalg.norm(lk - ex)
    r = np.cross(f, up)
    r /= np.linalg.norm(r)
    u = np.cross(r, f)
    s = 0.5 * W / math.tan(math.radians(cam.fov_deg) / 2)
    dirs = np.zeros((H, W, 3))
    for j in range(H):
        for i in range(W):
            d = f + r * ((i + 0.5 - W / 2) / s) + u * (-(j + 0.5 - H / 2) / s)
            dirs[j, i] = d / np.linalg.norm(d)
    return ex, dirs


def _integrate_pixel(eye, d, pos, h, rho0, E, A, chi):
    """Solve dI/dr = sum_p (E_p - A_p I) rho_p(x(r)) from behind the farthest particle to the eye.

    r in Eq. 1 runs along the direction the radiation travels, i.e. towards the observer, so with t the
    distance from the eye we integrate from large t down to 0 (dI/dt = -rhs).
    """
    rel = pos - eye
    tc = rel @ d                                  # closest-approach parameter per particle
    b2 = np.sum(rel * rel, axis=1) - tc * tc      # squared impact parameter
    act = b2 <= (chi * h) ** 2
    if not act.any():
        return np.zeros(3)
    pos, h, rho0, E, A, tc = pos[act], h[act], rho0[act], E[act], A[act], tc[act]
    t_far, t_near = (tc + 7 * h).max(), max((tc - 7 * h).min(), 0.0)

    def rhs(t, I):
        x = eye + d * t
        rho = rho0 * np.exp(-np.sum((x - pos) ** 2, axis=1) / h ** 2)
        return -((E - A * I[None, :]) * rho[:, None]).sum(0)

    sol = solve_ivp(rhs, (t_far, t_near), np.zeros(3), rtol=1e-10, atol=1e-14, max_step=h.min() / 3)
    assert sol.success
    return sol.y[:, -1]


def test_additive_image_is_the_solution_of_eq1_with_E_equal_A():
    """Overlapping particles, E_p = A_p: oracle image with apply_transfer == ODE solution."""
    W = H = 12
    cam = camera((0.0, 0.0, 2.5), fov=0.5)
    s = 0.5 * W / math.tan(math.radians(0.25))               # ~1375 px per unit at z_c = 1
    px_unit = 2.5 / s                                        # world size of a pixel at the target plane
    rng = np.random.default_rng(7)
    n = 5
    pos = np.stack([rng.uniform(-3, 3, n) * px_unit, rng.uniform(-3, 3, n) * px_unit,
                    rng.uniform(-0.01, 0.01, n)], 1)
    h = rng.uniform(1.2, 2.5, n) * px_unit
    rho0 = rng.uniform(100.0, 300.0, n)
    rgb = rng.uniform(0.2, 1.0, (n, 3))
    f = fields(pos[:, 0], pos[:, 1], pos[:, 2], h, I=rho0)
    sps = [NS(begin=k, end=k + 1, brightness=1.5, absorb=1.0, use_colormap=False, fixed_rgb=tuple(rgb[k]),
              scalar_min=0.0, scalar_max=1.0, scalar_log10=False) for k in range(n)]
    img = so.render(f, sps, [None] * n, cam, W, H, chi=3.0, r_large=1e9, apply_transfer=True)
    eye, dirs = _ray_dirs(cam, W, H)
    E = 1.5 * np.asarray(rgb, np.float32).astype(float)
    p32 = np.stack([f["x"], f["y"], f["z"]], 1).astype(float)
    ref = np.zeros_like(img)
    for j in range(H):
        for i in range(W):
            ref[j, i] = _integrate_pixel(eye, dirs[j, i], p32, f["h"].astype(float), f["I"].astype(float), E, E, 3.0)
    assert ref.max() > 0.2                                    # optically thick enough that 1-exp(-S) != S
    assert np.abs(img - ref).max() <= 5e-4 * ref.max()
    # asymmetric scene: a transposed or mirrored image must not pass
    assert np.abs(img.transpose(1, 0, 2) - ref).max() > 0.05 * ref.max()
    assert np.abs(img[::-1] - ref).max() > 0.05 * ref.max()
    assert np.abs(img[:, ::-1] - ref).max() > 0.05 * ref.max()


def test_ordered_image_is_the_solution_of_eq1_for_separated_particles():
    """E != A, particles well separated along the ray: far-to-near composition == ODE."""
    W = H = 8
    cam = camera((0.0, 0.0, 2.5), fov=0.5)
    s = 0.5 * W / math.tan(math.radians(0.25))
    px_unit = 2.5 / s
    n = 4
    pos = np.array([[0.3, -0.2, 0.30], [-0.6, 0.4, 0.10], [0.2, 0.5, -0.10], [-0.1, -0.4, -0.30]])
    pos[:, :2] *= px_unit * 1.5
    h = np.array([1.5, 2.0, 1.8, 2.4]) * px_unit
    rho0 = np.array([150.0, 220.0, 120.0, 260.0])
    rgb = np.array([[1.0, 0.2, 0.1], [0.1, 0.9, 0.3], [0.2, 0.3, 1.0], [0.9, 0.8, 0.1]])
    kap = np.array([0.5, 2.0, 1.0, 3.0])
    f = fields(pos[:, 0], pos[:, 1], pos[:, 2], h, I=rho0)
    sps = [NS(begin=k, end=k + 1, brightness=1.0, absorb=float(kap[k]), use_colormap=False,
              fixed_rgb=tuple(rgb[k]), scalar_min=0.0, scalar_max=1.0, scalar_log10=False) for k in range(n)]
    img = so.render(f, sps, [None] * n, cam, W, H, chi=3.0, r_large=1e9, additive=False)
    eye, dirs = _ray_dirs(cam, W, H)
    p32 = np.stack([f["x"], f["y"], f["z"]], 1).astype(float)
    E = np.asarray(rgb, np.float32).astype(float)
    A = np.repeat(np.asarray(kap, np.float32).astype(float)[:, None], 3, 1)
    ref = np.zeros_like(img)
    for j in range(H):
        for i in range(W):
            ref[j, i] = _integrate_pixel(eye, dirs[j, i], p32, f["h"].astype(float), f["I"].astype(float), E, A, 3.0)
    assert np.abs(img - ref).max() <= 5e-4 * ref.max()
    # the order matters: visiting near-to-far instead gives a different picture
    cam16 = so.camera_constants(cam.eye, cam.lookat, cam.up, cam.fov_deg, W, H)
    g = so.geometry(f["x"], f["y"], f["z"], f["h"], cam16, 3.0, 0.5, 1e9, 1e-6, W, H, 16)
    Ea, col, kappa = so.amplitude(f["I"], f["scalar"], f["h"], sps, [None] * n)
    wrong = so.render_ordered(g, Ea, col, kappa, 3.0, W, H, order=so.depth_order(g)[::-1].copy())
    assert np.abs(wrong - ref).max() > 0.02 * ref.max()


def test_depth_order_is_far_to_near_with_index_ties():
    g = dict(cls=np.array([2, 0, 2, 1, 2, 2], np.int8), zc=np.array([1.0, 9.0, 3.0, 2.0, 3.0, 0.5], np.float32))
    assert so.depth_order(g).tolist() == [2, 4, 3, 0, 5]


def test_ordered_with_zero_absorption_equals_additive_sum():
    rng = np.random.default_rng(3)
    n, W, H = 300, 48, 40
    f = fields(rng.uniform(-0.5, 0.5, n), rng.uniform(-0.4, 0.4, n), rng.uniform(-0.3, 0.3, n),
               rng.uniform(0.002, 0.05, n), I=rng.uniform(0.5, 2, n), scalar=rng.uniform(0, 1, n))
    lut = np.asarray(rng.uniform(0, 1, (7, 3)), np.float32)
    sp = [species(n, use_colormap=True, absorb=0.0, brightness=0.7)]
    cam = camera((0.1, 0.2, 2.0))
    a = so.render(f, sp, [lut], cam, W, H, additive=True)
    o = so.render(f, sp, [lut], cam, W, H, additive=False)
    assert a.max() > 0
    np.testing.assert_allclose(o, a, rtol=1e-12, atol=1e-15 * a.max())


# ------------------------------------------------------------------------------------------------
# invariants of the additive mode
# ------------------------------------------------------------------------------------------------
def _random_scene(n, seed, hmin=0.004, hmax=0.03):
    rng = np.random.default_rng(seed)
    return fields(rng.uniform(-0.6, 0.6, n), rng.uniform(-0.6, 0.6, n), rng.uniform(-0.5, 0.5, n),
                  rng.uniform(hmin, hmax, n), I=rng.uniform(0.2, 3.0, n), scalar=rng.uniform(-0.2, 1.2, n))


def test_permutation_invariance_in_additive_mode():
    """'the solution of equation (1) does not depend on the particles integration order'."""
    n, W, H = 2000, 64, 64
    f = _random_scene(n, 11)
    lut = np.asarray(np.random.default_rng(1).uniform(0, 1, (16, 3)), np.float32)
    sp = [species(n, use_colormap=True)]
    cam = camera((0.0, 0.3, 2.2))
    a = so.render(f, sp, [lut], cam, W, H)
    perm = np.random.default_rng(2).permutation(n)
    b = so.render({k: v[perm] for k, v in f.items()}, sp, [lut], cam, W, H)
    assert a.max() > 0
    assert np.abs(a - b).max() <= 1e-12 * a.max()


def test_flux_conservation_for_on_screen_particles():
    """Sum over pixels == sum_p E col pi sp^2 (1 - exp(-chi^2)): the 2-D integral of the clipped Gaussian.

    Exact for SMALL particles; for point-sampled discs the lattice sum converges to the integral
    (relative error < 1e-4 once sigma >= 2 px)."""
    W = H = 200
    cam = camera((0.0, 0.0, 2.0), fov=40.0)
    s = 0.5 * W / math.tan(math.radians(20.0))
    rng = np.random.default_rng(5)
    n = 60
    sig_px = np.concatenate([rng.uniform(2.0, 6.0, n // 2), rng.uniform(0.01, 0.16, n // 2)])
    z = rng.uniform(-0.2, 0.2, n)
    k = s / (2.0 - z)
    f = fields(rng.uniform(-0.3, 0.3, n), rng.uniform(-0.3, 0.3, n), z, sig_px / k, I=rng.uniform(0.5, 2, n))
    sp = [species(n, fixed_rgb=(0.9, 0.5, 0.25), brightness=2.0)]
    img, g, _ = so.render(f, sp, [None], cam, W, H, return_geometry=True)
    assert set(np.unique(g["cls"])) == {so.SMALL, so.MEDIUM}
    assert (g["pbox"][:, 0] > 0).all() and (g["pbox"][:, 1] < W - 1).all()
    E = 2.0 * np.asarray([0.9, 0.5, 0.25], np.float32).astype(float)
    col = math.sqrt(math.pi) * f["h"].astype(float) * f["I"].astype(float)
    flux = (col * math.pi * g["sp"].astype(float) ** 2 * (1 - math.exp(-9.0))).sum()
    np.testing.assert_allclose(img.sum((0, 1)), E * flux, rtol=1e-4)
    only_small = g["cls"] == so.SMALL
    fs = {k_: v[only_small] for k_, v in f.items()}
    img_s = so.render(fs, [species(int(only_small.sum()), fixed_rgb=(0.9, 0.5, 0.25), brightness=2.0)], [None], cam, W, H)
    flux_s = (col[only_small] * math.pi * g["sp"][only_small].astype(float) ** 2 * (1 - math.exp(-9.0))).sum()
    np.testing.assert_allclose(img_s.sum((0, 1)), E * flux_s, rtol=1e-12)


def test_all_small_particles_reduce_to_a_weighted_histogram():
    """Small particles 'fall inside single pixels': the image is a 2-D histogram."""
    W, H = 96, 64
    rng = np.random.default_rng(9)
    n = 5000
    f = fields(rng.uniform(-0.8, 0.8, n), rng.uniform(-0.5, 0.5, n), rng.uniform(-0.1, 0.1, n),
               np.full(n, 1e-4), I=rng.uniform(0.5, 2.0, n))
    sp = [species(n)]
    cam = camera((0.0, 0.0, 2.0), fov=60.0)
    img, g, _ = so.render(f, sp, [None], cam, W, H, return_geometry=True)
    on = g["cls"] == so.SMALL
    assert on.sum() > 1000 and (g["cls"][~on] == so.CULLED).all()
    wgt = (math.sqrt(math.pi) * f["h"].astype(float) * f["I"].astype(float)
           * math.pi * g["sp"].astype(float) ** 2 * (1 - math.exp(-9.0)))
    hist, _, _ = np.histogram2d(g["py"][on].astype(float), g["px"][on].astype(float), bins=[H, W],
                                range=[[0, H], [0, W]], weights=wgt[on])
    for c in range(3):
        np.testing.assert_allclose(img[:, :, c], hist, rtol=1e-12, atol=1e-18)


def test_zero_outside_the_clip_disc():
    """'Any rays passing at distances larger than chi sigma_p are unaffected'."""
    W = H = 64
    cam = camera((0.0, 0.0, 2.0), fov=40.0)
    s = 0.5 * W / math.tan(math.radians(20.0))
    f = fields([0.013], [-0.021], [0.0], [4.0 * 2.0 / s])
    img, g, _ = so.render(f, [species(1)], [None], cam, W, H, return_geometry=True)
    jj, ii = np.mgrid[0:H, 0:W]
    d = np.hypot(ii + 0.5 - float(g["px"][0]), jj + 0.5 - float(g["py"][0]))
    r = 3.0 * float(g["sp"][0])
    assert (img[d > r + 1e-3] == 0).all()
    assert (img[d < r - 1e-3] > 0).all()
    # the profile is exp(-d^2/sigma^2) (no factor 2, Eq. 2): at d = sigma the value is 1/e of the peak
    peak = math.sqrt(math.pi) * float(f["h"][0])
    near = np.abs(d - float(g["sp"][0])).argmin()
    dn = d.flat[near]
    assert abs(img[:, :, 0].flat[near] / peak - math.exp(-dn ** 2 / float(g["sp"][0]) ** 2)) < 1e-12
    assert abs(math.log(img[:, :, 0].flat[near] / peak) + 1.0) < 0.2


# ------------------------------------------------------------------------------------------------
# classification, labels, tiles
# ------------------------------------------------------------------------------------------------
def test_fig2_five_particle_scenario():
    sc = json.load(open(os.path.join(GOLDEN, "fig2_scene.json")))
    names = {"C": so.CULLED, "S": so.SMALL, "M": so.MEDIUM, "L": so.LARGE}
    P = sc["particles"]
    for view in sc["views"]:
        cam = so.camera_constants(view["eye"], sc["lookat"], sc["up"], sc["fov_deg"], sc["width"], sc["height"])
        g = so.geometry(P["x"], P["y"], P["z"], P["h"], cam, sc["chi"], sc["r_small"], sc["r_large"], 1e-6,
                        sc["width"], sc["height"], sc["tile"])
        assert g["cls"].tolist() == [names[c] for c in view["classes"]]
        assert g["ilabel"].tolist() == view["ilabel"]
    # particle 2 in the second view: centre off-screen, still active
    assert g["px"][1] >= sc["width"] and g["pbox"][1, 0] <= sc["width"] - 1


def test_class_thresholds_are_inclusive_where_the_reading_says():
    """r = r_sml is Small (PAPER.md:158 '<='); r = r_0 is Medium (reading R7 of :159-160)."""
    W = H = 64                              # fov 90 -> s = 32; z_c = 32 -> k = 1 exactly
    cam = so.camera_constants((0, 0, 32), (0, 0, 0), (0, 1, 0), 90.0, W, H)
    h = np.array([0.1, 0.125, 0.25, 2.0, 2.5], np.float32)          # chi = 4 below: products are exact
    g = so.geometry(np.zeros(5), np.zeros(5), np.zeros(5), h, cam, 4.0, 0.5, 8.0, 1e-6, W, H, 16)
    assert g["rp"].tolist() == pytest.approx([4 * float(h[0]), 0.5, 1.0, 8.0, 10.0], abs=0)
    assert g["cls"].tolist() == [so.SMALL, so.SMALL, so.MEDIUM, so.MEDIUM, so.LARGE]


def test_behind_camera_nan_and_offscreen_are_culled():
    W = H = 32
    cam = so.camera_constants((0, 0, 2), (0, 0, 0), (0, 1, 0), 60.0, W, H)
    x = np.array([0, 0, np.nan, 50, 0, 0.0], np.float32)
    z = np.array([3.0, 2.0, 0, 0, 0, 0], np.float32)            # behind, in the eye plane, NaN, far off-screen
    h = np.array([0.1, 0.1, 0.1, 0.1, np.nan, -0.1], np.float32)
    g = so.geometry(x, np.zeros(6), z, h, cam, 3.0, 0.5, 64.0, 1e-6, W, H, 16)
    assert (g["cls"] == so.CULLED).all() and (g["ilabel"] == -2).all()


def test_resolution_scaling_doubles_the_radius():
    """r(p) is proportional to N_pix (Eq. 7): doubling W, H doubles sigma_px exactly."""
    f = _random_scene(500, 21)
    out = []
    for W in (128, 256):
        cam = so.camera_constants((0, 0.1, 2.2), (0, 0, 0), (0, 1, 0), 45.0, W, W)
        out.append(so.geometry(f["x"], f["y"], f["z"], f["h"], cam, 3.0, 0.5, 64.0, 1e-6, W, W, 16))
    a, b = out
    ok = a["zc"] > 1e-6
    # s doubles only up to its own float32 rounding, so allow 1 ulp
    np.testing.assert_allclose(b["sp"][ok], 2 * a["sp"][ok], rtol=2.4e-7)
    np.testing.assert_allclose(b["px"][ok] - 128.0, 2 * (a["px"][ok] - 64.0), rtol=1e-5, atol=1e-4)
    assert (b["cls"] >= a["cls"])[ok].all()                     # classes can only move up


def test_projection_maps_the_field_of_view_edge_to_the_image_edge():
    """A point seen at angle fov/2 to the right of the axis lands on x = W; one above lands on row < H/2."""
    W, H, fov = 200, 100, 50.0
    eye = np.array([0.3, -0.2, 3.0])
    cam = so.camera_constants(eye, (0.3, -0.2, 0.0), (0, 1, 0), fov, W, H)
    np.testing.assert_allclose(np.array(cam[0:3]), [1, 0, 0], atol=1e-7)     # looking down -z: right = +x
    np.testing.assert_allclose(np.array(cam[3:6]), [0, 1, 0], atol=1e-7)
    t = math.tan(math.radians(fov / 2))
    pts = np.array([[eye[0] + 2 * t, eye[1], 1.0], [eye[0], eye[1] + 0.5, 1.0], [eye[0], eye[1], 1.0]])
    g = so.geometry(pts[:, 0], pts[:, 1], pts[:, 2], np.full(3, 1e-3), cam, 3.0, 0.5, 64.0, 1e-6, W, H, 16)
    np.testing.assert_allclose(g["px"], [W, W / 2, W / 2], rtol=1e-5)
    assert g["py"][1] < H / 2 and abs(g["py"][2] - H / 2) < 1e-4


def test_camera_basis_is_orthonormal_and_right_handed():
    cam = so.camera_constants((1.0, 2.0, 3.0), (0.2, -0.1, 0.4), (0.1, 1.0, 0.2), 33.0, 640, 480).astype(float)
    r, u, f = cam[0:3], cam[3:6], cam[6:9]
    for a in (r, u, f):
        assert abs(np.linalg.norm(a) - 1) < 1e-6
    assert abs(r @ u) < 1e-6 and abs(r @ f) < 1e-6 and abs(u @ f) < 1e-6
    np.testing.assert_allclose(np.cross(r, f), u, atol=1e-6)
    assert u @ np.array([0.1, 1.0, 0.2]) > 0
    assert cam[12] == pytest.approx(320 / math.tan(math.radians(16.5)), rel=1e-6)
    with pytest.raises(ValueError):
        so.camera_constants((0, 0, 0), (0, 1, 0), (0, 2, 0), 45.0, 64, 64)          # up parallel to view
    with pytest.raises(ValueError):
        so.camera_constants((0, 0, 0), (0, 0, 0), (0, 1, 0), 45.0, 64, 64)          # eye == lookat


def test_tile_counts_match_a_brute_force_recount():
    W, H, T = 150, 100, 16                                        # ragged last tile column and row
    f = _random_scene(3000, 33, hmin=0.001, hmax=0.08)
    cam = so.camera_constants((0, 0, 2.0), (0, 0, 0), (0, 1, 0), 50.0, W, H)
    g = so.geometry(f["x"], f["y"], f["z"], f["h"], cam, 3.0, 0.5, 20.0, 1e-6, W, H, T)
    assert len(np.unique(g["cls"])) == 4
    ntx, nty = -(-W // T), -(-H // T)
    brute = np.zeros((nty, ntx), np.int64)
    for p in range(3000):
        if g["cls"][p] in (so.SMALL, so.MEDIUM):
            x0, x1, y0, y1 = g["pbox"][p]
            for ty in range(nty):
                for tx in range(ntx):
                    if x0 <= min(tx * T + T - 1, W - 1) and x1 >= tx * T and y0 <= min(ty * T + T - 1, H - 1) and y1 >= ty * T:
                        brute[ty, tx] += 1
    counts = so.tile_counts(g, W, H, T)
    assert (counts == brute).all()
    area = (g["tbox"][:, 1] - g["tbox"][:, 0] + 1) * (g["tbox"][:, 3] - g["tbox"][:, 2] + 1)
    assert counts.sum() == area[(g["cls"] == so.SMALL) | (g["cls"] == so.MEDIUM)].sum()
    # every pixel the float32 predicate accepts lies inside the pixel box
    for p in np.flatnonzero(g["cls"] >= so.MEDIUM)[:200]:
        jj, ii = np.mgrid[0:H, 0:W]
        dx = (ii.astype(np.float32) + np.float32(0.5)) - g["px"][p]
        dy = (jj.astype(np.float32) + np.float32(0.5)) - g["py"][p]
        inside = dx * dx + dy * dy <= g["rp"][p] * g["rp"][p] * np.float32(0.999)
        x0, x1, y0, y1 = g["pbox"][p]
        assert (ii[inside] >= x0).all() and (ii[inside] <= x1).all()
        assert (jj[inside] >= y0).all() and (jj[inside] <= y1).all()


# ------------------------------------------------------------------------------------------------
# colour look-up table (PAPER.md:85 'look-up tables (or palettes)'; :76, :166 normalisation / log)
# ------------------------------------------------------------------------------------------------
def test_colour_map_entries_clamp_and_linear_ramp():
    K = 5
    lut = np.asarray(np.random.default_rng(4).uniform(0, 1, (K, 3)), np.float32)
    sc = np.array([10.0 + 5.0 * k for k in range(K)] + [0.0, 99.0, 12.5], np.float32)
    n = sc.shape[0]
    sp = [species(n, use_colormap=True, scalar_min=10.0, scalar_max=30.0, brightness=1.0)]
    E, col, _ = so.amplitude(np.ones(n), sc, np.ones(n), sp, [lut])
    np.testing.assert_allclose(E[:K], lut.astype(float), rtol=1e-15)
    np.testing.assert_allclose(E[K], lut[0].astype(float))
    np.testing.assert_allclose(E[K + 1], lut[-1].astype(float))
    np.testing.assert_allclose(E[K + 2], 0.5 * (lut[0].astype(float) + lut[1].astype(float)), rtol=1e-12)
    assert col == pytest.approx(math.sqrt(math.pi))
    # two entries = a plain linear ramp; log10 normalisation
    ramp = np.array([[0, 0, 0], [1, 2, 4]], np.float32)
    sp2 = [species(3, use_colormap=True, scalar_min=-1.0, scalar_max=1.0, scalar_log10=True, brightness=0.5)]
    E2, _, _ = so.amplitude(np.ones(3), np.array([0.1, 1.0, 10.0], np.float32), np.ones(3), sp2, [ramp])
    np.testing.assert_allclose(E2, 0.5 * np.outer([0.0, 0.5, 1.0], [1, 2, 4]), atol=1e-7)


def test_two_species_use_their_own_parameters():
    n = 6
    lut = np.array([[0, 0, 1], [1, 0, 0]], np.float32)
    sps = [NS(begin=0, end=4, brightness=2.0, absorb=0.5, use_colormap=True, fixed_rgb=(0, 0, 0),
              scalar_min=0.0, scalar_max=1.0, scalar_log10=False),
           NS(begin=4, end=6, brightness=0.25, absorb=3.0, use_colormap=False, fixed_rgb=(1.0, 0.5, 0.25),
              scalar_min=0.0, scalar_max=1.0, scalar_log10=False)]
    E, col, kappa = so.amplitude(np.full(n, 2.0), np.full(n, 0.25), np.full(n, 0.5), sps, [lut, None])
    np.testing.assert_allclose(E[:4], np.tile([0.5, 0.0, 1.5], (4, 1)))
    np.testing.assert_allclose(E[4:], np.tile([0.25, 0.125, 0.0625], (2, 1)))
    np.testing.assert_allclose(col, math.sqrt(math.pi))
    assert kappa.tolist() == [0.5] * 4 + [3.0] * 2


# ------------------------------------------------------------------------------------------------
# closed-form single-Gaussian image: every pixel, to double rounding
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("X,Y,h,chi", [(0.0, 0.0, 2.0, 3.0), (3.25, -2.5, 2.5, 3.0), (-7.75, 5.125, 1.5, 2.0),
                                       (29.5, -30.0, 3.0, 3.0)])
def test_single_gaussian_image_closed_form_every_pixel(X, Y, h, chi):
    """One particle, E = A: S(i, j) = b colour I sqrt(pi) h exp(-d^2 / sp^2) inside the clip disc d <= chi sp, 0 outside.

    fov 90 degrees, W = 64, eye 32 units from the particle's plane: s = 32 and k = s / z_c = 1 exactly, so the screen
    centre (32 + X, 32 - Y) and sp = h are exact in float32 and the expected image below is exact up to double rounding.
    The last case sits in the image corner (clipped box, off-axis in both directions)."""
    W = H = 64
    cam = camera((0.0, 0.0, 32.0), fov=90.0)
    I0, b = 1.75, 0.6
    rgb = (0.9, 0.5, 0.125)
    f = fields([X], [Y], [0.0], [h], I=[I0])
    sp = [species(1, fixed_rgb=rgb, brightness=b)]
    img, g, cam16 = so.render(f, sp, [None], cam, W, H, chi=chi, r_large=1e9, return_geometry=True)
    assert float(cam16[12]) == 32.0 and float(g["px"][0]) == 32.0 + X and float(g["py"][0]) == 32.0 - Y
    assert float(g["sp"][0]) == h
    jj, ii = np.mgrid[0:H, 0:W]
    d2 = (ii + 0.5 - (32.0 + X)) ** 2 + (jj + 0.5 - (32.0 - Y)) ** 2
    peak = float(np.float32(b)) * float(np.float32(I0)) * math.sqrt(math.pi) * h
    expect = np.where(d2 <= (chi * h) ** 2, peak * np.exp(-d2 / h ** 2), 0.0)
    assert (expect > 0).sum() > 20
    for c in range(3):
        np.testing.assert_allclose(img[:, :, c], float(np.float32(rgb[c])) * expect, rtol=1e-14, atol=0.0)
    # exact transfer of the E = A solution
    img_t = so.render(f, sp, [None], cam, W, H, chi=chi, r_large=1e9, apply_transfer=True)
    np.testing.assert_allclose(img_t[:, :, 0], -np.expm1(-float(np.float32(rgb[0])) * expect), rtol=1e-14, atol=0.0)


def test_pixel_box_is_the_tight_bounding_box_of_the_clip_disc():
    """C1: x0 = ceil((p_x - r) - 0.5), x1 = floor((p_x + r) - 0.5) clamped to the screen -- brute force over every
    column and row: column i belongs to the box iff |i + 0.5 - p_x| <= r (the disc reaches that column's centre line),
    rows likewise.  A box one pixel too wide or too narrow on any side fails.  Particles whose disc edge lies within
    1e-4 px of a column / row centre line are the documented float32 edge case and are skipped (they must be rare)."""
    W, H = 150, 100
    f = _random_scene(4000, 77, hmin=0.001, hmax=0.08)
    cam = so.camera_constants((0, 0, 2.0), (0, 0, 0), (0, 1, 0), 50.0, W, H)
    g = so.geometry(f["x"], f["y"], f["z"], f["h"], cam, 3.0, 0.5, 20.0, 1e-6, W, H, 16)
    big = np.flatnonzero(g["cls"] >= so.MEDIUM)
    assert big.size > 1500
    cols, rows = np.arange(W) + 0.5, np.arange(H) + 0.5
    skipped = 0
    for p in big:
        px, py, r = float(g["px"][p]), float(g["py"][p]), float(g["rp"][p])
        ex, ey = np.abs(cols - px) - r, np.abs(rows - py) - r
        if np.abs(ex).min() < 1e-4 or np.abs(ey).min() < 1e-4:
            skipped += 1
            continue
        ci, rj = np.flatnonzero(ex <= 0), np.flatnonzero(ey <= 0)
        assert ci.size and rj.size                       # active: the box is not empty
        assert g["pbox"][p].tolist() == [ci[0], ci[-1], rj[0], rj[-1]], p
    assert skipped < 0.01 * big.size
    # inactive although r > r_small: no column or no row centre line is reached on screen
    off = np.flatnonzero((g["cls"] == so.CULLED) & (g["rp"] > 0.5) & (g["zc"] > 1e-6))
    assert off.size > 10
    for p in off:
        px, py, r = float(g["px"][p]), float(g["py"][p]), float(g["rp"][p])
        ex, ey = np.abs(cols - px) - r, np.abs(rows - py) - r
        if np.abs(ex).min() < 1e-4 or np.abs(ey).min() < 1e-4:
            continue
        assert not ((ex <= 0).any() and (ey <= 0).any()), p


# ------------------------------------------------------------------------------------------------
# pre-processing: normalisation range found from the data (PAPER.md:76, :166 fn. 1), vector colours (:85)
# ------------------------------------------------------------------------------------------------
def test_scalar_range_is_the_min_max_of_the_finite_values_per_species():
    rng = np.random.default_rng(12)
    n = 5000
    sc = rng.lognormal(0.0, 2.0, n).astype(np.float32)
    sc[::97] = np.nan
    sc[5::301] = np.inf
    sc[7::211] = -1.0                                            # log10 of a negative number: skipped in the log species
    sc[11::503] = 0.0                                            # log10(0) = -inf: skipped
    sps = [species(3000, use_colormap=True, scalar_log10=True), species(0, use_colormap=True)]
    sps[1].begin, sps[1].end = 3000, n
    got = so.scalar_range(sc, sps)
    a = np.log10(sc[:3000].astype(np.float64), where=sc[:3000] > 0, out=np.full(3000, np.nan)).astype(np.float32)
    a = a[np.isfinite(a)]
    b = sc[3000:][np.isfinite(sc[3000:])]
    assert got[0] == (float(a.min()), float(a.max()))
    assert got[1] == (float(b.min()), float(b.max())) and got[1][0] == -1.0
    # a species without a finite value: (0, 1)
    assert so.scalar_range(np.full(4, np.nan, np.float32), [species(4, use_colormap=True)]) == [(0.0, 1.0)]


def test_automatic_range_equals_the_same_frame_with_the_range_given():
    n, W, H = 1500, 64, 48
    f = _random_scene(n, 31)
    lut = np.asarray(np.random.default_rng(2).uniform(0, 1, (9, 3)), np.float32)
    auto = [species(n, use_colormap=True, auto_range=True, scalar_min=123.0, scalar_max=124.0)]     # given values are ignored
    lo, hi = float(f["scalar"].min()), float(f["scalar"].max())
    given = [species(n, use_colormap=True, scalar_min=lo, scalar_max=hi)]
    cam = camera((0.0, 0.2, 2.1))
    a = so.render(f, auto, [lut], cam, W, H)
    b = so.render(f, given, [lut], cam, W, H)
    assert a.max() > 0 and np.array_equal(a, b)
    # the extreme particles get the first and the last table entry exactly
    E, _, _ = so.amplitude(f["I"], f["scalar"], f["h"], so.resolve_ranges(f, auto), [lut])
    np.testing.assert_allclose(E[f["scalar"].argmin()], lut[0].astype(float), rtol=0, atol=0)
    np.testing.assert_allclose(E[f["scalar"].argmax()], lut[-1].astype(float), rtol=1e-15)


def test_vector_colour_mode_maps_components_to_channels():
    """rho^R = v_x, rho^G = v_y, rho^B = v_z, each normalised over the species' range and clamped."""
    vr = np.array([-2.0, 2.0, 0.0, 5.0, np.nan], np.float32)
    vg = np.array([2.0, -2.0, 1.0, -9.0, 0.0], np.float32)
    vb = np.array([0.0, 0.0, -1.0, 2.0, 0.0], np.float32)
    n = 5
    sp = [species(n, vector_colour=True, scalar_min=-2.0, scalar_max=2.0, brightness=0.5)]
    E, col, _ = so.amplitude(np.ones(n), np.zeros(n), np.ones(n), sp, [None], vec=(vr, vg, vb))
    np.testing.assert_allclose(E, 0.5 * np.array([[0, 1, 0.5], [1, 0, 0.5], [0.5, 0.75, 0.25], [1, 0, 1], [0, 0.5, 0.5]]), atol=1e-15)
    # the image of a vector-coloured set is the stack of three single-channel images: channel c sees only component c
    rng = np.random.default_rng(8)
    m, W, H = 800, 48, 40
    f = _random_scene(m, 41)
    f["cr"], f["cg"], f["cb"] = (rng.uniform(-1, 1, m).astype(np.float32) for _ in range(3))
    spv = [species(m, vector_colour=True, scalar_min=-1.0, scalar_max=1.0)]
    cam = camera((0.1, 0.0, 2.0))
    img = so.render(f, spv, [None], cam, W, H)
    for c, key in enumerate(("cr", "cg", "cb")):
        ramp = np.array([[0, 0, 0], [1, 1, 1]], np.float32)               # K = 2 table: colour = t, all channels
        f1 = dict(f, scalar=f[key])
        one = so.render(f1, [species(m, use_colormap=True, scalar_min=-1.0, scalar_max=1.0)], [ramp], cam, W, H)
        np.testing.assert_allclose(img[:, :, c], one[:, :, c], rtol=1e-13, atol=1e-300)
    # automatic range of a vector species: over the three components together
    spa = so.resolve_ranges(f, [species(m, vector_colour=True, auto_range=True)])
    allv = np.concatenate([f["cr"], f["cg"], f["cb"]])
    assert (spa[0].scalar_min, spa[0].scalar_max) == (float(allv.min()), float(allv.max()))
