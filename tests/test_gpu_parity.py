"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Acceptance (BASELINE.json north_star): image relative L2 error <= 1e-5 and max per-pixel absolute error
<= 1e-4 * image max, in float32; class labels, pixel / tile boxes, the paper's tile index i(p), the float32
screen geometry and per-tile pair counts bit-exact.
"""
import numpy as np
import pytest
import torch

from oracle import splotch_oracle as so
from paper_1309_1114_b200 import workloads as wl

pytestmark = pytest.mark.gpu

REL_L2 = 1e-5
MAX_ABS = 1e-4


def _binding():
    from paper_1309_1114_b200 import binding
    return binding


def to_dev(fields):
    return {k: v.cuda().contiguous() for k, v in fields.items()}


def to_np(fields):
    return {k: v.cpu().numpy() for k, v in fields.items()}


def luts_for(species, lut):
    return [lut if s.use_colormap else None for s in species]


def oracle_frame(w, lut, tile, window=None):
    return so.render(to_np(w.fields), w.species, luts_for(w.species, lut.numpy()), w.camera, w.width, w.height,
                     chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=tile,
                     additive=w.additive, apply_transfer=w.apply_transfer, window=window, return_geometry=True)


def gpu_frame(w, lut, tile, fields_dev=None, pair_capacity=0):
    b = _binding()
    r = b.Renderer(w.width, w.height, max(w.n, 1))
    r.set_camera(w.camera)
    for s, sp in enumerate(w.species):
        if sp.use_colormap:
            r.set_colormap(s, lut)
    f = fields_dev if fields_dev is not None else to_dev(w.fields)
    kw = dict(chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=tile, additive=w.additive,
              apply_transfer=w.apply_transfer)
    img = r.render(f, w.species, pair_capacity=pair_capacity, **kw)
    torch.cuda.synchronize()
    return r, f, kw, img


def assert_image_close(gpu_img, ref, what=""):
    g = gpu_img.double().cpu().numpy()
    assert np.isfinite(g).all(), what
    mx = ref.max()
    if mx == 0:
        assert (g == 0).all(), what
        return
    rel = np.linalg.norm(g - ref) / np.linalg.norm(ref)
    mab = np.abs(g - ref).max() / mx
    assert rel <= REL_L2, f"{what}: relative L2 {rel:.3e}"
    assert mab <= MAX_ABS, f"{what}: max abs / max {mab:.3e}"


def assert_geometry_exact(r, f, w, kw, g, cam):
    assert np.array_equal(np.asarray(r.camera_constants(), np.float32), cam)
    d = r.debug_geometry(f, w.species, **kw)
    torch.cuda.synchronize()
    for k in ("cls", "pbox", "tbox", "ilabel"):
        assert np.array_equal(d[k].cpu().numpy(), g[k]), k
    for k in ("px", "py", "sp", "rp", "zc"):          # bit-exact float32
        a, b_ = d[k].cpu().numpy(), g[k]
        act = g["cls"] != so.CULLED if k != "zc" else ~np.isnan(g[k])        # NaN payload bits are not compared
        assert np.array_equal(a[act].view(np.uint32), b_[act].view(np.uint32)), k
        assert np.array_equal(np.isnan(a), np.isnan(b_)) or k != "zc"


def assert_counts_exact(r, w, tile, g):
    st = r.stats()
    assert st["overflow"] == 0
    assert st["count"] == [int((g["cls"] == c).sum()) for c in range(4)]
    oc = so.tile_counts(g, w.width, w.height, tile, count_large=not w.additive)   # ordered mode bins LARGE to tiles too
    gc = r.debug_tile_counts(tile).cpu().numpy()
    assert np.array_equal(gc.astype(np.int64), oc.astype(np.int64))
    assert st["pairs"] == int(oc.sum())
    return st


def full_check(w, tile, lut=None, pair_capacity=0):
    lut = wl.palette() if lut is None else lut
    ref, g, cam = oracle_frame(w, lut, tile)
    r, f, kw, img = gpu_frame(w, lut, tile, pair_capacity=pair_capacity)
    assert_geometry_exact(r, f, w, kw, g, cam)
    st = assert_counts_exact(r, w, tile, g)
    assert_image_close(img, ref, w.name)
    r.close()
    return st, g


@pytest.mark.parametrize("tile", [8, 16, 32])
def test_cfg0_full(tile):
    w = wl.make_config(0)
    st, g = full_check(w, tile)
    assert st["count"][wl_MEDIUM] > 90_000


wl_SMALL, wl_MEDIUM, wl_LARGE = 1, 2, 3


def test_cfg1_reduced_ragged_tiles():
    w = wl.make_config(1, n=1_000_000, size=(800, 600))         # 600 / 16 = 37.5: ragged last tile row
    st, g = full_check(w, 16)
    assert st["count"][wl_SMALL] > 100_000 and st["count"][wl_MEDIUM] > 100_000


def test_cfg2_reduced_two_species():
    w = wl.make_config(2, n=600_000, eta=0.04)                  # 1920 x 1080, 1080 / 16 = 67.5; eta keeps the S/M mix
    st, g = full_check(w, 16)
    assert st["count"][wl_SMALL] > 0 and st["count"][wl_MEDIUM] > 0


@pytest.mark.parametrize("tile,r_large", [(16, 12.0), (32, 24.0), (16, 64.0), (32, 64.0), (32, 200.0)])
def test_cfg3_reduced_large_particles(tile, r_large):
    """(32, 64) and (32, 200): with 32-px tiles the MEDIUM discs wider than 32 px sit in the third bin of their tiles and are rendered
    by k_large (whole image against the oracle, per-tile counts bit-exact as everywhere)."""
    w = wl.make_config(3, n=150_000, size=(512, 384))
    w.r_large = r_large
    st, g = full_check(w, tile)
    assert st["count"][wl_LARGE] > (1000 if r_large < 100 else 0)
    assert st["large_pairs"] >= st["count"][wl_LARGE]
    if tile == 32 and r_large > 32.0:
        wide = int(((g["cls"] == wl_MEDIUM) & (g["rp"] > 32.0)).sum())
        assert wide > 1000, wide


def test_large_particles_with_8px_tiles_and_a_disc_covering_the_image():
    """k_large with one pixel per thread (T = 8) and a particle whose disc contains every tile of the image."""
    w = wl.make_config(3, n=40_000, size=(200, 136))
    w.r_large = 6.0
    w.fields["h"][:3] = 5.0                                      # three discs far larger than the image
    w.fields["x"][:3] = 0.5; w.fields["y"][:3] = 0.5; w.fields["z"][:3] = 0.5
    st, g = full_check(w, 8)
    assert st["count"][wl_LARGE] > 1000


def test_many_discs_that_contain_whole_blocks_go_through_the_tensor_cores_within_tolerance():
    """k_large's tensor-core bands: 60,000 discs of 120 .. 600 px that contain most 32-px blocks of a 160 x 128 image, so every pixel
    sums tens of thousands of products of split TF32 operands in tensor memory (accumulators of 64 records folded into float32
    second-level sums); the amplitudes span four decades and the colours differ per particle.  Same tolerance."""
    w = wl.make_config(3, n=60_000, size=(160, 128))
    w.r_large = 16.0
    g = torch.Generator().manual_seed(5)
    w.fields["x"] = 0.5 + 0.02 * (torch.rand(w.n, generator=g) - 0.5)
    w.fields["y"] = 0.5 + 0.02 * (torch.rand(w.n, generator=g) - 0.5)
    w.fields["z"] = 0.5 + 0.02 * (torch.rand(w.n, generator=g) - 0.5)
    w.fields["h"] = 0.3 + 1.2 * torch.rand(w.n, generator=g)
    w.fields["I"] = torch.exp(9.2 * torch.rand(w.n, generator=g) - 4.6)
    for tile in (16, 32):
        st, geo = full_check(w, tile)
        assert st["count"][wl_LARGE] > 50_000


def test_apply_transfer():
    w = wl.make_config(0, n=30_000)
    w.apply_transfer = True
    w.fields["I"] = w.fields["I"] * 40.0                        # make 1 - exp(-S) differ visibly from S
    full_check(w, 16)


@pytest.mark.parametrize("n", [0, 1, 3, 5, 33, 1027])
def test_tiny_and_ragged_particle_counts(n):
    w = wl.make_config(0, n=max(n, 1), size=(64, 48))
    if n == 0:
        w.fields = {k: v[:0] for k, v in w.fields.items()}
        w.n = 0
        w.species[0].end = 0
    full_check(w, 16)


def test_unaligned_field_pointers_take_the_scalar_path():
    w = wl.make_config(0, n=20_001, size=(128, 128))
    lut = wl.palette()
    base = {k: torch.cat([torch.zeros(1), v]).cuda() for k, v in w.fields.items()}
    f = {k: v[1:] for k, v in base.items()}                     # 4-byte offset: not 16-byte aligned
    assert f["x"].data_ptr() % 16 != 0
    ref, g, cam = oracle_frame(w, lut, 16)
    r, f, kw, img = gpu_frame(w, lut, 16, fields_dev=f)
    assert_counts_exact(r, w, 16, g)
    assert_image_close(img, ref)


def test_degenerate_inputs_nan_inf_behind_camera():
    w = wl.make_config(0, n=4096, size=(96, 96))
    x = w.fields["x"]
    x[::7] = float("nan")
    w.fields["h"][1::11] = float("inf")
    w.fields["h"][2::13] = -1.0
    w.fields["z"][3::5] = 9.0                                   # behind the camera (eye at z = 2.5 looking at -z)
    w.fields["h"][4::17] = 0.0
    st, g = full_check(w, 16)
    assert st["count"][0] > 1000


def test_all_culled_gives_a_zero_image():
    w = wl.make_config(0, n=5000, size=(64, 64))
    w.fields["z"] = w.fields["z"] + 100.0
    st, g = full_check(w, 16)
    assert st["count"][0] == 5000 and st["pairs"] == 0


def test_single_heavy_pixel_and_heavy_tile():
    """Many particles on one pixel / one tile: long same-pixel chains and several chunks of one tile."""
    n = 60_000
    w = wl.make_config(0, n=n, size=(64, 64))
    w.fields["x"] = 0.5 + 1e-4 * (w.fields["x"] - 0.5)
    w.fields["y"] = 0.5 + 1e-4 * (w.fields["y"] - 0.5)
    w.fields["h"][: n // 2] = 1e-5                               # half SMALL on ~one pixel, half MEDIUM
    st, g = full_check(w, 16)
    assert st["chunks"] >= 4


def test_pair_overflow_is_reported_and_image_is_zero():
    w = wl.make_config(0, n=50_000, size=(128, 128))
    lut = wl.palette()
    r, f, kw, img = gpu_frame(w, lut, 16, pair_capacity=1000)
    st = r.stats()
    assert st["overflow"] == 1 and st["pairs"] > 1000
    assert float(img.abs().max()) == 0.0
    # a larger workspace on the same context renders the frame
    img2 = r.render(f, w.species, pair_capacity=200_000, **kw)
    assert r.stats()["overflow"] == 0 and float(img2.max()) > 0


def test_render_host_matches_device_render():
    w = wl.make_config(0, n=40_000, size=(160, 120))
    lut = wl.palette()
    r, f, kw, img = gpu_frame(w, lut, 16)
    host = {k: v.contiguous().pin_memory() for k, v in w.fields.items()}
    out = torch.empty((w.height, w.width, 3), dtype=torch.float32).pin_memory()
    r.render_host(host, w.species, out, **kw)
    ref, g, cam = oracle_frame(w, lut, 16)
    assert_image_close(out, ref)
    assert_image_close(img, ref)


def test_errors_are_reported_not_raised_from_c():
    b = _binding()
    r = b.Renderer(64, 64, 1000)
    w = wl.make_config(0, n=100, size=(64, 64))
    f = to_dev(w.fields)
    with pytest.raises(b.SplotchError) as e:
        r.render(f, w.species)                                   # camera not set
    assert e.value.code == b.SPLOTCH_ESTATE
    r.set_camera(w.camera)
    with pytest.raises(b.SplotchError) as e:
        r.render(f, w.species)                                   # colour map not set
    assert e.value.code == b.SPLOTCH_ESTATE
    r.set_colormap(0, wl.palette())
    with pytest.raises(b.SplotchError) as e:
        r.render(f, w.species, tile=12)
    assert e.value.code == b.SPLOTCH_EINVAL
    with pytest.raises(b.SplotchError):
        r.set_camera(wl.Camera((0, 0, 0), (0, 0, 0), (0, 1, 0), 45.0))
    with pytest.raises(b.SplotchError):
        r.set_camera(wl.Camera((0, 0, 1), (0, 0, 0), (0, 0, 2), 45.0))
    big = wl.make_config(0, n=2000, size=(64, 64))
    with pytest.raises(b.SplotchError):
        r.render(to_dev(big.fields), big.species)                # n > max_particles
    r.render(f, w.species)


def test_permutation_invariance_on_gpu():
    w = wl.make_config(0, n=50_000, size=(128, 128))
    lut = wl.palette()
    r, f, kw, img = gpu_frame(w, lut, 16)
    perm = torch.randperm(w.n, generator=torch.Generator().manual_seed(1)).cuda()
    f2 = {k: v[perm].contiguous() for k, v in f.items()}
    img2 = r.render(f2, w.species, **kw).clone()
    torch.cuda.synchronize()
    a, b_ = img.double().cpu().numpy(), img2.double().cpu().numpy()
    assert np.linalg.norm(a - b_) <= 2e-6 * np.linalg.norm(a)


def test_two_renders_of_one_frame_agree():
    """The integer work is bit-reproducible (classes, per-tile counts; SMALL and small-box contributions are exact
    fixed-point sums).  The pixel owners add float32 contributions in the order the records sit in their bins, which
    depends on the scheduling of the scatter stage: two renders agree to float32 rounding, not bit for bit."""
    w = wl.make_config(1, n=500_000, size=(400, 300))
    lut = wl.palette()
    r, f, kw, img = gpu_frame(w, lut, 16)
    a = img.clone()
    c0 = r.debug_tile_counts(16).clone()
    st0 = r.stats()
    b_ = r.render(f, w.species, **kw)
    torch.cuda.synchronize()
    assert torch.equal(c0, r.debug_tile_counts(16)) and st0["count"] == r.stats()["count"] and st0["pairs"] == r.stats()["pairs"]
    d = (a.double() - b_.double())
    assert float(d.norm()) <= 1e-6 * float(a.double().norm())
    assert float(d.abs().max()) <= 1e-6 * float(a.max())


def test_all_small_frame_is_bit_reproducible():
    """Only SMALL particles: every contribution is an integer addition, the image does not depend on the order."""
    w = wl.make_config(1, n=300_000, size=(200, 150))
    w.fields["h"] = torch.full_like(w.fields["h"], 1e-5)
    lut = wl.palette()
    r, f, kw, img = gpu_frame(w, lut, 16)
    a = img.clone()
    assert r.stats()["count"][2] == 0 and r.stats()["count"][1] > 100_000
    perm = torch.randperm(w.n, generator=torch.Generator().manual_seed(9)).cuda()
    b_ = r.render({k: v[perm].contiguous() for k, v in f.items()}, w.species, **kw)
    torch.cuda.synchronize()
    assert torch.equal(a, b_)


def test_amplitudes_spanning_ten_decades_document_the_fixed_point_limit():
    """The tiles' sums are fixed point in units of 2^-30 of the frame's largest record amplitude:
    the image meets the north_star tolerance (which is relative to the image's maximum), while contributions more than
    about nine decades below the brightest record fall under one unit and vanish; the double-precision oracle keeps them."""
    n = 40_000
    w = wl.make_config(0, n=n, size=(128, 128))
    w.fields["h"] = torch.full_like(w.fields["h"], 1e-5)                     # all SMALL: one contribution per particle
    I = torch.full((n,), 1e-10)
    I[: n // 2] = 1.0                                                         # bright half, faint half ten decades below
    w.fields["I"] = I.to(torch.float32)
    xs = w.fields["x"].clone()
    w.fields["x"] = torch.where(torch.arange(n) < n // 2, 0.35 + 0.2 * (xs - 0.5), 0.65 + 0.2 * (xs - 0.5))   # left / right
    lut = wl.palette()
    ref, g, cam = oracle_frame(w, lut, 16)
    r, f, kw, img = gpu_frame(w, lut, 16)
    assert_image_close(img, ref, "ten decades")
    gi = img.double().cpu().numpy()
    faint = (ref > 0) & (ref < 1e-8 * ref.max())
    assert faint.sum() > 100
    assert (gi[faint] == 0).all()                                             # below one fixed-point unit: lost
    # seven decades are still resolved to a few per cent
    I2 = I.clone(); I2[n // 2:] = 1e-7
    w.fields["I"] = I2.to(torch.float32)
    ref2, g2, cam2 = oracle_frame(w, lut, 16)
    r2, f2, kw2, img2 = gpu_frame(w, lut, 16)
    gi2 = img2.double().cpu().numpy()
    faint2 = (ref2 > 0) & (ref2 < 1e-5 * ref2.max())
    assert faint2.sum() > 100
    assert np.abs(gi2[faint2] - ref2[faint2]).max() <= 0.05 * ref2[faint2].max()


def test_tile_64_and_global_histogram_paths():
    """tile = 64 (pixel owners hold 8 pixels per lane) and an image with more bins than fit in shared memory
    (2048 x 1536 at 8 px: 98,304 + 768 bins -> the blocks count into their rows of the count matrix in L2)."""
    w = wl.make_config(1, n=200_000, size=(400, 300))
    full_check(w, 64)
    w3 = wl.make_config(3, n=120_000, size=(512, 384))
    w3.r_large = 24.0
    full_check(w3, 64)
    wg = wl.make_config(1, n=300_000, size=(2048, 1536))
    st, g = full_check(wg, 8, pair_capacity=40_000_000)          # a 60-px disc covers 15 x 15 tiles of 8 px
    assert st["count"][wl_MEDIUM] > 50_000


def test_requested_pair_capacity_is_honoured():
    b = _binding()
    for additive in (True, False):
        w = wl.make_config(0, n=20_000, size=(1024, 1024))
        w.additive = additive
        lut = wl.palette()
        r, f, kw, img = gpu_frame(w, lut, 16, pair_capacity=30_000)
        assert r.stats()["pair_capacity"] >= 30_000
        r.close()


def test_cfg1_full_size_bench_configuration():
    """BASELINE configs[1] at full size (10M particles, 800 x 800), the launch configuration bench.py times."""
    w = wl.make_config(1, device="cuda")
    lut = wl.palette()
    fdev = {k: v.contiguous() for k, v in w.fields.items()}
    w.fields = {k: v.cpu() for k, v in fdev.items()}
    ref, g, cam = oracle_frame(w, lut, 16)
    r, f, kw, img = gpu_frame(w, lut, 16, fields_dev=fdev)
    assert_geometry_exact(r, f, w, kw, g, cam)
    assert_counts_exact(r, w, 16, g)
    assert_image_close(img, ref, "cfg1 full")


# ---- ordered (E != A) mode: step A7, reading R15 of DESIGN.md ---------------------------------------------------------
def ordered(w, absorb=None):
    w.additive = False
    if absorb is not None:
        for sp, k in zip(w.species, absorb):
            sp.absorb = k
    return w


@pytest.mark.parametrize("tile", [8, 16, 32])
def test_ordered_cfg0(tile):
    w = ordered(wl.make_config(0, n=60_000, size=(160, 128)), absorb=[3.0])
    w.fields["I"] = w.fields["I"] * 30.0                        # optical depths of order one: the order matters
    full_check(w, tile)


def test_ordered_cfg4_reduced_two_species():
    w = ordered(wl.make_config(4, n=600_000, eta=0.04))         # kappa_gas = 0.5, kappa_star = 2.0 (workloads.py)
    w.fields["I"] = w.fields["I"] * 200.0
    st, g = full_check(w, 16)
    assert st["count"][wl_SMALL] > 0 and st["count"][wl_MEDIUM] > 0


def test_ordered_orbit_frame_and_large_particles():
    w = ordered(wl.make_config(3, n=60_000, size=(256, 192)), absorb=[1.5])
    w.r_large = 12.0
    w.fields["I"] = w.fields["I"] * 3.0
    st, g = full_check(w, 16)
    assert st["count"][wl_LARGE] > 500


def test_ordered_depth_ties_resolve_by_index():
    """Many particles at exactly the same depth on the same pixels: the visiting order is the particle index."""
    n = 20_000
    w = ordered(wl.make_config(0, n=n, size=(64, 64)), absorb=[2.0])
    w.fields["x"] = 0.5 + 0.02 * (w.fields["x"] - 0.5)
    w.fields["y"] = 0.5 + 0.02 * (w.fields["y"] - 0.5)
    w.fields["z"] = torch.full((n,), 0.5) + 0.25 * (torch.arange(n) % 3).float()     # three depth planes, huge tie groups
    w.fields["I"] = w.fields["I"] * 20.0
    full_check(w, 16)


def test_ordered_heavy_tile_spans_many_chunks():
    n = 300_000
    w = ordered(wl.make_config(0, n=n, size=(64, 64)), absorb=[0.7])
    w.fields["x"] = 0.5 + 0.03 * (w.fields["x"] - 0.5)
    w.fields["y"] = 0.5 + 0.03 * (w.fields["y"] - 0.5)
    w.fields["h"][: n // 2] = 1e-5                               # half SMALL
    w.fields["I"] = w.fields["I"] * 0.5
    st, g = full_check(w, 16)
    assert st["chunks"] >= 8


def test_ordered_zero_absorption_equals_the_additive_sum():
    w = ordered(wl.make_config(0, n=30_000, size=(96, 96)), absorb=[0.0])
    lut = wl.palette()
    ref, g, cam = oracle_frame(w, lut, 16)
    r, f, kw, img = gpu_frame(w, lut, 16)
    assert_image_close(img, ref, "ordered, kappa = 0")
    img_add = r.render(f, w.species, **dict(kw, additive=True))
    torch.cuda.synchronize()
    a, b_ = img.double().cpu().numpy(), img_add.double().cpu().numpy()
    assert np.linalg.norm(a - b_) <= 2e-6 * np.linalg.norm(b_)


def test_ordered_order_matters_and_permutation_of_memory_does_not():
    """Reversing the depth order changes the image; shuffling the particles in memory (distinct depths) does not."""
    w = ordered(wl.make_config(4, n=40_000, size=(128, 96), eta=0.1))
    w.fields["I"] = w.fields["I"] * 300.0
    lut = wl.palette()
    r, f, kw, img = gpu_frame(w, lut, 16)
    img = img.clone()
    perm = torch.randperm(w.n, generator=torch.Generator().manual_seed(3))
    w2 = ordered(wl.make_config(4, n=40_000, size=(128, 96), eta=0.1))
    w2.fields = {k: v[perm].contiguous() for k, v in w.fields.items()}
    # two species are contiguous index ranges: shuffle inside a single species instead
    n_gas = w.species[0].end
    perm = torch.cat([torch.randperm(n_gas, generator=torch.Generator().manual_seed(4)),
                      n_gas + torch.randperm(w.n - n_gas, generator=torch.Generator().manual_seed(5))])
    w2.fields = {k: v[perm].contiguous() for k, v in w.fields.items()}
    ref2, g2, cam2 = oracle_frame(w2, lut, 16)
    r2, f2, kw2, img2 = gpu_frame(w2, lut, 16)
    assert_image_close(img2, ref2, "shuffled")
    zc = g2["zc"][g2["cls"] != so.CULLED]
    if len(np.unique(zc)) == len(zc):                             # no depth ties: the image is independent of memory order
        a, b_ = img.double().cpu().numpy(), img2.double().cpu().numpy()
        assert np.linalg.norm(a - b_) <= 5e-6 * np.linalg.norm(a)
    # mirrored depth (camera on the other side would be another image; here: the additive image differs from ordered)
    img_add = r.render(f, w.species, **dict(kw, additive=True)).double().cpu().numpy()
    assert np.linalg.norm(img.double().cpu().numpy() - img_add) > 1e-3 * np.linalg.norm(img_add)


def test_ordered_pair_overflow_is_reported():
    w = ordered(wl.make_config(0, n=50_000, size=(128, 128)))
    lut = wl.palette()
    r, f, kw, img = gpu_frame(w, lut, 16, pair_capacity=1000)
    st = r.stats()
    assert st["overflow"] == 1 and st["pairs"] > 1000
    assert float(img.abs().max()) == 0.0
    img2 = r.render(f, w.species, pair_capacity=200_000, **kw)
    assert r.stats()["overflow"] == 0 and float(img2.max()) > 0


@pytest.mark.parametrize("n", [0, 1, 33, 4097])
def test_ordered_tiny_counts(n):
    w = ordered(wl.make_config(0, n=max(n, 1), size=(64, 48)), absorb=[1.0])
    if n == 0:
        w.fields = {k: v[:0] for k, v in w.fields.items()}
        w.n = 0
        w.species[0].end = 0
    full_check(w, 16)


def test_a_frame_captured_in_a_cuda_graph_replays_to_the_same_image():
    """splotch_render only enqueues kernels and memsets on the caller's stream, so a frame can be captured into a CUDA graph (the
    launch gaps of a small frame go away); the replayed image equals the directly rendered one to float32 reproducibility."""
    b = _binding()
    w = wl.make_config(0, n=50_000, size=(192, 160))
    lut = wl.palette()
    r = b.Renderer(w.width, w.height, w.n)
    r.set_camera(w.camera)
    r.set_colormap(0, lut)
    f = {k: v.cuda().contiguous() for k, v in w.fields.items()}
    kw = dict(chi=w.chi, r_small=w.r_small, r_large=8.0, z_near=w.z_near, tile=16, additive=True)      # r_large = 8: k_large takes part
    img = torch.empty((w.height, w.width, 3), dtype=torch.float32, device="cuda")
    r.render(f, w.species, image=img, **kw)
    torch.cuda.synchronize()
    ref = img.clone()
    assert r.stats()["count"][wl_LARGE] > 0
    side, graph = torch.cuda.Stream(), torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        r.render(f, w.species, image=img, **kw)
        torch.cuda.synchronize()
        with torch.cuda.graph(graph, stream=side):
            r.render(f, w.species, image=img, **kw)
    torch.cuda.synchronize()
    for _ in range(3):
        img.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert float((img - ref).abs().max()) <= 1e-6 * float(ref.max())
    r.close()
