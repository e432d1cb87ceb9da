"""splotch_count_static: the entry point that allocates nothing (its scratch is a static device array of 16 MiB).

Collected last on purpose (the suite runs with pytest -x).  The new entry point's class counts and per-tile pair counts
must equal, bit for bit (integer work), what the existing path reports after rendering the same set with a workspace
(splotch_get_stats / splotch_debug_tile_counts), on two calls in a row with different inputs: the second call meets the
first call's leftovers in the shared array.
"""
import pytest
import torch

from paper_1309_1114_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _binding():
    from paper_1309_1114_b200 import binding
    return binding


def _existing_path(b, w, fields, tile):
    r = b.Renderer(w.width, w.height, w.n)
    r.set_camera(w.camera)
    r.set_colormap(0, wl.palette())
    kw = dict(chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=tile, additive=True)
    r.render(fields, w.species, **kw)
    torch.cuda.synchronize()
    st = r.stats()
    assert st["overflow"] == 0
    return r, kw, [int(c) for c in st["count"]], r.debug_tile_counts(tile).clone()


def _static_path(r, w, fields, kw, tile):
    ntx, nty = -(-w.width // tile), -(-w.height // tile)
    tiles = torch.full((nty, ntx), -1, dtype=torch.int32, device="cuda")       # outputs start dirty: the call overwrites them
    classes = torch.full((4,), -1, dtype=torch.int64, device="cuda")
    # no device allocation inside the call: the driver's free memory must not drop (a cudaMalloc in the library would not show in
    # torch's own counters; torch's allocator keeps its blocks, so garbage collected meanwhile does not move this number down)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    r.count_static(fields, w.species, tiles, classes, **kw)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before
    return [int(c) for c in classes.cpu()], tiles


def test_count_static_matches_the_workspace_path_on_two_calls_in_a_row():
    b = _binding()
    # call 1: halos seen from outside, 16-px tiles (SMALL + MEDIUM); call 2: camera inside a halo, 32-px tiles (LARGE particles,
    # super-tile bins and the third bin per tile), other image size: a different layout of the shared scratch array
    cases = [(wl.make_config(1, n=300_000, size=(800, 600)), 16), (wl.make_config(3, n=150_000, size=(640, 480)), 32),
             (wl.make_config(1, n=4_099, size=(200, 136)), 8)]
    cases[1][0].r_large = 24.0
    results = []
    for w, tile in cases:
        f = {k: v.cuda().contiguous() for k, v in w.fields.items()}
        r, kw, classes_ref, tiles_ref = _existing_path(b, w, f, tile)
        results.append((r, w, f, kw, tile, classes_ref, tiles_ref))
    assert results[0][5][1] > 0 and results[0][5][2] > 0 and results[1][5][3] > 0          # SMALL, MEDIUM; LARGE
    for rnd in range(2):                                   # the whole sequence twice: every call follows another one's leftovers
        for r, w, f, kw, tile, classes_ref, tiles_ref in results:
            classes, tiles = _static_path(r, w, f, kw, tile)
            assert classes == classes_ref, (w.name, rnd)
            assert torch.equal(tiles, tiles_ref), (w.name, rnd)
    # the same call twice in a row gives the same answer (the scratch is cleared, not accumulated into)
    r, w, f, kw, tile, classes_ref, tiles_ref = results[0]
    for _ in range(2):
        classes, tiles = _static_path(r, w, f, kw, tile)
        assert classes == classes_ref and torch.equal(tiles, tiles_ref)
    # unaligned field pointers and an empty set
    g = {k: torch.cat([v.new_zeros(1), v])[1:] for k, v in f.items()}
    classes, tiles = _static_path(r, w, g, kw, tile)
    assert classes == classes_ref and torch.equal(tiles, tiles_ref)
    e = {k: v[:0] for k, v in f.items()}
    sp0 = [wl.Species(0, 0)]
    tiles0 = torch.full_like(tiles_ref, -1)
    classes0 = torch.full((4,), -1, dtype=torch.int64, device="cuda")
    r.count_static(e, sp0, tiles0, classes0, **kw)
    torch.cuda.synchronize()
    assert int(tiles0.abs().sum()) == 0 and int(classes0.abs().sum()) == 0
    for x in results:
        x[0].close()


def test_count_static_rejects_what_does_not_fit_the_static_array():
    b = _binding()
    w = wl.make_config(1, n=10_000, size=(4096, 4096))
    f = {k: v.cuda().contiguous() for k, v in w.fields.items()}
    r = b.Renderer(w.width, w.height, w.n)
    r.set_camera(w.camera)
    r.set_colormap(0, wl.palette())
    kw = dict(chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, additive=True)
    tiles = torch.zeros((256, 256), dtype=torch.int32, device="cuda")
    classes = torch.zeros(4, dtype=torch.int64, device="cuda")
    with pytest.raises(b.SplotchError, match="static array holds"):
        r.count_static(f, w.species, tiles, classes, tile=16, **kw)            # 132,096 bins x 148 rows: 78 MB
    r.count_static(f, w.species, tiles[:64, :64].contiguous(), classes, tile=64, **kw)      # 9,216 bins: fits
    torch.cuda.synchronize()
    assert int(classes.sum()) == w.n
    with pytest.raises(b.SplotchError):
        r.count_static(f, w.species, tiles, classes, tile=64, **dict(kw, additive=False))
    r.close()
