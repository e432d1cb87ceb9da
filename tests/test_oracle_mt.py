"""The all-cores oracle drivers (oracle/splotch_oracle_mt.c) against the single-threaded definition: bit-identical.

The row-band scheme (mirroring the paper's OpenMP tiles) only cuts the image rows into
bands and calls the unchanged single-threaded functions on each band, so every pixel receives the same contributions
in the same order.  This is what allows the all-cores driver to stand in for the definition in the full-size tests."""
import numpy as np
import pytest

from oracle import splotch_oracle as so
from paper_1309_1114_b200 import workloads as wl


def _np(fields):
    return {k: v.numpy() for k, v in fields.items()}


@pytest.mark.parametrize("cfg,n,size,additive,threads", [
    (1, 60_000, (200, 150), True, 4), (1, 60_000, (200, 150), True, 3), (4, 40_000, (192, 108), False, 4),
    (3, 20_000, (256, 192), True, 5), (3, 20_000, (256, 192), False, 2), (0, 5_000, (64, 7), True, 16),
])
def test_row_band_driver_is_bit_identical(cfg, n, size, additive, threads):
    w = wl.make_config(cfg, n=n, size=size)
    if not additive:
        w.fields["I"] = w.fields["I"] * 50.0
    lut = wl.palette().numpy()
    luts = [lut if s.use_colormap else None for s in w.species]
    kw = dict(chi=w.chi, r_small=w.r_small, r_large=12.0, z_near=w.z_near, tile=16, additive=additive,
              apply_transfer=additive, return_geometry=True)
    a, ga, _ = so.render(_np(w.fields), w.species, luts, w.camera, w.width, w.height, threads=1, **kw)
    b, gb, _ = so.render(_np(w.fields), w.species, luts, w.camera, w.width, w.height, threads=threads, **kw)
    assert a.max() > 0
    assert np.array_equal(a.view(np.uint64), b.view(np.uint64))
    for k in ga:
        assert np.array_equal(ga[k].view(np.uint8), gb[k].view(np.uint8)), k


def test_amplitude_ranges_are_bit_identical_across_a_species_boundary():
    n = (1 << 18) + 777                       # two ranges of the per-particle driver, species boundary inside the first
    w = wl.make_config(2, n=n, size=(64, 64))
    lut = wl.palette().numpy()
    luts = [lut if s.use_colormap else None for s in w.species]
    f = _np(w.fields)
    a = so.amplitude(f["I"], f["scalar"], f["h"], w.species, luts, threads=1)
    b = so.amplitude(f["I"], f["scalar"], f["h"], w.species, luts, threads=3)
    for u, v in zip(a, b):
        assert np.array_equal(u.view(np.uint64), v.view(np.uint64))


def test_window_inside_the_band_driver():
    w = wl.make_config(1, n=30_000, size=(160, 120))
    lut = wl.palette().numpy()
    win = (17, 90, 33, 101)
    a = so.render(_np(w.fields), w.species, [lut], w.camera, w.width, w.height, window=win, threads=1)
    b = so.render(_np(w.fields), w.species, [lut], w.camera, w.width, w.height, window=win, threads=4)
    assert np.array_equal(a.view(np.uint64), b.view(np.uint64)) and a[40:100, 20:90].max() > 0
    assert a[:33].max() == 0 and a[:, :17].max() == 0


def test_host_cores_is_reported():
    assert so.host_cores() >= 1 and so.lib().orc_mt_threads() >= 1
