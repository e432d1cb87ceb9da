"""Pre-processing on the device: the normalisation range found from the data (PAPER.md:76, :166 fn. 1) and
the vector colour mode rho^R = v_x, rho^G = v_y, rho^B = v_z, against the oracle."""
import numpy as np
import pytest
import torch

from oracle import splotch_oracle as so
from paper_1309_1114_b200 import workloads as wl

pytestmark = pytest.mark.gpu
REL_L2, MAX_ABS = 1e-5, 1e-4


def _binding():
    from paper_1309_1114_b200 import binding
    return binding


def _oracle(w, lut, tile, additive=True):
    luts = [lut.numpy() if s.use_colormap and not s.vector_colour else None for s in w.species]
    return so.render({k: v.numpy() for k, v in w.fields.items()}, w.species, luts, w.camera, w.width, w.height,
                     chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=tile, additive=additive, threads=0)


def _renderer(w, lut):
    r = _binding().Renderer(w.width, w.height, max(w.n, 1))
    r.set_camera(w.camera)
    for s, sp in enumerate(w.species):
        if sp.use_colormap and not sp.vector_colour:
            r.set_colormap(s, lut)
    return r


def _close(img, ref, what):
    g = img.double().cpu().numpy()
    assert np.isfinite(g).all()
    rel = np.linalg.norm(g - ref) / np.linalg.norm(ref)
    mab = np.abs(g - ref).max() / ref.max()
    assert rel <= REL_L2 and mab <= MAX_ABS, f"{what}: rel L2 {rel:.3e}, max abs {mab:.3e}"


def _with_vectors(w, seed=5):
    g = torch.Generator().manual_seed(seed)
    for k in ("cr", "cg", "cb"):
        w.fields[k] = (torch.randn(w.n, generator=g) * 120.0 + 30.0).to(torch.float32)       # a velocity-like field
    return w


@pytest.mark.parametrize("additive", [True, False])
def test_automatic_range_two_species(additive):
    """Species 0: colour map over log10(scalar) with the range found on the device; species 1: colour map over the scalar
    itself with a given range.  NaN / Inf / non-positive scalars are left out of the extrema."""
    w = wl.make_config(2, n=300_000, size=(320, 200), eta=0.06)
    n0 = w.species[0].end
    sc = w.fields["scalar"].clone()
    sc[:n0] = torch.pow(10.0, sc[:n0].double() * 0.5 - 1.0).to(torch.float32)        # positive, wide range: log10 is meaningful
    sc[::1001] = float("nan")
    sc[5::2003] = float("inf")
    sc[7::3001] = -1.0
    w.fields["scalar"] = sc
    w.species[0].scalar_log10, w.species[0].auto_range = True, True
    w.species[0].scalar_min, w.species[0].scalar_max = 7.0, 7.0                     # ignored
    w.species[1].use_colormap, w.species[1].scalar_min, w.species[1].scalar_max = True, float(sc[n0:][torch.isfinite(sc[n0:])].min()), 9.0
    if not additive:
        w.fields["I"] = w.fields["I"] * 100.0
    lut = wl.palette()
    ref = _oracle(w, lut, 16, additive)
    r = _renderer(w, lut)
    dev = {k: v.cuda() for k, v in w.fields.items()}
    img = r.render(dev, w.species, chi=w.chi, r_small=w.r_small, r_large=w.r_large, tile=16, additive=additive)
    torch.cuda.synchronize()
    _close(img, ref, "auto range")
    r.close()


@pytest.mark.parametrize("additive,auto", [(True, False), (True, True), (False, True)])
def test_vector_colour_mode(additive, auto):
    w = _with_vectors(wl.make_config(1, n=250_000, size=(300, 200)))
    w.species[0].vector_colour, w.species[0].auto_range = True, auto
    w.species[0].scalar_min, w.species[0].scalar_max = -200.0, 300.0
    if not additive:
        w.fields["I"] = w.fields["I"] * 100.0
    lut = wl.palette()
    ref = _oracle(w, lut, 16, additive)
    r = _renderer(w, lut)
    dev = {k: v.cuda() for k, v in w.fields.items()}
    img = r.render(dev, w.species, chi=w.chi, r_small=w.r_small, r_large=w.r_large, tile=16, additive=additive)
    torch.cuda.synchronize()
    _close(img, ref, "vector colours")
    # the three channels differ (a grey image would mean the components were not told apart)
    g = img.double().cpu().numpy()
    assert np.abs(g[:, :, 0] - g[:, :, 1]).max() > 1e-3 * g.max()
    r.close()


def test_missing_vector_fields_are_reported():
    b = _binding()
    w = wl.make_config(0, n=1000, size=(64, 64))
    w.species[0].vector_colour = True
    r = _renderer(w, wl.palette())
    with pytest.raises(b.SplotchError) as e:
        r.render({k: v.cuda() for k, v in w.fields.items()}, w.species)
    assert e.value.code == b.SPLOTCH_EINVAL
    r.close()


def test_host_chunks_with_automatic_range_and_vector_colours():
    """splotch_render_host: the ranges are reduced over the whole set in a first pass through the staging buffer, then the
    chunks are coloured; species boundary inside a chunk."""
    w = _with_vectors(wl.make_config(2, n=200_000, size=(256, 160), eta=0.06))
    w.species[0].auto_range = True
    w.species[1].vector_colour, w.species[1].auto_range = True, True
    lut = wl.palette()
    ref = _oracle(w, lut, 16)
    r = _renderer(w, lut)
    r.set_host_chunk(30_000)
    out = torch.empty((w.height, w.width, 3), dtype=torch.float32).pin_memory()
    r.render_host({k: v.contiguous().pin_memory() for k, v in w.fields.items()}, w.species, out, chi=w.chi,
                  r_small=w.r_small, r_large=w.r_large, tile=16)
    _close(out, ref, "host chunks, auto range + vectors")
    r.close()
