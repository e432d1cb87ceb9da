"""The paper's own medium-particle scheme as an alternative renderer (Table 1: t_x = 8,
n_p = 16, r_0 = 8): same image as the oracle (and so as the default renderer), its constraints reported as errors."""
import numpy as np
import pytest
import torch

from oracle import splotch_oracle as so
from paper_1309_1114_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _binding():
    from paper_1309_1114_b200 import binding
    return binding


def _frame(w, tile, r_large, np_=16, transfer=False, renderer=1):
    lut = wl.palette()
    r = _binding().Renderer(w.width, w.height, w.n)
    r.set_camera(w.camera)
    for s, sp in enumerate(w.species):
        if sp.use_colormap:
            r.set_colormap(s, lut)
    dev = {k: v.cuda() for k, v in w.fields.items()}
    img = r.render(dev, w.species, chi=w.chi, r_small=w.r_small, r_large=r_large, tile=tile, additive=True,
                   apply_transfer=transfer, renderer=renderer, btile_np=np_)
    torch.cuda.synchronize()
    st = r.stats()
    luts = [lut.numpy() if s.use_colormap else None for s in w.species]
    ref, g, _ = so.render({k: v.numpy() for k, v in w.fields.items()}, w.species, luts, w.camera, w.width, w.height,
                          chi=w.chi, r_small=w.r_small, r_large=r_large, tile=tile, additive=True, apply_transfer=transfer,
                          return_geometry=True, threads=0)
    r.close()
    return img.double().cpu().numpy(), ref, g, st


@pytest.mark.parametrize("cfg,n,size,tile,r0,np_", [(1, 300_000, (320, 240), 8, 8.0, 16), (1, 300_000, (322, 243), 16, 8.0, 64),
                                                    (0, 60_000, (160, 160), 8, 5.0, 3), (3, 80_000, (384, 256), 16, 16.0, 16),
                                                    (2, 200_000, (256, 144), 8, 8.0, 16)])
def test_btile_renderer_matches_the_oracle(cfg, n, size, tile, r0, np_):
    w = wl.make_config(cfg, n=n, size=size, eta=0.06 if cfg == 2 else None)
    g_img, ref, g, st = _frame(w, tile, r0, np_)
    assert st["overflow"] == 0
    assert st["count"] == [int((g["cls"] == c).sum()) for c in range(4)]
    assert st["count"][2] > 1000
    # one record per SMALL and per MEDIUM particle: the paper bins by the tile of the centre, not by coverage
    assert st["pairs"] == st["count"][1] + st["count"][2]
    rel = np.linalg.norm(g_img - ref) / np.linalg.norm(ref)
    mab = np.abs(g_img - ref).max() / ref.max()
    assert rel <= 1e-5 and mab <= 1e-4, (rel, mab)


def test_btile_transfer_and_default_renderer_agree():
    w = wl.make_config(1, n=150_000, size=(200, 200))
    w.fields["I"] = w.fields["I"] * 40.0
    a, ref, _, _ = _frame(w, 8, 8.0, transfer=True)
    b, _, _, _ = _frame(w, 8, 8.0, transfer=True, renderer=0)
    assert np.abs(a - ref).max() <= 1e-4 * ref.max() and np.abs(a - b).max() <= 1e-4 * ref.max()


def test_btile_constraints_are_errors():
    b = _binding()
    w = wl.make_config(0, n=1000, size=(64, 64))
    r = b.Renderer(64, 64, 1000)
    r.set_camera(w.camera)
    r.set_colormap(0, wl.palette())
    dev = {k: v.cuda() for k, v in w.fields.items()}
    for kw in (dict(tile=8, r_large=9.0), dict(tile=32, r_large=8.0), dict(tile=8, r_large=8.0, additive=False)):
        with pytest.raises(b.SplotchError) as e:
            r.render(dev, w.species, renderer=1, **kw)                  # r_0 > tile; tile too large; ordered mode
        assert e.value.code == b.SPLOTCH_EINVAL
    r.render(dev, w.species, renderer=1, tile=8, r_large=8.0)
    r.close()
