"""splotch_render_host in additive mode: the paper's per-chunk offload loop (Fig. 3) with the copy of
the next chunk overlapping the kernels of the current one (:354).  The chunked frame must equal the oracle's frame (and so
the one-shot frame) to the north_star tolerance, whatever the chunk size, the species boundaries and the order in which
the amplitudes grow; a set whose pairs exceed the workspace's record capacity renders as long as each chunk fits."""
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


def _renderer(w, lut, chunk):
    r = _binding().Renderer(w.width, w.height, max(w.n, 1))
    r.set_camera(w.camera)
    for s, sp in enumerate(w.species):
        if sp.use_colormap:
            r.set_colormap(s, lut)
    r.set_host_chunk(chunk)
    return r


def _oracle(w, lut, tile):
    luts = [lut.numpy() if s.use_colormap else None for s in w.species]
    return so.render({k: v.numpy() for k, v in w.fields.items()}, w.species, luts, w.camera, w.width, w.height,
                     chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=tile, additive=True,
                     return_geometry=True, threads=0)


def _close(img, ref, what):
    g = img.double().numpy()
    rel = np.linalg.norm(g - ref) / np.linalg.norm(ref)
    mab = np.abs(g - ref).max() / ref.max()
    assert rel <= REL_L2 and mab <= MAX_ABS, f"{what}: rel L2 {rel:.3e}, max abs {mab:.3e}"


def _host(fields):
    return {k: v.contiguous().pin_memory() for k, v in fields.items()}


@pytest.mark.parametrize("cfg,n,size,chunk,tile", [(1, 300_000, (320, 240), 40_000, 16), (2, 250_000, (256, 160), 33_332, 16),
                                                   (3, 120_000, (384, 256), 17_000, 32), (0, 50_000, (128, 128), 50_000, 8)])
def test_chunked_host_frame_matches_the_oracle(cfg, n, size, chunk, tile):
    w = wl.make_config(cfg, n=n, size=size, eta=0.06 if cfg == 2 else None)
    if cfg == 3:
        w.r_large = 16.0
    lut = wl.palette()
    ref, g, _ = _oracle(w, lut, tile)
    r = _renderer(w, lut, chunk)
    kw = dict(chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=tile, additive=True)
    out = torch.empty((w.height, w.width, 3), dtype=torch.float32).pin_memory()
    r.render_host(_host(w.fields), w.species, out, **kw)
    st = r.stats()
    assert st["overflow"] == 0 and st["n"] == w.n
    assert st["count"] == [int((g["cls"] == c).sum()) for c in range(4)]          # totals over the chunks
    assert st["pairs"] == int(so.tile_counts(g, w.width, w.height, tile).sum())
    _close(out, ref, f"cfg{cfg} in chunks of {chunk}")
    # the one-shot device frame of the same context agrees as well
    dev = {k: v.cuda() for k, v in w.fields.items()}
    img = r.render(dev, w.species, **kw)
    torch.cuda.synchronize()
    _close(img.cpu(), ref, "one shot")
    r.close()


def test_out_of_core_set_larger_than_the_record_capacity():
    w = wl.make_config(0, n=400_000, size=(512, 512))            # ~2.7 pairs per particle
    lut = wl.palette()
    ref, g, _ = _oracle(w, lut, 16)
    pairs = int(so.tile_counts(g, w.width, w.height, 16).sum())
    cap = pairs // 8              # the workspace (sized for either mode) then holds about half of the frame's records
    r = _renderer(w, lut, 40_000)                                # ten chunks of ~ pairs / 10 records each
    kw = dict(chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=16, additive=True)
    dev = {k: v.cuda() for k, v in w.fields.items()}
    img = r.render(dev, w.species, pair_capacity=cap, **kw)
    torch.cuda.synchronize()
    assert r.stats()["overflow"] == 1 and float(img.abs().max()) == 0.0          # resident rendering cannot hold it
    out = torch.empty((w.height, w.width, 3), dtype=torch.float32).pin_memory()
    r.render_host(_host(w.fields), w.species, out, pair_capacity=cap, **kw)
    st = r.stats()
    assert st["overflow"] == 0 and st["pairs"] == pairs and st["pair_capacity"] < pairs
    _close(out, ref, "out of core")
    r.close()


def test_amplitudes_that_grow_from_chunk_to_chunk_rescale_the_sums():
    """Particles ordered from faint to bright over six decades: every chunk raises the fixed-point unit of the tiles'
    sums, the earlier chunks' sums are shifted to it (k_rescale)."""
    w = wl.make_config(0, n=120_000, size=(160, 160))
    order = torch.argsort(w.fields["h"])
    w.fields = {k: v[order].contiguous() for k, v in w.fields.items()}
    w.fields["I"] = torch.logspace(-3, 3, w.n, dtype=torch.float64).to(torch.float32)
    lut = wl.palette()
    ref, g, _ = _oracle(w, lut, 16)
    r = _renderer(w, lut, 10_000)
    out = torch.empty((w.height, w.width, 3), dtype=torch.float32).pin_memory()
    r.render_host(_host(w.fields), w.species, out, chi=w.chi, r_small=w.r_small, r_large=w.r_large, tile=16)
    _close(out, ref, "growing amplitudes")
    r.close()


def test_empty_set_and_single_chunk():
    w = wl.make_config(0, n=1000, size=(64, 64))
    lut = wl.palette()
    r = _renderer(w, lut, 0)                                     # automatic chunk size: one chunk
    out = torch.empty((64, 64, 3), dtype=torch.float32).pin_memory()
    r.render_host(_host(w.fields), w.species, out, tile=16)
    ref, g, _ = _oracle(w, lut, 16)
    _close(out, ref, "single chunk")
    empty = {k: v[:0].contiguous() for k, v in w.fields.items()}
    w.species[0].end = 0
    r.render_host(empty, w.species, out, tile=16)
    assert float(out.abs().max()) == 0.0
    r.close()
