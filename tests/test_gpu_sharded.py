"""The sharded frame on one GPU: two shards rendered one after the other through ShardedRenderer's code path
(sharded_frame with the library as the partial renderer), summed, transfer applied after the sum by the library."""
import numpy as np
import pytest
import torch

from oracle import splotch_oracle as so
from paper_1309_1114_b200 import sharded, workloads as wl

pytestmark = pytest.mark.gpu


def test_two_shards_on_one_gpu_sum_to_the_oracle_frame():
    from paper_1309_1114_b200 import binding
    w = wl.make_config(2, n=200_000, size=(256, 160), eta=0.06)
    w.fields["I"] = w.fields["I"] * 30.0                              # 1 - exp(-S) differs visibly from S
    lut = wl.palette()
    r = binding.Renderer(w.width, w.height, w.n)
    r.set_camera(w.camera)
    r.set_colormap(0, lut)
    prm = dict(chi=w.chi, r_small=w.r_small, r_large=w.r_large, tile=16, additive=True, apply_transfer=True)
    total = None
    for rank in range(2):
        lo, hi = sharded.shard_range(w.n, rank, 2)
        f = {k: v.cuda() for k, v in sharded.shard_fields(w.fields, lo, hi).items()}
        sp = sharded.shard_species(w.species, lo, hi)
        part = sharded.sharded_frame(lambda ff, ss, pp: r.render(ff, ss, **pp).clone(), f, sp, dict(prm, apply_transfer=False))
        total = part if total is None else total + part              # what the all-reduce does
    img = r.apply_transfer(total)
    torch.cuda.synchronize()
    ref = so.render({k: v.numpy() for k, v in w.fields.items()}, w.species, [lut.numpy(), None], w.camera, w.width, w.height,
                    chi=w.chi, r_small=w.r_small, r_large=w.r_large, tile=16, additive=True, apply_transfer=True, threads=0)
    g = img.double().cpu().numpy()
    assert np.linalg.norm(g - ref) <= 1e-5 * np.linalg.norm(ref) and np.abs(g - ref).max() <= 1e-4 * ref.max()
    r.close()


@pytest.mark.parametrize("tile", [16, 32])
def test_shards_composed_from_their_fixed_point_sums_in_one_kernel(tile):
    """splotch_compose_shards: three shards rendered into three workspaces (on one GPU; on several GPUs the pointers would be
    peer-mapped), composed by ONE kernel from the tiles' exact fixed-point sums: the image equals the oracle's frame of the whole
    set, does not depend on the order of the shards (bit for bit), and a rank can compose its own share of the tiles."""
    from paper_1309_1114_b200 import binding
    w = wl.make_config(3, n=180_000, size=(320, 224))                # LARGE particles too: k_large feeds the same sums
    w.r_large = 40.0
    w.fields["I"] = w.fields["I"] * 0.05
    w.fields["I"][:60_000] *= 1.0e3                                   # the shards' amplitudes, and so their fixed-point units, differ
    lut = wl.palette()
    prm = dict(chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=tile, additive=True, apply_transfer=False)
    rs = []
    for rank in range(3):
        lo, hi = sharded.shard_range(w.n, rank, 3)
        r = binding.Renderer(w.width, w.height, w.n)
        r.set_camera(w.camera)
        r.set_colormap(0, lut)
        f = {k: v.cuda().contiguous() for k, v in sharded.shard_fields(w.fields, lo, hi).items()}
        r.render(f, sharded.shard_species(w.species, lo, hi), **prm)
        torch.cuda.synchronize()
        assert r.stats()["overflow"] == 0
        rs.append(r)
    ws = [r.last_workspace for r in rs]
    img = rs[0].compose_shards(ws, tile, apply_transfer=True)
    rev = rs[0].compose_shards(ws[::-1], tile, apply_transfer=True)
    torch.cuda.synchronize()
    assert torch.equal(img, rev)                                      # exact sums: the order of the shards does not matter
    ref = so.render({k: v.numpy() for k, v in w.fields.items()}, w.species, [lut.numpy()], w.camera, w.width, w.height,
                    chi=w.chi, r_small=w.r_small, r_large=w.r_large, z_near=w.z_near, tile=tile, additive=True,
                    apply_transfer=True, threads=0)
    g = img.double().cpu().numpy()
    assert np.linalg.norm(g - ref) <= 1e-5 * np.linalg.norm(ref) and np.abs(g - ref).max() <= 1e-4 * ref.max()
    # two ranks compose half of the tiles each into one image
    ntx, nty = -(-w.width // tile), -(-w.height // tile)
    half = (ntx * nty) // 2
    both = torch.zeros_like(img)
    rs[1].compose_shards(ws, tile, image=both, tile_range=(0, half), apply_transfer=True)
    rs[2].compose_shards(ws, tile, image=both, tile_range=(half, ntx * nty), apply_transfer=True)
    torch.cuda.synchronize()
    assert torch.equal(both, img)
    with pytest.raises(binding.SplotchError):
        rs[0].compose_shards(ws * 6, tile)                           # more than 16 shards
    for r in rs:
        r.close()
