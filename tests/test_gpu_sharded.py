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
