"""Particle sharding in additive mode: the rank logic on two CPU ranks over gloo.

The partial renderer is injectable, so each rank renders its shard with the CPU oracle here (the GPU path is covered on
one GPU by tests/test_gpu_sharded.py); what is checked is the sharding itself: index ranges, species ranges cut to the
shard, ranges of auto_range species agreed across ranks, one sum all-reduce, transfer applied after the sum."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from oracle import splotch_oracle as so
    from paper_1309_1114_b200 import sharded, workloads as wl
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.make_config(2, n=30_001, size=(96, 64), eta=0.06)             # two species, boundary inside rank 1's shard
    w.species[0].auto_range = True
    lut = wl.palette().numpy()
    lo, hi = sharded.shard_range(w.n, rank, world)
    f = sharded.shard_fields(w.fields, lo, hi)
    sp = sharded.shard_species(w.species, lo, hi)

    def oracle_partial(fields, species, prm):
        luts = [lut if s.use_colormap else None for s in species]
        img = so.render({k: v.numpy() for k, v in fields.items()}, species, luts, w.camera, w.width, w.height,
                        chi=w.chi, r_small=w.r_small, r_large=w.r_large, additive=True, apply_transfer=prm["apply_transfer"])
        return torch.from_numpy(img)

    img = sharded.sharded_frame(oracle_partial, f, sp, dict(additive=True, apply_transfer=True), dist)
    out.put((rank, lo, hi, [(s.begin, s.end) for s in sp], img.numpy()))
    dist.destroy_process_group()


def test_two_ranks_sum_to_the_whole_frame():
    sys.path.insert(0, ROOT)
    from oracle import splotch_oracle as so
    from paper_1309_1114_b200 import workloads as wl
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29633, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = wl.make_config(2, n=30_001, size=(96, 64), eta=0.06)
    w.species[0].auto_range = True
    lut = wl.palette().numpy()
    ref = so.render({k: v.numpy() for k, v in w.fields.items()}, w.species, [lut, None], w.camera, w.width, w.height,
                    chi=w.chi, r_small=w.r_small, r_large=w.r_large, additive=True, apply_transfer=True)
    (r0, lo0, hi0, sp0, a), (r1, lo1, hi1, sp1, b) = res
    assert (lo0, hi0, lo1, hi1) == (0, 15004, 15004, 30001)               # shares rounded up to a multiple of 4
    n_gas = (6 * 30_001) // 10
    assert sp0 == [(0, 15004), (15004, 15004)] and sp1 == [(0, n_gas - 15004), (n_gas - 15004, 30001 - 15004)]
    assert np.array_equal(a, b)                                           # every rank holds the full image
    assert ref.max() > 0 and np.abs(a - ref).max() <= 1e-12 * ref.max()   # double-precision partial sums: rounding order only


def test_ordered_mode_is_refused_and_ranges_cover_the_set():
    sys.path.insert(0, ROOT)
    import pytest
    from paper_1309_1114_b200 import sharded
    with pytest.raises(ValueError):
        sharded.sharded_frame(lambda f, s, p: None, {}, [], dict(additive=False))
    for n in (0, 1, 5, 4096, 10_000_003):
        for world in (1, 2, 3, 8):
            r = [sharded.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n and all(a[1] == b[0] for a, b in zip(r, r[1:]))
            assert all(lo % 4 == 0 for lo, _ in r if lo < n)
