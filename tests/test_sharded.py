"""Row-band sharding of one map over several ranks: host logic on CPU with gloo (world_size 2),
bit-identity of the band decomposition on the GPU."""
import dataclasses
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1406_0559_b200 import fields, sharded


def test_row_bands_cover_the_lattice_once_and_are_tile_aligned():
    for n2, world in [(3414, 2), (35110, 8), (122880, 8), (96000, 3), (100, 4), (64, 2), (1, 1), (0, 2), (6400, 7)]:
        bands = sharded.row_bands(n2, world)
        assert len(bands) == world
        pos = 0
        for j0, nj in bands:
            assert nj >= 0 and (nj == 0 or j0 == pos) and (nj == 0 or j0 % sharded.TILE == 0)
            pos += nj
        assert pos == n2
        tiles = [(nj + sharded.TILE - 1) // sharded.TILE for _, nj in bands]
        assert max(tiles) - min(tiles) <= 1  # balanced to within one tile


def test_row_bands_rejects_bad_arguments():
    with pytest.raises(ValueError):
        sharded.row_bands(10, 0)
    with pytest.raises(ValueError):
        sharded.row_bands(-1, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _gloo_worker(rank, world, port, q):
    """Each rank shoots its band with the ORACLE (the CPU stand-in for the per-rank kernel launch), then the maps go
    through the same allreduce_map the GPU path uses."""
    import oracle

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = dataclasses.replace(fields.CONFIGS[1], npix=64, sub=4)
        xy, m = fields.lens_field(cfg)
        args = (cfg.kappa, cfg.gamma, cfg.s, cfg.map_side, cfg.npix, cfg.ray_spacing)
        g = oracle.geometry(*args)
        j0, nj = sharded.row_bands(g.n2, world)[rank]
        r = oracle.shoot_block(*args, xy, m, block=(0, j0, g.n1, nj))
        st = r["stats"]
        count = torch.from_numpy(r["count"].astype(np.int32))
        counters = torch.tensor([st["rays_in_map"], st["rays_outside"], st["rays_lost"], st["rays_total"]], dtype=torch.int64)
        sharded.allreduce_map(count, counters)
        if rank == 0:
            full = oracle.shoot_block(*args, xy, m)
            q.put((bool(np.array_equal(count.numpy(), full["count"])), counters.tolist(),
                   [full["stats"][k] for k in ("rays_in_map", "rays_outside", "rays_lost", "rays_total")], g.n1 * g.n2))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_band_sum_equals_the_full_map():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    same, counters, full_counters, rays = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert same and counters == full_counters and counters[3] == rays


@pytest.mark.gpu
def test_band_decomposition_is_bit_identical_on_gpu():
    # three emulated ranks, one after another on one GPU (no rank waits on another): summed band maps == 1-launch map
    from paper_1406_0559_b200 import mlens

    cfg = dataclasses.replace(fields.CONFIGS[4], npix=256, sub=3)
    xy, m = fields.lens_field(cfg)
    with mlens.Mlens.from_config(cfg, xy, m) as h:
        full, _, st_full = h.shoot(want_mag=False)
        full = full.clone()
        acc = torch.zeros_like(full)
        tot = 0
        for rank in range(3):
            c, mag, st = sharded.shoot_sharded(h, rank, 3)
            acc += c
            tot += st["rays_total"]
            assert mag is not None and st["band"][0] % sharded.TILE == 0
        assert tot == st_full["rays_total"] == h.geometry.n1 * h.geometry.n2
        assert torch.equal(acc, full)
