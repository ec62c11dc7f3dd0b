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


class _OracleHandle:
    """Stand-in for ``mlens.Mlens`` on a box without a GPU: same five members ``shoot_sharded`` uses, CPU tensors, the
    FP64 oracle as the band shooter.  Test infrastructure only."""

    def __init__(self, oracle, cfg, xy, m):
        self.o, self.cfg, self.xy, self.m = oracle, cfg, xy, m
        self.args = (cfg.kappa, cfg.gamma, cfg.s, cfg.map_side, cfg.npix, cfg.ray_spacing)
        self.geometry = oracle.geometry(*self.args)
        self.npix = cfg.npix
        self.ctr = dict(rays_total=0, rays_in_map=0, rays_outside=0, rays_lost=0)
        self.max_count = -1
        self.calls = []

    def reset_stats(self, stream=None):
        self.calls.append("reset")
        for k in self.ctr:
            self.ctr[k] = 0

    def shoot_block(self, i0, j0, ni, nj, count=None, stream=None):
        self.calls.append(("band", i0, j0, ni, nj))
        c = count.numpy()  # shares memory with the tensor: accumulates in place, like the kernel
        r = self.o.shoot_block(*self.args, self.xy, self.m, block=(i0, j0, ni, nj), count=c)
        for k in self.ctr:
            self.ctr[k] += r["stats"][k]

    def stats(self, stream=None):
        return dict(self.ctr, n_lens=len(self.m), max_count=self.max_count, elapsed_ms=0.0, kernel_ms=0.0)

    def magnification(self, count, mag=None, stream=None):
        self.calls.append("mag")
        self.max_count = int(count.max())
        return torch.from_numpy(self.o.magnification(count.numpy(), self.geometry.n_avg))


def _gloo_worker(rank, world, port, q):
    """Every rank runs the REAL sharded.shoot_sharded (band plan, zeroing, counters tensor, both all-reduces, Eq. 4 on the
    summed map, max_count refresh) on CPU tensors over gloo; only the per-band kernel launch is replaced by the oracle."""
    import oracle

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = dataclasses.replace(fields.CONFIGS[1], npix=64, sub=4)
        xy, m = fields.lens_field(cfg)
        h = _OracleHandle(oracle, cfg, xy, m)
        count = torch.full((cfg.npix, cfg.npix), 7, dtype=torch.int32)  # stale contents: shoot_sharded must zero them
        count, mag, st = sharded.shoot_sharded(h, rank, world, count=count, device="cpu")
        full = oracle.shoot_block(*h.args, xy, m)
        ok = bool(np.array_equal(count.numpy(), full["count"]))
        ok_mag = bool(np.array_equal(mag.numpy(), oracle.magnification(full["count"], h.geometry.n_avg)))
        band = sharded.row_bands(h.geometry.n2, world)[rank]
        q.put((rank, ok, ok_mag, [st[k] for k in ("rays_in_map", "rays_outside", "rays_lost", "rays_total")],
               [full["stats"][k] for k in ("rays_in_map", "rays_outside", "rays_lost", "rays_total")],
               st["max_count"] == int(full["count"].max()), st["band"] == band,
               h.calls == ["reset", ("band", 0, band[0], h.geometry.n1, band[1]), "mag"]))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_shoot_sharded_equals_the_full_map():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=180) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[0] for g in got] == [0, 1]
    for rank, ok, ok_mag, counters, full_counters, ok_max, ok_band, ok_calls in got:  # identical result on every rank
        assert ok and ok_mag and counters == full_counters and ok_max and ok_band and ok_calls, (rank, counters, full_counters)


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


# ---------------------------------------------------------------------------------------------------------------
# many maps on one GPU (paper_1406_0559_b200/survey.py): the paper's own way of scaling
# ---------------------------------------------------------------------------------------------------------------
def test_survey_parameter_grid_builds_the_jobs():
    from paper_1406_0559_b200 import survey

    base = fields.MapConfig("grid", 64, 4.0, 0.3, 0.1, 0.0, 4, "unit", 900)
    jobs = survey.parameter_grid(base, [0.3, 0.5], [0.0, 0.2], [0.0, 0.9])
    assert len(jobs) == 8 and [j.cfg.seed for j in jobs] == list(range(900, 908))
    assert {(j.cfg.kappa, j.cfg.gamma, j.cfg.s) for j in jobs} == {(k, g, s) for k in (0.3, 0.5) for g in (0.0, 0.2) for s in (0.0, 0.9)}
    for j in jobs:  # Eq. 3: N* follows kappa_* = (1 - s) kappa of each grid point
        assert len(j.lens_m) == j.cfg.n_lens and j.lens_xy.shape == (j.cfg.n_lens, 2)
    if not torch.cuda.is_available():
        with pytest.raises(RuntimeError):
            survey.run_survey(jobs[:1])


@pytest.mark.gpu
def test_survey_driver_matches_one_map_at_a_time():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1406_0559_b200 import mlens, survey

    base = fields.MapConfig("grid", 160, 6.0, 0.4, 0.1, 0.0, 4, "salpeter", 910)
    jobs = survey.parameter_grid(base, [0.35, 0.6], [0.0, 0.15], [0.0, 0.5, 0.9])  # 12 maps, different lattices and N*
    ref = []
    for j in jobs:
        with mlens.Mlens.from_config(j.cfg, j.lens_xy, j.lens_m) as h:
            c, m, st = h.shoot()
            ref.append((c.cpu(), m.cpu(), st))
    for k in (1, 3, 4):
        r = survey.run_survey(jobs, n_streams=k)
        assert r["n_streams"] == k and len(r["stats"]) == len(jobs)
        for (c, m, st), c2, m2, st2 in zip(ref, r["count"], r["mag"], r["stats"]):
            assert torch.equal(c, c2) and torch.equal(m, m2)  # same kernels, same tiles: bit-identical
            for key in ("rays_total", "rays_in_map", "rays_outside", "rays_lost", "max_count"):
                assert st[key] == st2[key], key
    # caller-owned numpy result buffers, counts only
    bufs = [np.empty((j.cfg.npix, j.cfg.npix), np.int32) for j in jobs]
    r = survey.run_survey(jobs, n_streams=2, want_mag=False, out_count=bufs)
    assert r["mag"] is None and all(np.array_equal(b, c.numpy()) for b, (c, _, _) in zip(bufs, ref))
