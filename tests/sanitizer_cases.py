"""Small invocations of every hand-written kernel, for `compute-sanitizer` (SURVEY.md §5 "race detection / sanitizers").

Not a pytest module (no test_ prefix): run ONE tool per gpurun call, as /opt/skills/guides/B200_PROFILING.md requires —

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py

Cases: (a) production shooting kernel, lens list resident as one chunk, every binning route, near-lens list in play;
(b) the same kernel streaming a 5000-lens list in double-buffered chunks (mbarrier phases, bulk copies); (c) near-list
overflow -> FP64 fallback; (d) mlens_mpd with more than 48 Ki bins (shared + global bins) and (e) mlens_index_map /
mlens_unindex_map; (f) the -DMLENS_ABLATIONS kernels (FP64, plain FP32, round-1 kernel) if that library is built.
Sizes are tiny: the tools slow kernels down by 10-1000x.  Each case checks its result so that a run is also a smoke test.
The summaries of the runs are kept under profiles/.
"""
import dataclasses
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1406_0559_b200 import fields, mlens  # noqa: E402


def case_single_chunk():
    cfg = dataclasses.replace(fields.CONFIGS[1], npix=64, sub=3)
    xy, m = fields.random_field(24, cfg.disc_radius, 3, "salpeter")
    maps = []
    with mlens.Mlens.from_config(cfg, xy, m) as h:
        for mode in (0, 1, 2, 3):
            h.set_option("binning", mode)
            count, mag, st = h.shoot()
            assert st["rays_in_map"] + st["rays_outside"] + st["rays_lost"] == st["rays_total"]
            maps.append(count.cpu().numpy().copy())
        out = h.shoot_block(3, 5, 70, 66, want_rays=True)
        assert out["pix"].shape == (66, 70)
    assert all(np.array_equal(maps[0], c) for c in maps[1:])
    return f"single chunk: {st['rays_total']} rays x 24 lenses, 4 binning routes identical"


def case_multi_chunk():
    cfg = fields.MapConfig("chunks", 64, 6.0, 0.55, 0.1, 0.0, 2, "salpeter", 31)
    xy, m = fields.random_field(5000, 60.0, 31, "salpeter")
    with mlens.Mlens.from_config(cfg, xy, m) as h:
        g = h.geometry
        cnt = torch.zeros((cfg.npix, cfg.npix), dtype=torch.int32, device="cuda")
        h.shoot_block(g.n1 // 2 - 64, g.n2 // 2 - 96, 128, 192, count=cnt)
        st = h.stats()
    assert st["rays_total"] == 128 * 192 and int(cnt.sum()) == st["rays_in_map"]
    return f"multi chunk: 128x192 rays x 5000 lenses (3 chunks of 2048), in_map {st['rays_in_map']}"


def case_near_overflow():
    L, npix, sub = 4.0, 32, 2
    u = fields.uniform01(99, 0, 2 * 60)
    cluster = np.stack([0.3 * (u[0::2] - 0.5), 0.3 * (u[1::2] - 0.5)], axis=1).astype(np.float32)
    m = np.full((60,), 0.05, np.float32)
    cfg = fields.MapConfig("overflow", npix, L, 0.2, 0.05, 0.0, sub, "unit", 0)
    with mlens.Mlens.from_config(cfg, cluster, m) as h:
        g = h.geometry
        cnt = torch.zeros((npix, npix), dtype=torch.int32, device="cuda")
        h.shoot_block(0, 0, g.n1, g.n2, count=cnt)
        st = h.stats()
    assert st["rays_total"] == g.n1 * g.n2
    return f"near-list overflow: {g.n1}x{g.n2} rays, 60 lenses inside one tile, in_map {st['rays_in_map']}"


def case_mpd_and_index():
    npix = 256
    u = fields.uniform01(7, 0, npix * npix)
    count = (u * u * 60000).astype(np.int32).reshape(npix, npix)  # > 48 Ki distinct bins in play: shared-memory bins + global 64-bit bins
    with mlens.Mlens(0.3, 0.2, 0.0, 4.0, npix, 4.0 / npix / 2, np.zeros((1, 2), np.float32)) as h:
        c = torch.from_numpy(count).cuda()
        n_bins = int(count.max()) + 2
        hist, ms = h.mpd(c, n_bins)
        assert np.array_equal(hist.cpu().numpy(), np.bincount(count.ravel(), minlength=n_bins))
        values, indexed = h.index_map(c)
        back = h.unindex_map(indexed, values.contiguous())
        assert torch.equal(back, c) and np.array_equal(values.cpu().numpy(), np.unique(count))
        mag = h.magnification(c)
        assert mag.shape == (npix, npix)
    return f"mpd ({n_bins} bins) + index_map ({values.numel()} distinct values) + magnification"


def case_ablation_kernels():
    if not os.path.exists(mlens.LIB_PATH_ABLATIONS):
        return "ablation kernels: library not built, skipped"
    cfg = dataclasses.replace(fields.CONFIGS[4], npix=64, sub=2)
    xy, m = fields.lens_field(cfg)
    res = {}
    with mlens.Mlens.from_config(cfg, xy, m, ablations=True) as h:
        g = h.geometry
        blk = (g.n1 // 2 - 64, g.n2 // 2 - 64, 128, 128)
        for kern in (1, 0, 2, 4):
            h.set_option("kernel", kern)
            cnt = torch.zeros((cfg.npix, cfg.npix), dtype=torch.int32, device="cuda")
            h.reset_stats()
            h.shoot_block(*blk, count=cnt)
            res[kern] = h.stats()["rays_in_map"]
            assert int(cnt.sum()) == res[kern]
    return f"kernels 1/0/2/4 on a 128x128 block x {len(m)} lenses: in_map {res}"


if __name__ == "__main__":
    torch.cuda.set_device(0)
    for case in (case_single_chunk, case_multi_chunk, case_near_overflow, case_mpd_and_index, case_ablation_kernels):
        print(case(), flush=True)
        torch.cuda.synchronize()
    print("sanitizer_cases: all cases ran", flush=True)
