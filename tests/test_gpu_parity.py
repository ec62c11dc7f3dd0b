"""GPU parity (P10): the CUDA path, through the C ABI, against the FP64 oracle on the same seeded inputs.

Tolerances are BASELINE.json north_star's:
  (i)   per ray and component |alpha_gpu - alpha_fp64| <= 2e-5 * sum_i m_i/|x - x_i|
        (checked on y: the macro term is formed identically on both sides, so delta-y = -delta-alpha);
  (ii)  pixel id bit-exact for every ray whose FP64 source position is > 1e-3 pixel from a pixel edge;
  (iii) map L1 difference <= 1e-4 of the rays landing in the map.
"""
import dataclasses

import numpy as np
import pytest

from paper_1406_0559_b200 import fields

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_ALPHA = 2e-5
EDGE_BAND = 1e-3
TOL_L1 = 1e-4
# a per-axis position error e (pixels) mis-bins a ray with probability |e| and each mis-binned ray adds 2
# to the L1, so L1/in_map ~ 4 E|e|; the 1e-4 budget therefore needs a MEAN |e| <= 2.5e-5 px.  Asserted below on the rays
# that land in the map (the ones the L1 is made of) and on the rays far from every lens (the FP32 loop alone).
TOL_MEAN_ERR_PX = 2.5e-5
MIN_IN_MAP_RAYS = 100_000  # per config: below this check (ii) and the L1 budget have no teeth (cfg 4 bins only 12 % of its rays)


@pytest.fixture(scope="module")
def ml():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1406_0559_b200 import mlens

    mlens.lib()
    mlens.lib(ablations=True)  # the -DMLENS_ABLATIONS build: debug / ablation kernels for the tests that name them
    return mlens


def _args(cfg):
    return (cfg.kappa, cfg.gamma, cfg.s, cfg.map_side, cfg.npix, cfg.ray_spacing)


def _far_from_every_lens(x, lens_xy, lens_m, tree):
    """Rays farther than rho_i = 0.5 sqrt(max(m_i, 1)) (the kernel's near-list radius) from their 4 nearest
    lenses: the population whose deflection comes from the FP32 loop alone."""
    k = min(4, len(lens_xy))
    if k == 0:
        return np.ones(x.shape[:-1], bool)
    dist, idx = tree.query(x.reshape(-1, 2), k=k)
    dist, idx = dist.reshape(-1, k), idx.reshape(-1, k)
    rho = 0.5 * np.sqrt(np.maximum(lens_m.astype(np.float64), 1.0))
    return (dist > rho[idx]).all(axis=1).reshape(x.shape[:-1])


def check_block(ml, oracle, h, cfg, xy, m, block, acc_gpu=None, acc_ref=None, tree=None):
    """Per-ray and per-block comparison; returns dict of counters for aggregation."""
    i0, j0, ni, nj = block
    cnt = torch.zeros((cfg.npix, cfg.npix), dtype=torch.int32, device="cuda")
    out = h.shoot_block(i0, j0, ni, nj, count=cnt, want_rays=True)
    # The same block again WITHOUT per-ray outputs: that launch takes the lean instantiation
    # shoot_fp32_kernel<..., BIN_RUNS> — the one mlens_shoot launches and bench.py times — whereas the launch above (per-ray
    # outputs wanted) takes the <..., -1> instantiation of the same source.  Same rays, same pixels: bit-identical maps, so
    # every element-wise comparison with the oracle below also holds for the benchmarked kernel.
    cnt_lean = torch.zeros((cfg.npix, cfg.npix), dtype=torch.int32, device="cuda")
    h.shoot_block(i0, j0, ni, nj, count=cnt_lean)
    torch.cuda.synchronize()
    assert torch.equal(cnt_lean, cnt), f"count-only (production) launch differs from the per-ray-output launch in block {block}"
    y_gpu = out["y"].cpu().numpy()
    pix_gpu = out["pix"].cpu().numpy()
    cnt_gpu = cnt_lean.cpu().numpy()
    ref = oracle.shoot_block(*_args(cfg), xy, m, block=block, want_rays=True)
    y_ref, pix_ref, scale = ref["y"], ref["pix"], ref["scale"]
    finite = np.isfinite(y_ref).all(axis=2)
    # (i) deflection tolerance
    dy = np.abs(y_gpu - y_ref)
    bound = TOL_ALPHA * scale[..., None] + 1e-12
    bad_alpha = int((dy[finite] > np.broadcast_to(bound, dy.shape)[finite]).sum())
    assert bad_alpha == 0, f"{bad_alpha} deflection components exceed 2e-5*sum(m/r) in block {block}"
    assert np.array_equal(pix_gpu == -2, ~finite)
    # (ii) pixel assignment away from edges
    u = (y_ref + cfg.map_side / 2.0) / cfg.pixel
    dist = np.abs(u - np.round(u)).min(axis=2)
    far_edge = finite & (dist > EDGE_BAND)
    mism_far = int((pix_gpu[far_edge] != pix_ref[far_edge]).sum())
    assert mism_far == 0, f"{mism_far} rays > 1e-3 px from an edge got a different pixel in block {block}"
    mism_all = int((pix_gpu != pix_ref).sum())
    # block map == histogram of the block's own pixel ids (binning is exact integer work)
    hist = np.bincount(pix_gpu[pix_gpu >= 0].ravel(), minlength=cfg.npix**2).reshape(cfg.npix, cfg.npix)
    assert np.array_equal(hist, cnt_gpu)
    if acc_gpu is not None:
        acc_gpu += cnt_gpu
        acc_ref += ref["count"]
    # position error in pixels, per component, by population
    err = dy / cfg.pixel
    in_map = pix_ref >= 0
    res = {"rays": ni * nj, "in_map": ref["stats"]["rays_in_map"], "mismatch": mism_all,
           "l1": int(np.abs(cnt_gpu.astype(np.int64) - ref["count"]).sum()),
           "err_sum_in_map": float(err[in_map].sum()), "err_n_in_map": 2 * int(in_map.sum()),
           "err_max_in_map": float(err[in_map].max()) if in_map.any() else 0.0,
           "mean_err_px": float(err[finite].mean()) if finite.any() else 0.0,
           "max_err_px": float(err[finite].max()) if finite.any() else 0.0}
    if tree is not None:
        g = h.geometry
        ii, jj = np.meshgrid(np.arange(i0, i0 + ni), np.arange(j0, j0 + nj))
        x = np.stack([(ii + 0.5 - g.n1 / 2.0) * cfg.ray_spacing, (jj + 0.5 - g.n2 / 2.0) * cfg.ray_spacing], axis=-1)
        far = _far_from_every_lens(x, xy, m, tree) & finite
        near = finite & ~far
        res.update(err_sum_far=float(err[far].sum()), err_n_far=2 * int(far.sum()),
                   err_sum_near=float(err[near].sum()), err_n_near=2 * int(near.sum()),
                   err_max_near=float(err[near].max()) if near.any() else 0.0)
    return res


# ---------------------------------------------------------------------------------------------------------------
# closed forms and edge cases through the CUDA path
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel", [1, 0])
def test_no_lens_uniform_map_is_exact(ml, oracle, kernel):
    # P1(b) through the GPU: kappa=0.3, gamma=0.2, all smooth: counts {220, 240}, mean 222.5 — exact integers
    L, npix, sub = 4.0, 64, 10
    with ml.Mlens(0.3, 0.2, 1.0, L, npix, L / npix / sub, np.zeros((0, 2), np.float32), ablations=kernel != 1) as h:
        h.set_option("kernel", kernel)
        count, mag, st = h.shoot()
    c = count.cpu().numpy()
    assert set(np.unique(c).tolist()) == {220, 240} and c.mean() == 222.5
    ref = oracle.shoot_block(0.3, 0.2, 1.0, L, npix, L / npix / sub, np.zeros((0, 2), np.float32), None)
    assert np.array_equal(c, ref["count"])
    assert st["rays_total"] == ref["stats"]["rays_total"] and st["rays_in_map"] == ref["stats"]["rays_in_map"]
    assert st["rays_lost"] == 0 and st["max_count"] == 240
    assert np.array_equal(mag.cpu().numpy(), oracle.magnification(c, 100.0))


def test_tiny_config_full_map(ml, oracle):
    # configs[0]: the whole map against the oracle (2.1e7 rays, 13 lenses; ragged n2 = 3414 = 53*64 + 22)
    cfg = fields.CONFIGS[1]
    xy, m = fields.lens_field(cfg)
    with ml.Mlens.from_config(cfg, xy, m) as h:
        assert (h.geometry.n1, h.geometry.n2) == (6144, 3414)
        count, mag, st = h.shoot()
        host_count, host_mag, host_st = h.shoot_host()
        pin_c = torch.empty((cfg.npix, cfg.npix), dtype=torch.int32, pin_memory=True)
        pin_m = torch.empty((cfg.npix, cfg.npix), dtype=torch.float32, pin_memory=True)
        h.shoot_host(count=pin_c.numpy(), mag=pin_m.numpy())  # caller-owned (pinned) result buffers
        assert np.array_equal(pin_c.numpy(), host_count) and np.array_equal(pin_m.numpy(), host_mag)
    ref = oracle.shoot_block(*_args(cfg), xy, m)
    c = count.cpu().numpy()
    l1 = int(np.abs(c.astype(np.int64) - ref["count"]).sum())
    assert st["rays_total"] == ref["stats"]["rays_total"] == 6144 * 3414
    assert st["rays_in_map"] + st["rays_outside"] + st["rays_lost"] == st["rays_total"]
    assert int(c.sum(dtype=np.int64)) == st["rays_in_map"]
    assert abs(st["rays_in_map"] - ref["stats"]["rays_in_map"]) <= l1
    assert l1 <= TOL_L1 * ref["stats"]["rays_in_map"], (l1, ref["stats"]["rays_in_map"])
    assert st["max_count"] == int(c.max())
    assert np.array_equal(mag.cpu().numpy(), oracle.magnification(c, ref["geometry"].n_avg))
    # host-buffer entry point gives the same map (integer REDs: order-independent => deterministic)
    assert np.array_equal(host_count, c) and np.array_equal(host_mag, mag.cpu().numpy())
    assert host_st["rays_in_map"] == st["rays_in_map"]


def test_ragged_and_degenerate_blocks(ml, oracle):
    cfg = dataclasses.replace(fields.CONFIGS[1], npix=128, sub=6)
    xy, m = fields.random_field(40, cfg.disc_radius, 5, "salpeter")
    with ml.Mlens.from_config(cfg, xy, m) as h:
        n1, n2 = h.geometry.n1, h.geometry.n2
        blocks = [(0, 0, 1, 1), (n1 - 1, n2 - 1, 1, 1), (3, 5, 64, 64), (7, 11, 65, 63), (0, 0, 200, 3), (n1 - 130, 0, 130, 257),
                  (0, n2 - 77, n1, 77), (n1 // 2 - 100, n2 // 2 - 100, 201, 199)]
        for b in blocks:
            r = check_block(ml, oracle, h, cfg, xy, m, b)
            assert r["l1"] <= max(2, 2 * r["mismatch"])
        # empty block: no work, no error; out-of-range block: EINVAL
        h.shoot_block(5, 5, 0, 0)
        with pytest.raises(ml.MlensError):
            h.shoot_block(0, 0, n1 + 1, 1)
        with pytest.raises(ml.MlensError):
            h.shoot_block(-1, 0, 1, 1)


def test_ray_exactly_on_a_lens_is_lost(ml, oracle):
    L, npix, sub = 4.0, 16, 2
    d = L / npix / sub
    g = oracle.geometry(0.0, 0.0, 0.0, L, npix, d)
    x_on_ray = np.array([[(5 + 0.5 - g.n1 / 2) * d, (9 + 0.5 - g.n2 / 2) * d]], np.float32)
    with ml.Mlens(0.0, 0.0, 0.0, L, npix, d, x_on_ray) as h:
        count, _, st = h.shoot()
        out = h.shoot_block(0, 0, g.n1, g.n2, want_rays=True)
    ref = oracle.shoot_block(0.0, 0.0, 0.0, L, npix, d, x_on_ray, None, want_rays=True)
    assert st["rays_lost"] == ref["stats"]["rays_lost"] == 1
    assert out["pix"].cpu().numpy()[9, 5] == -2
    assert np.array_equal(count.cpu().numpy(), ref["count"])


def test_multi_chunk_lens_list(ml, oracle):
    # N* > 3072 streams the list through shared memory in 2048-lens chunks (double-buffered bulk copies)
    cfg = fields.MapConfig("chunks", 128, 6.0, 0.55, 0.1, 0.0, 4, "salpeter", 31)
    xy, m = fields.random_field(5000, 60.0, 31, "salpeter")
    with ml.Mlens.from_config(cfg, xy, m) as h:
        n1, n2 = h.geometry.n1, h.geometry.n2
        tot = {"in_map": 0, "l1": 0}
        for b in [(0, 0, 256, 192), (n1 // 2 - 128, n2 // 2 - 96, 256, 192), (n1 - 200, n2 - 130, 200, 130)]:
            r = check_block(ml, oracle, h, cfg, xy, m, b)
            tot["in_map"] += r["in_map"]; tot["l1"] += r["l1"]
    assert tot["l1"] <= max(4, TOL_L1 * tot["in_map"])


def test_multi_chunk_whole_map_through_mlens_shoot(ml, oracle):
    # The production launch (mlens_shoot: count-only, run-combining REDs) with a list that is streamed in chunks
    # (N* = 5000 > 3072: three 2048-lens chunks, the config-2 code path), whole map against the oracle, L1 <= 1e-4.
    cfg = fields.MapConfig("chunks", 96, 6.0, 0.55, 0.1, 0.0, 3, "salpeter", 31)
    xy, m = fields.random_field(5000, 60.0, 31, "salpeter")
    with ml.Mlens.from_config(cfg, xy, m) as h:
        count, mag, st = h.shoot()
        c = count.cpu().numpy()
        mag_gpu = mag.cpu().numpy()
        n_avg = h.geometry.n_avg
    ref = oracle.shoot_block(*_args(cfg), xy, m)
    in_map = ref["stats"]["rays_in_map"]
    assert st["rays_total"] == ref["stats"]["rays_total"] and in_map > 100_000
    l1 = int(np.abs(c.astype(np.int64) - ref["count"]).sum())
    assert l1 <= max(4, TOL_L1 * in_map), (l1, in_map)
    assert int(c.sum()) == st["rays_in_map"] and st["rays_in_map"] + st["rays_outside"] + st["rays_lost"] == st["rays_total"]
    assert np.array_equal(mag_gpu, oracle.magnification(c, n_avg))


def test_binning_variants_and_fp64_kernel_agree(ml, oracle):
    cfg = dataclasses.replace(fields.CONFIGS[1], npix=192, sub=5)
    xy, m = fields.lens_field(cfg)
    maps = {}
    with ml.Mlens.from_config(cfg, xy, m, ablations=True) as h:
        for mode in (0, 1, 2, 3):
            h.set_option("binning", mode)
            count, _, st = h.shoot(want_mag=False)
            maps[mode] = (count.cpu().numpy().copy(), st)
        h.set_option("kernel", 0)
        c64, _, st64 = h.shoot(want_mag=False)
        c64 = c64.cpu().numpy()
    for mode in (1, 2, 3):  # same per-ray pixels, different routes to the map: bit-identical
        assert np.array_equal(maps[mode][0], maps[0][0]), mode
        assert maps[mode][1]["rays_in_map"] == maps[0][1]["rays_in_map"]
    ref = oracle.shoot_block(*_args(cfg), xy, m)
    in_map = ref["stats"]["rays_in_map"]
    assert np.abs(c64.astype(np.int64) - ref["count"]).sum() <= max(2, 1e-6 * in_map)  # FP64 kernel ~ oracle
    assert np.abs(maps[1][0].astype(np.int64) - ref["count"]).sum() <= TOL_L1 * in_map


@pytest.mark.parametrize("rays,tile_x,shared_pairs", [(16, 64, 0), (16, 64, 1), (16, 64, 2), (16, 64, 3), (16, 64, 4), (8, 64, 0),
                                                      (8, 64, 1), (8, 64, 2), (8, 64, 4), (8, 48, 0), (8, 48, 2), (8, 32, 1)])
def test_kernel_variants_meet_the_tolerances(ml, oracle, rays, tile_x, shared_pairs):
    # every instantiation of the production kernel's sweep grid (rays per thread x tile width x ray pairs per lens whose two
    # reciprocals come from one MUFU.RCP) must hold P10; random + lens-centred + in-map blocks of cfg 4, ragged against all
    # three tile widths
    cfg = fields.CONFIGS[4]
    xy, m = fields.lens_field(cfg)
    with ml.Mlens.from_config(cfg, xy, m, ablations=True) as h:
        h.set_option("rays_per_thread", rays)
        h.set_option("tile_x", tile_x)
        h.set_option("shared_pairs", shared_pairs)
        g = h.geometry
        blocks = fields.block_plan(g.n1, g.n2, xy, cfg.half_widths, cfg.ray_spacing, cfg.seed + 17, 3, 3, 0, size=200,
                                   n_straddle=0, n_inside=2, map_half_image=cfg.map_half_image)
        tot = {"in_map": 0, "l1": 0}
        for b in blocks:
            r = check_block(ml, oracle, h, cfg, xy, m, b)
            tot["in_map"] += r["in_map"]; tot["l1"] += r["l1"]
    assert tot["in_map"] > 20000 and tot["l1"] <= max(2, TOL_L1 * tot["in_map"]), tot


def test_far_lens_and_tiny_spacing_take_the_one_reciprocal_path(ml, oracle):
    # shared reciprocals multiply two squared distances in lattice units (lengths / d): a lens 2e4 R_E away with d = 1e-6
    # gives r^2 ~ 4e20 and a product beyond FP32, so the library must fall back to one MUFU.RCP per ray — and still match
    L, npix = 1.0e-3, 16
    d = 1.0e-6
    xy = np.array([[20000.0, 5000.0], [-3.0, 1.0], [0.5, -0.25]], np.float32)
    m = np.array([4.0, 1.0, 0.5], np.float32)
    cfg = fields.MapConfig("far", npix, L, 0.3, 0.1, 0.0, 1, "unit", 0)
    with ml.Mlens(0.3, 0.1, 0.0, L, npix, d, xy, m) as h:
        g = h.geometry
        for b in [(0, 0, 130, 70), (g.n1 // 2 - 100, g.n2 // 2 - 100, 200, 200)]:
            i0, j0, ni, nj = b
            out = h.shoot_block(i0, j0, ni, nj, want_rays=True)
            ref = oracle.shoot_block(0.3, 0.1, 0.0, L, npix, d, xy, m, block=b, want_rays=True)
            assert np.abs(out["y"].cpu().numpy() - ref["y"]).max() <= 2e-5 * ref["scale"].min()
            assert (out["pix"].cpu().numpy() != ref["pix"]).sum() <= 2


@pytest.mark.parametrize("shared", [0, 1])
def test_round_1_kernel_still_meets_the_tolerances(ml, oracle, shared):
    # "kernel" 4: the round-1 production kernel, kept in the ablations library as the A/B baseline of the timings
    cfg = fields.CONFIGS[5]
    xy, m = fields.lens_field(cfg)
    with ml.Mlens.from_config(cfg, xy, m, ablations=True) as h:
        h.set_option("kernel", 4)
        h.set_option("shared_rcp", shared)
        g = h.geometry
        blocks = fields.block_plan(g.n1, g.n2, xy, cfg.half_widths, cfg.ray_spacing, cfg.seed + 19, 2, 2, 1, size=200,
                                   n_straddle=0, n_inside=2, map_half_image=cfg.map_half_image)
        tot = {"in_map": 0, "l1": 0}
        for b in blocks:
            r = check_block(ml, oracle, h, cfg, xy, m, b)
            tot["in_map"] += r["in_map"]; tot["l1"] += r["l1"]
    assert tot["in_map"] > 20000 and tot["l1"] <= max(2, TOL_L1 * tot["in_map"]), tot


def test_near_list_overflow_falls_back_to_fp64(ml, oracle):
    # more lenses within rho of one tile than the near list holds (32): those tiles take Eq. 1 in plain FP64
    L, npix, sub = 4.0, 64, 4
    d = L / npix / sub
    u = fields.uniform01(99, 0, 2 * 60)
    cluster = np.stack([0.3 * (u[0::2] - 0.5), 0.3 * (u[1::2] - 0.5)], axis=1)  # 60 lenses inside a 0.3 x 0.3 box
    far, _ = fields.random_field(20, 6.0, 98)
    xy = np.concatenate([cluster.astype(np.float32), far])
    m = np.full((len(xy),), 0.05, np.float32)
    cfg = fields.MapConfig("overflow", npix, L, 0.2, 0.05, 0.0, sub, "unit", 0)
    with ml.Mlens.from_config(cfg, xy, m) as h:
        g = h.geometry
        for b in [(g.n1 // 2 - 96, g.n2 // 2 - 96, 192, 192), (0, 0, 130, 70)]:
            r = check_block(ml, oracle, h, cfg, xy, m, b)
            assert r["l1"] <= max(2, 2 * r["mismatch"]) and r["mismatch"] <= 2


@pytest.mark.parametrize("case", range(12))
def test_seeded_random_small_maps_against_the_oracle(ml, oracle, case):
    # whole small maps with seeded random parameters: both parities of both macro factors (kappa + gamma > 1: saddle /
    # over-focused images), negative shear, all-smooth and no-smooth matter, unit and Salpeter masses, maps narrower than
    # one tile, lens counts from 0 to a few hundred
    u = fields.uniform01(9000 + case, 0, 16)
    kappa = [0.2, 0.45, 0.7, 1.3, 1.6, 0.9][case % 6] + 0.05 * u[0]
    gamma = (0.6 * u[1] - 0.3) if case % 3 else (0.5 + 0.4 * u[1])
    if abs(1 - kappa - gamma) < 0.05 or abs(1 - kappa + gamma) < 0.05:
        gamma += 0.11
    s = [0.0, 0.3, 1.0, 0.8][case % 4]
    npix = [24, 40, 64, 17][case % 4]
    sub = [3, 2, 4, 5][(case // 2) % 4]
    L = [2.0, 6.0, 1.0][case % 3]
    n_lens = 0 if s == 1.0 else [3, 40, 150, 12][case % 4]
    masses = "salpeter" if case % 2 else "unit"
    cfg = fields.MapConfig(f"rnd{case}", npix, L, kappa, gamma, s, sub, masses, 9100 + case)
    xy, m = fields.random_field(n_lens, max(cfg.disc_radius, 1.0), 9100 + case, masses)
    with ml.Mlens.from_config(cfg, xy, m) as h:
        count, mag, st = h.shoot()
        c = count.cpu().numpy().astype(np.int64)
        g = h.geometry
    ref = oracle.shoot_block(*_args(cfg), xy, m)
    rs = ref["stats"]
    l1 = int(np.abs(c - ref["count"]).sum())
    assert (g.n1, g.n2) == (ref["geometry"].n1, ref["geometry"].n2)
    assert st["rays_total"] == rs["rays_total"] == g.n1 * g.n2 and st["rays_lost"] == rs["rays_lost"]
    assert st["rays_in_map"] + st["rays_outside"] + st["rays_lost"] == st["rays_total"]
    assert l1 <= max(2, TOL_L1 * rs["rays_in_map"]), (case, kappa, gamma, s, l1, rs)
    assert abs(st["rays_in_map"] - rs["rays_in_map"]) <= l1
    assert np.array_equal(mag.cpu().numpy(), oracle.magnification(c.astype(np.int32), g.n_avg))


def test_mirror_symmetry_on_gpu(ml):
    # P6 through the CUDA path
    cfg = dataclasses.replace(fields.CONFIGS[1], npix=128, sub=6)
    xy, m = fields.random_field(30, cfg.disc_radius, 9, "salpeter")
    xm = xy.copy(); xm[:, 0] = -xm[:, 0]
    with ml.Mlens.from_config(cfg, xy, m) as h:
        a, _, st = h.shoot(want_mag=False)
    with ml.Mlens.from_config(cfg, xm, m) as h:
        b, _, _ = h.shoot(want_mag=False)
    a, b = a.cpu().numpy().astype(np.int64), b.cpu().numpy().astype(np.int64)
    assert np.abs(a - b[:, ::-1]).sum() <= 2e-4 * st["rays_in_map"]


# ---------------------------------------------------------------------------------------------------------------
# the five configurations: seeded sub-blocks (random, lens-centred, border) + full-map invariants
# ---------------------------------------------------------------------------------------------------------------
# SURVEY.md §8(d) "Sub-block parity plan (P10)": K = 64 blocks of 256 x 256 rays per config — seeded random unaligned
# blocks (24 anywhere + 8 inside the map's macro pre-image = 32), 16 centred on lenses, 8 on the lattice border, 8 whose
# macro-image straddles the map edge.
N_BLOCKS = dict(n_random=24, n_lens_centred=16, n_border=8, n_straddle=8, n_inside=8)


@pytest.mark.parametrize("cfg_id", [1, 2, 3, 4, 5])
def test_config_sub_blocks(ml, oracle, cfg_id):
    from scipy.spatial import cKDTree

    cfg = fields.CONFIGS[cfg_id]
    xy, m = fields.lens_field(cfg)
    tree = cKDTree(xy.astype(np.float64))
    with ml.Mlens.from_config(cfg, xy, m) as h:
        g = h.geometry
        blocks = fields.block_plan(g.n1, g.n2, xy, cfg.half_widths, cfg.ray_spacing, cfg.seed, size=256,
                                   map_half_image=cfg.map_half_image, **N_BLOCKS)
        assert len(blocks) == 64
        acc_gpu = np.zeros((cfg.npix, cfg.npix), np.int64)
        acc_ref = np.zeros((cfg.npix, cfg.npix), np.int64)
        tot = {}
        for b in blocks:
            r = check_block(ml, oracle, h, cfg, xy, m, b, acc_gpu, acc_ref, tree)
            for k, v in r.items():
                tot[k] = max(tot.get(k, 0.0), v) if "max" in k else tot.get(k, 0) + v
    l1 = int(np.abs(acc_gpu - acc_ref).sum())
    mean_in = tot["err_sum_in_map"] / max(1, tot["err_n_in_map"])
    mean_far = tot["err_sum_far"] / max(1, tot["err_n_far"])
    mean_near = tot["err_sum_near"] / max(1, tot["err_n_near"])
    print(f"cfg{cfg_id}: {len(blocks)} blocks, {tot['rays']} rays, in_map {tot['in_map']}, pixel mismatches {tot['mismatch']}, "
          f"L1 {l1} ({l1 / max(1, tot['in_map']):.2e}); mean|err| in-map {mean_in:.2e} px (max {tot['err_max_in_map']:.2e}), "
          f"far from lenses {mean_far:.2e} px ({tot['err_n_far'] // 2} rays), near a lens {mean_near:.2e} px "
          f"({tot['err_n_near'] // 2} rays, max {tot['err_max_near']:.2e}); max over all rays {tot['max_err_px']:.2e} px")
    assert tot["in_map"] >= MIN_IN_MAP_RAYS, tot["in_map"]
    assert l1 <= TOL_L1 * tot["in_map"], (l1, tot)
    assert mean_in <= TOL_MEAN_ERR_PX and mean_far <= TOL_MEAN_ERR_PX, (mean_in, mean_far)
    assert tot["err_max_in_map"] < EDGE_BAND  # criterion (ii) can only hold if no in-map ray is off by the band's width


def test_config_3_band_l1_against_the_oracle(ml, oracle):
    # SURVEY.md §8(d) asks for the full-map L1 of cfg 3 against the oracle (4.2e12 interactions: ~6 min of oracle on 16
    # host cores — too long for the test budget).  Taken instead on a contiguous 1/8-lattice band of whole rows around the
    # lattice centre (196608 x 6144 rays = 1.2e9 rays, 5.2e11 interactions, ~45 s of oracle), accumulated into a map
    # (DESIGN.md "Parity plan").
    cfg = fields.CONFIGS[3]
    xy, m = fields.lens_field(cfg)
    with ml.Mlens.from_config(cfg, xy, m) as h:
        g = h.geometry
        nj = g.n2 // 8
        j0 = (g.n2 // 2 - nj // 2) // 64 * 64
        cnt = torch.zeros((cfg.npix, cfg.npix), dtype=torch.int32, device="cuda")
        h.reset_stats()
        h.shoot_block(0, j0, g.n1, nj, count=cnt)
        st = h.stats()
        c = cnt.cpu().numpy().astype(np.int64)
    ref = oracle.shoot_block(*_args(cfg), xy, m, block=(0, j0, g.n1, nj))
    rs = ref["stats"]
    l1 = int(np.abs(c - ref["count"]).sum())
    print(f"cfg3 band rows [{j0}, {j0 + nj}): {rs['rays_total']} rays, in_map {rs['rays_in_map']} (gpu {st['rays_in_map']}), L1 {l1} "
          f"({l1 / rs['rays_in_map']:.2e})")
    assert st["rays_total"] == rs["rays_total"] == g.n1 * nj and rs["rays_in_map"] > 1e8
    assert st["rays_lost"] == rs["rays_lost"] and abs(st["rays_in_map"] - rs["rays_in_map"]) <= l1
    assert l1 <= TOL_L1 * rs["rays_in_map"]


@pytest.mark.parametrize("cfg_id", [2, 3, 4, 5])
def test_full_map_invariants(ml, oracle, cfg_id):
    # the launch configuration bench.py times: whole lattice, default options
    cfg = fields.CONFIGS[cfg_id]
    xy, m = fields.lens_field(cfg)
    with ml.Mlens.from_config(cfg, xy, m) as h:
        g = h.geometry
        count, mag, st = h.shoot()
        assert st["rays_total"] == g.n1 * g.n2
        assert st["rays_in_map"] + st["rays_outside"] + st["rays_lost"] == st["rays_total"]
        assert int(count.sum(dtype=torch.int64).item()) == st["rays_in_map"]
        assert st["max_count"] == int(count.max().item()) and st["max_count"] < 2**31 - 1
        # magnification: bit-exact Eq. 4 on sampled pixels
        idx = (fields.uniform01(cfg.seed + 5, 0, 4096) * cfg.npix**2).astype(np.int64)
        c_s = count.view(-1)[torch.from_numpy(idx).cuda()].cpu().numpy()
        m_s = mag.view(-1)[torch.from_numpy(idx).cuda()].cpu().numpy()
        assert np.array_equal(m_s, oracle.magnification(c_s, g.n_avg))
        # sampled rays, one by one, against the oracle: per-ray pixel ids via 1x1 blocks are too slow; use 64 8x8 blocks
        u = fields.uniform01(cfg.seed + 6, 0, 128)
        mism = 0
        for k in range(64):
            i0, j0 = int(u[2 * k] * (g.n1 - 8)), int(u[2 * k + 1] * (g.n2 - 8))
            r = check_block(ml, oracle, h, cfg, xy, m, (i0, j0, 8, 8))
            mism += r["mismatch"]
        assert mism <= 2
    mean_mu = st["rays_in_map"] / (cfg.npix**2 * cfg.sub**2)
    print(f"cfg{cfg_id}: full map {st['elapsed_ms']:.1f} ms, <mu>/mu_th = {mean_mu / cfg.mu_th:.4f}, max count {st['max_count']}")
    if cfg_id in (3, 5):
        assert abs(mean_mu / cfg.mu_th - 1) < 0.15


def test_config_1_full_map_against_the_oracle(ml, oracle):
    # the one BASELINE.json config whose whole lattice the oracle shoots in about a second: full-map L1, all counters
    cfg = fields.CONFIGS[1]
    xy, m = fields.lens_field(cfg)
    with ml.Mlens.from_config(cfg, xy, m) as h:
        count, mag, st = h.shoot()
        count = count.cpu().numpy().astype(np.int64)
        mag = mag.cpu().numpy()
        g = h.geometry
    ref = oracle.shoot_block(*_args(cfg), xy, m)
    rs = ref["stats"]
    assert st["rays_total"] == rs["rays_total"] == g.n1 * g.n2
    l1 = int(np.abs(count - ref["count"]).sum())
    print(f"cfg1 full map: in_map {st['rays_in_map']} (oracle {rs['rays_in_map']}), L1 {l1}, lost {st['rays_lost']}")
    assert l1 <= TOL_L1 * rs["rays_in_map"]
    assert abs(st["rays_in_map"] - rs["rays_in_map"]) <= l1 and st["rays_lost"] == rs["rays_lost"]
    assert np.array_equal(mag, oracle.magnification(count.astype(np.int32), g.n_avg))


def test_whole_lattice_production_kernel_against_the_fp64_kernel(ml):
    # CUDA against CUDA, so no parity credit — but it is the one affordable check that NO tile position of a whole
    # multi-million-tile lattice misbehaves: cfg 3's full map (9.7e9 rays, 2.4e6 tiles) through the production kernel and
    # through the plain FP64 one-ray-per-thread kernel (itself held to 1e-6 of the oracle on small maps, above)
    cfg = fields.CONFIGS[3]
    xy, m = fields.lens_field(cfg)
    with ml.Mlens.from_config(cfg, xy, m, ablations=True) as h:
        a, _, sa = h.shoot(want_mag=False)
        a = a.clone()
        h.set_option("kernel", 0)
        b, _, sb = h.shoot(want_mag=False)
        l1 = int((a.to(torch.int64) - b.to(torch.int64)).abs().sum().item())
    print(f"cfg3 whole lattice: production {sa['elapsed_ms']:.0f} ms, FP64 kernel {sb['elapsed_ms']:.0f} ms, in_map {sa['rays_in_map']} / "
          f"{sb['rays_in_map']}, L1 {l1} ({l1 / sb['rays_in_map']:.2e})")
    assert sa["rays_total"] == sb["rays_total"] == 196608 * 49152 and sa["rays_lost"] == sb["rays_lost"]
    assert l1 <= TOL_L1 * sb["rays_in_map"] and abs(sa["rays_in_map"] - sb["rays_in_map"]) <= l1


def test_plain_fp32_ablation_fails_the_tolerances(ml, oracle):
    # "kernel" 2 sums Eq. 1 in plain FP32 in global coordinates (no difference form).  It is the evidence for
    # same blocks, same oracle — the plain form misses the L1 budget that the production
    # kernel meets with room to spare.  (The deflection tolerance (i) alone is loose enough for plain FP32.)
    cfg = fields.CONFIGS[4]
    xy, m = fields.lens_field(cfg)
    res = {}
    with ml.Mlens.from_config(cfg, xy, m, ablations=True) as h:
        g = h.geometry
        blocks = fields.block_plan(g.n1, g.n2, xy, cfg.half_widths, cfg.ray_spacing, cfg.seed + 23, 4, 2, 0, size=192)
        for kern in (1, 2):
            h.set_option("kernel", kern)
            l1 = in_map = 0
            err = []
            for b in blocks:
                cnt = torch.zeros((cfg.npix, cfg.npix), dtype=torch.int32, device="cuda")
                out = h.shoot_block(*b, count=cnt, want_rays=True)
                ref = oracle.shoot_block(*_args(cfg), xy, m, block=b, want_rays=True)
                l1 += int(np.abs(cnt.cpu().numpy().astype(np.int64) - ref["count"]).sum())
                in_map += ref["stats"]["rays_in_map"]
                err.append(np.abs(out["y"].cpu().numpy() - ref["y"]).max() / cfg.pixel)
            res[kern] = (l1 / max(1, in_map), max(err))
    print(f"cfg4 ablation: difference form L1/in_map {res[1][0]:.2e} (max |dy| {res[1][1]:.2e} px); "
          f"plain FP32 L1/in_map {res[2][0]:.2e} (max |dy| {res[2][1]:.2e} px)")
    assert res[1][0] <= TOL_L1
    assert res[2][0] > 10 * TOL_L1 and res[2][0] > 20 * max(res[1][0], 1e-6)


def test_shipped_library_refuses_the_ablation_kernels(ml):
    # libmlens.so (no -DMLENS_ABLATIONS) holds the production kernel only: the public ABI cannot select a kernel that
    # misses the parity tolerances
    cfg = dataclasses.replace(fields.CONFIGS[1], npix=64, sub=2)
    xy, m = fields.lens_field(cfg)
    with ml.Mlens.from_config(cfg, xy, m) as h:
        for key, value in (("kernel", 0), ("kernel", 2), ("kernel", 4), ("shared_rcp", 1), ("rays_per_thread", 8),
                           ("tile_x", 48), ("shared_pairs", 1)):
            with pytest.raises(ml.MlensError) as e:
                h.set_option(key, value)
            assert e.value.code == ml.EINVAL
        h.set_option("kernel", 1)
        h.set_option("binning", 2)


def test_two_streams_on_one_handle(ml, oracle):
    # mlens.h "Concurrency": shoot_block launches of one handle may overlap on different streams (each launch owns its
    # dynamic tile counter).  Two half-lattice launches on two streams, repeated, must give the single-launch map.
    cfg = dataclasses.replace(fields.CONFIGS[4], npix=256, sub=3)
    xy, m = fields.lens_field(cfg)
    with ml.Mlens.from_config(cfg, xy, m) as h:
        g = h.geometry
        full, _, st_full = h.shoot(want_mag=False)
        full = full.clone()
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        half = (g.n2 // 2) // 64 * 64
        for _ in range(3):
            cnt = torch.zeros_like(full)
            torch.cuda.synchronize()
            h.reset_stats()
            torch.cuda.synchronize()
            h.shoot_block(0, 0, g.n1, half, count=cnt, stream=s1)
            h.shoot_block(0, half, g.n1, g.n2 - half, count=cnt, stream=s2)
            torch.cuda.synchronize()
            st = h.stats()
            assert st["rays_total"] == g.n1 * g.n2 and st["rays_in_map"] == st_full["rays_in_map"]
            assert torch.equal(cnt, full)


def test_more_launches_in_flight_than_tile_counter_slots(ml):
    # The ring of per-launch tile counters has 256 slots.  600 four-row launches dealt to two streams with no host
    # synchronisation in between: launch n + 256 waits (on the device) for launch n, so no live counter is re-zeroed —
    # a re-zeroed counter would hand tiles out twice and the summed map would exceed the single-launch map.
    cfg = dataclasses.replace(fields.CONFIGS[4], npix=128, sub=5, map_side=12.0)
    xy, m = fields.lens_field(cfg)
    with ml.Mlens.from_config(cfg, xy, m) as h:
        g = h.geometry
        assert g.n2 >= 600 * 4
        full = torch.zeros((cfg.npix, cfg.npix), dtype=torch.int32, device="cuda")
        h.reset_stats()
        h.shoot_block(0, 0, g.n1, 600 * 4, count=full)
        torch.cuda.synchronize()
        st_full = h.stats()
        cnt = torch.zeros_like(full)
        h.reset_stats()
        torch.cuda.synchronize()
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        for k in range(600):
            h.shoot_block(0, 4 * k, g.n1, 4, count=cnt, stream=streams[k % 2])
        torch.cuda.synchronize()
        st = h.stats()
        assert st["rays_total"] == st_full["rays_total"] == g.n1 * 600 * 4
        assert abs(st["rays_in_map"] - st_full["rays_in_map"]) <= max(4, TOL_L1 * st_full["rays_in_map"])
        # rows 4k..4k+3 of a launch are not tile-aligned with the single launch's 64-row tiles: the maps agree to the
        # parity tolerance, and ray conservation is exact
        l1 = int((cnt.long() - full.long()).abs().sum().item())
        assert l1 <= max(4, TOL_L1 * st_full["rays_in_map"]), l1
        assert int(cnt.sum().item()) == st["rays_in_map"]


def test_shipped_library_one_reciprocal_per_ray_option(ml, oracle):
    # the shipped library's two instantiations (two shared ray pairs — the default — and one MUFU.RCP per ray, which is also
    # the automatic fallback for extreme coordinates) through the public option, both against the oracle
    cfg = dataclasses.replace(fields.CONFIGS[4], npix=200, sub=3)
    xy, m = fields.lens_field(cfg)
    ref = oracle.shoot_block(*_args(cfg), xy, m)
    maps = {}
    with ml.Mlens.from_config(cfg, xy, m) as h:
        for sp in (2, 0):
            h.set_option("shared_pairs", sp)
            c, _, st = h.shoot(want_mag=False)
            maps[sp] = c.cpu().numpy().astype(np.int64)
            l1 = int(np.abs(maps[sp] - ref["count"]).sum())
            assert st["rays_total"] == ref["stats"]["rays_total"] and l1 <= max(2, TOL_L1 * ref["stats"]["rays_in_map"]), (sp, l1)
    assert np.abs(maps[0] - maps[2]).sum() <= max(4, 2 * TOL_L1 * ref["stats"]["rays_in_map"])


def test_spacing_below_the_fp32_range_is_refused(ml):
    # lattice units divide every length by d: lens distances / d beyond ~2e18 would overflow |w|^2 in FP32 -> MLENS_ERANGE
    # from the launch (never a silently wrong map)
    xy = np.array([[3.0e5, 0.0]], np.float32)
    with ml.Mlens(0.3, 0.1, 0.0, 1.0e-12, 4, 1.0e-14, xy) as h:
        with pytest.raises(ml.MlensError) as e:
            h.shoot()
        assert e.value.code == ml.ERANGE


def test_handles_recycle_pooled_memory_and_trim(ml):
    # device blocks of destroyed handles stay in the library's pool and are reused; mlens_trim_memory returns them
    cfg = dataclasses.replace(fields.CONFIGS[1], npix=512, sub=2)
    xy, m = fields.lens_field(cfg)
    torch.cuda.synchronize()
    maps = []
    for _ in range(4):
        with ml.Mlens.from_config(cfg, xy, m) as h:
            c, mg, st = h.shoot_host()
            maps.append(c.copy())
    assert all(np.array_equal(maps[0], c) for c in maps[1:])
    free0, _ = torch.cuda.mem_get_info()
    ml.trim_memory()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0  # the cached result buffers (2 x 1 MB here) went back; nothing is in use any more
    with ml.Mlens.from_config(cfg, xy, m) as h:  # and the pool still works after a trim
        c, _, _ = h.shoot_host()
    assert np.array_equal(c, maps[0])
