"""P9 — the seeded generator: counts of Eq. 3, disc uniformity, Salpeter spectrum, determinism."""
import numpy as np
import pytest

from paper_1406_0559_b200 import fields


def test_splitmix64_reference_values():
    # splitmix64 with seed 0: first outputs of the published reference sequence (Steele, Lea & Flood 2014)
    z = fields.splitmix64(0, 0, 3)
    assert [int(v) for v in z] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]


@pytest.mark.parametrize("cfg_id,n_lens,rstar", [(1, 13, 6.5892), (2, 19837, 181.83), (3, 430, 92.770),
                                                  (4, 2333, 50.912), (5, 705, 48.466)])
def test_config_fields(cfg_id, n_lens, rstar):
    cfg = fields.CONFIGS[cfg_id]
    assert cfg.n_lens == n_lens
    assert abs(cfg.disc_radius / rstar - 1) < 1e-4
    xy, m = fields.lens_field(cfg)
    assert xy.dtype == np.float32 and m.dtype == np.float32 and xy.shape == (n_lens, 2) and m.shape == (n_lens,)
    r = np.hypot(xy[:, 0].astype(np.float64), xy[:, 1].astype(np.float64))
    assert r.max() <= cfg.disc_radius * (1 + 1e-6)
    # Eq. 3 inverted: kappa_* recovered from the total mass in the disc (A = pi R*^2, <M> = 1)
    assert abs(m.astype(np.float64).sum() / cfg.disc_radius**2 / cfg.kappa_star - 1) < 0.04
    assert abs(m.astype(np.float64).mean() - 1) < 1e-6
    xy2, m2 = fields.lens_field(cfg)
    assert np.array_equal(xy, xy2) and np.array_equal(m, m2)


def test_disc_is_uniform_in_area():
    xy = fields.disc_positions(20000, 3.0, 5)
    q = np.sort((xy**2).sum(axis=1) / 9.0)  # r^2/R^2 ~ U(0,1)
    ks = np.abs(q - (np.arange(q.size) + 0.5) / q.size).max()
    assert ks < 1.63 / np.sqrt(q.size)  # KS 1 % critical value
    ang = np.arctan2(xy[:, 1], xy[:, 0])
    assert abs(np.cos(ang).mean()) < 0.02 and abs(np.sin(ang).mean()) < 0.02


def test_salpeter_spectrum():
    m = fields.salpeter_masses(200000, 3)
    assert abs(m.mean() - 1) < 1e-12
    raw = m / m.max() * 1.0  # back on (0.01, 1] up to the largest draw
    assert raw.min() >= 0.0099 and raw.max() <= 1.0
    # log-slope of dN/dm from a histogram in log m
    edges = np.logspace(np.log10(0.012), np.log10(0.8), 16)
    h, _ = np.histogram(raw, bins=edges)
    mid = np.sqrt(edges[1:] * edges[:-1])
    slope = np.polyfit(np.log(mid), np.log(h / np.diff(edges)), 1)[0]
    assert abs(slope + 2.35) < 0.1


def test_block_plan_is_inside_lattice():
    cfg = fields.CONFIGS[5]
    xy, _ = fields.lens_field(cfg)
    n1, n2 = 240_000, 96_000
    blocks = fields.block_plan(n1, n2, xy, cfg.half_widths, cfg.ray_spacing, cfg.seed)
    assert len(blocks) >= 48
    for i0, j0, ni, nj in blocks:
        assert 0 <= i0 and i0 + ni <= n1 and 0 <= j0 and j0 + nj <= n2 and ni == nj == 256
    assert blocks == fields.block_plan(n1, n2, xy, cfg.half_widths, cfg.ray_spacing, cfg.seed)
