"""Map statistics: the full MPD of PAPER.md:307 and the map means of PAPER.md:299.

CPU: the oracle's MPD is pinned to closed forms and brute force (never to itself).  GPU: mlens_mpd against the oracle,
bit-exact (integer work)."""
import dataclasses
from collections import Counter

import numpy as np
import pytest

from paper_1406_0559_b200 import fields
from test_oracle_pins import _lattice_points_in_pixel_preimage


# ---------------------------------------------------------------------------------------------------------------
# P11 — oracle pins
# ---------------------------------------------------------------------------------------------------------------
def test_p11_mpd_of_the_no_lens_map_is_the_closed_form(oracle):
    # kappa=0.3, gamma=0.2, no lenses (P1 case b): count(ix,iy) = c1(ix)*c2(iy) with c1 = 20 everywhere and c2 in {11,12};
    # the MPD is therefore two spikes whose heights follow from the 1-D lattice-point counts alone.
    L, npix, sub = 4.0, 64, 10
    r = oracle.shoot_block(0.3, 0.2, 1.0, L, npix, L / npix / sub, np.zeros((0, 2), np.float32), None)
    c1 = _lattice_points_in_pixel_preimage(npix, L, sub, 0.5)
    c2 = _lattice_points_in_pixel_preimage(npix, L, sub, 0.9)
    expect = Counter()
    for a, na in Counter(c1.tolist()).items():
        for b, nb in Counter(c2.tolist()).items():
            expect[a * b] += na * nb
    hist, st = oracle.mpd(r["count"], 512, r["geometry"].n_avg)
    assert {int(k): int(v) for k, v in enumerate(hist) if v} == dict(expect) and set(expect) == {220, 240}
    assert st["sum_count"] == r["stats"]["rays_in_map"] and st["n_clamped"] == 0
    assert (st["min_count"], st["max_count"]) == (220, 240)
    assert st["mean_count"] == 222.5 and abs(st["mean_mu"] - 2.225) < 1e-15  # <mu> = <N>/N_avg, N_avg = 100


def test_p11_mpd_brute_force_invariants_and_clamping(oracle):
    rng = np.random.default_rng(5)
    count = rng.integers(0, 50, size=(37, 41)).astype(np.int32)
    count[3, 4] = 1000; count[0, 0] = 63; count[1, 1] = 62
    hist, st = oracle.mpd(count, 64, 16.0)
    brute = [0] * 64
    for v in count.reshape(-1).tolist():  # pure-Python restatement of the definition
        brute[min(v, 63)] += 1
    assert hist.tolist() == brute
    assert int(hist.sum()) == count.size == st["n_pixels"]
    assert st["n_clamped"] == 2 and hist[63] == 2 and hist[62] == 1  # 1000 and 63 share the last bin
    assert st["sum_count"] == int(count.sum(dtype=np.int64)) and st["max_count"] == 1000 and st["min_count"] == int(count.min())
    # unclamped: first moment of the MPD reproduces <N> (the two mapmeta.dat numbers are tied by Eq. 4)
    hist2, st2 = oracle.mpd(count, 1002, 16.0)
    assert st2["n_clamped"] == 0 and int((hist2 * np.arange(1002, dtype=np.uint64)).sum()) == st2["sum_count"]
    assert st2["mean_mu"] == st2["mean_count"] / 16.0
    assert np.array_equal(hist2.astype(np.int64), np.bincount(count.reshape(-1), minlength=1002))


# ---------------------------------------------------------------------------------------------------------------
# GPU parity
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("npix,n_bins,hi", [(64, 4096, 3000), (250, 100, 5000), (1023, 20000, 19000), (1, 2, 5), (2048, 9000, 40000), (512, 70000, 69000),
                                            (4096, 30000, 29000), (130, 38000, 37000)])
def test_mlens_mpd_matches_the_oracle_bit_for_bit(oracle, npix, n_bins, hi):
    import torch

    from paper_1406_0559_b200 import mlens

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    # synthetic count maps with the shapes of real ones: a smooth bulk (most pixels in a few bins: the shared-memory
    # aggregation path), a long caustic tail beyond the shared-memory bins, zeros, and a ragged pixel count (npix odd)
    u = fields.uniform01(11 + npix, 0, npix * npix)
    count = (200 + 30 * np.sin(np.arange(npix * npix) * 1e-3) + (u > 0.98) * u * hi).astype(np.int32)
    count[u < 0.01] = 0
    cfg = fields.MapConfig("mpd", npix, 4.0, 0.3, 0.1, 0.0, 5, "unit", 3)
    with mlens.Mlens.from_config(cfg, np.zeros((1, 2), np.float32), None) as h:
        c_dev = torch.from_numpy(count).cuda().reshape(npix, npix)
        hist, st = h.mpd(c_dev, n_bins)
        hist2, _ = h.mpd(c_dev, n_bins, hist=hist)  # the call zeroes the bins itself: a second run must not add up
        ref_hist, ref = oracle.mpd(count, n_bins, h.geometry.n_avg)
        assert np.array_equal(hist2.cpu().numpy().astype(np.uint64), ref_hist)
        for k in ("n_pixels", "sum_count", "n_clamped", "min_count", "max_count"):
            assert st[k] == ref[k], k
        assert st["mean_count"] == ref["mean_count"] and st["mean_mu"] == ref["mean_mu"]
        # an all-equal map: the flat-region vote (one add of 128 per warp) instead of 32-way same-address atomics
        flat = torch.full((npix, npix), 7, dtype=torch.int32, device="cuda")
        hf, sf = h.mpd(flat, n_bins)
        assert int(hf[min(7, n_bins - 1)].item()) == npix * npix and sf["sum_count"] == 7 * npix * npix


@pytest.mark.gpu
def test_mpd_of_a_shot_map_ties_to_the_ray_counters(oracle):
    import torch

    from paper_1406_0559_b200 import mlens

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    cfg = dataclasses.replace(fields.CONFIGS[3], npix=512, sub=4)
    xy, m = fields.lens_field(cfg)
    with mlens.Mlens.from_config(cfg, xy, m) as h:
        count, _, st = h.shoot(want_mag=False)
        hist, ms = h.mpd(count, st["max_count"] + 2)
        assert ms["sum_count"] == st["rays_in_map"] and ms["max_count"] == st["max_count"] and ms["n_clamped"] == 0
        assert int(hist.sum().item()) == cfg.npix**2
        ref_hist, _ = oracle.mpd(count.cpu().numpy(), st["max_count"] + 2, h.geometry.n_avg)
        assert np.array_equal(hist.cpu().numpy().astype(np.uint64), ref_hist)


# ---------------------------------------------------------------------------------------------------------------
# indexed maps
# ---------------------------------------------------------------------------------------------------------------
def test_p13_index_map_oracle_brute_force_and_roundtrip(oracle):
    count = np.array([[7, 3, 7, 100], [3, 3, 0, 100], [5, 7, 65000, 0]], np.int32)
    values, indexed = oracle.index_map(count)
    assert values.tolist() == [0, 3, 5, 7, 100, 65000]  # the index file: distinct values, ascending (by hand)
    assert indexed.tolist() == [[3, 1, 3, 4], [1, 1, 0, 4], [2, 3, 5, 0]]
    rng = np.random.default_rng(3)
    count = (rng.integers(0, 300, size=(40, 33)) * rng.integers(1, 4, size=(40, 33))).astype(np.int32)
    values, indexed = oracle.index_map(count)
    lookup = {v: k for k, v in enumerate(sorted(set(count.reshape(-1).tolist())))}  # pure-Python restatement
    assert values.tolist() == sorted(lookup) and indexed.tolist() == [[lookup[v] for v in row] for row in count.tolist()]
    assert np.array_equal(values[indexed], count)  # lossless ("without any loss of information")


@pytest.mark.gpu
@pytest.mark.parametrize("npix,hi", [(64, 3000), (1023, 19000), (3, 5), (2048, 900000)])
def test_index_map_matches_the_oracle_and_roundtrips(oracle, npix, hi):
    import torch

    from paper_1406_0559_b200 import mlens

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    u = fields.uniform01(21 + npix, 0, npix * npix)
    count = (200 + 30 * np.sin(np.arange(npix * npix) * 1e-3) + (u > 0.98) * u * hi).astype(np.int32).reshape(npix, npix)
    count[0, 0] = 0
    cfg = fields.MapConfig("idx", npix, 4.0, 0.3, 0.1, 0.0, 5, "unit", 3)
    with mlens.Mlens.from_config(cfg, np.zeros((1, 2), np.float32), None) as h:
        c_dev = torch.from_numpy(count).cuda()
        values, indexed = h.index_map(c_dev)
        ref_values, ref_indexed = oracle.index_map(count)
        assert np.array_equal(values.cpu().numpy(), ref_values)
        assert np.array_equal(indexed.cpu().numpy().astype(np.int32), ref_indexed)
        back = h.unindex_map(indexed, values.contiguous())
        assert torch.equal(back, c_dev)


@pytest.mark.gpu
def test_index_map_reports_too_many_distinct_values():
    import torch

    from paper_1406_0559_b200 import mlens

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    npix = 300  # 90 000 pixels, all different
    cfg = fields.MapConfig("idx", npix, 4.0, 0.3, 0.1, 0.0, 5, "unit", 3)
    with mlens.Mlens.from_config(cfg, np.zeros((1, 2), np.float32), None) as h:
        c_dev = torch.arange(npix * npix, dtype=torch.int32, device="cuda").reshape(npix, npix).contiguous()
        with pytest.raises(mlens.MlensError) as e:
            h.index_map(c_dev)
        assert e.value.code == mlens.ERANGE
