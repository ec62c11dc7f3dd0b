"""Minimal-bit-width storage of maps (Table B.6) and the re-binned MPD view.

CPU: the oracle's bit packing is pinned to the numbers Table B.6 prints, to a hand-worked bit stream and to Python's
arbitrary-precision integers; the re-binned MPD to a hand-worked example.  GPU: mlens_pack_map / mlens_unpack_map /
mlens_mpd_rebin against the oracle (bit-exact for the integer work)."""
import ctypes
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _table_b6():
    rows, need = [], []
    for line in open(os.path.join(GOLDEN, "table_b6_bit_widths.txt")):
        t = line.split("#")[0].split()
        if not t:
            continue
        if t[0] == "need":
            need.append((int(t[1]), int(t[2])))
        else:
            rows.append((int(t[0]), int(t[1]), int(t[2]), t[3] == "yes"))
    return rows, need


def test_p15_bit_widths_against_table_b6(oracle):
    rows, need = _table_b6()
    assert len(rows) == 6 and len(need) == 4
    for bits, max_printed, mb_printed, exact in rows:
        if exact:  # the printed maximum is 2^b - 1: it needs exactly b bits and one more needs b + 1
            assert oracle.bits_needed(max_printed) == bits
            if bits < 32:
                assert oracle.bits_needed(max_printed + 1) == bits + 1
        else:      # the printed 22-bit entry is 2^22 (typo for 2^22 - 1): it needs 23 bits, its predecessor 22
            assert oracle.bits_needed(max_printed) == bits + 1 and oracle.bits_needed(max_printed - 1) == bits
        # file size of a 10000^2 map: words of the packed stream x 4 bytes, in MiB, rounded as the table prints it
        packed = oracle.pack_bits(np.zeros(0, np.uint32), bits)
        assert packed.size == 0
        n_words = (10000 * 10000 * bits + 31) // 32
        assert round(n_words * 4 / 2**20) == mb_printed
    for value, bits in need:
        assert oracle.bits_needed(value) == bits
    assert oracle.bits_needed(0) == 1 and oracle.bits_needed(1) == 1 and oracle.bits_needed(2) == 2


def test_p15_hand_worked_bit_stream(oracle):
    # six 3-bit values, least-significant bit first: 5=101b -> stream bits 0..2 = 1,0,1; 2 -> 0,1,0; 7 -> 1,1,1; 0; 3 -> 1,1,0;
    # 6 -> 0,1,1.  Set bits: 0,2,4,6,7,8,12,13,16,17  =>  word = 1+4+16+64+128+256+4096+8192+65536+131072 = 209365
    packed = oracle.pack_bits([5, 2, 7, 0, 3, 6], 3)
    assert packed.tolist() == [209365]
    assert oracle.unpack_bits(packed, 6, 3).tolist() == [5, 2, 7, 0, 3, 6]
    # a value that straddles a word boundary: 20-bit values, the second one occupies bits 20..39
    vals = [0xABCDE, 0x12345, 0xFFFFF, 0x00001]
    packed = oracle.pack_bits(vals, 20)
    assert packed.tolist() == [0xABCDE | ((0x12345 & 0xFFF) << 20), (0x12345 >> 12) | (0xFFFFF << 8) | ((0x1 & 0xF) << 28), 0x1 >> 4]
    assert oracle.unpack_bits(packed, 4, 20).tolist() == vals


@pytest.mark.parametrize("bits", [1, 2, 7, 14, 16, 20, 22, 24, 31, 32])
def test_p15_bit_stream_is_the_big_integer(oracle, bits):
    # the whole stream read as ONE little-endian integer is sum_q v_q 2^(q*bits): Python's unbounded ints restate that
    rng = np.random.default_rng(bits)
    vals = rng.integers(0, 2**bits, size=257, dtype=np.uint64).astype(np.uint32)
    packed = oracle.pack_bits(vals, bits)
    big = sum(int(v) << (q * bits) for q, v in enumerate(vals.tolist()))
    words = [(big >> (32 * w)) & 0xFFFFFFFF for w in range((257 * bits + 31) // 32)]
    assert packed.tolist() == words
    assert np.array_equal(oracle.unpack_bits(packed, 257, bits), vals)


def test_p16_rebinned_mpd_hand_example(oracle):
    # 16 pixels, N_avg = 10: six with count 0, five with 10 (mu = 1), three with 100 (mu = 10), two with 1000 (mu = 100).
    # Four one-decade bins on [0.1, 1000): mu = 1 -> bin 1, 10 -> bin 2, 100 -> bin 3; the zero counts have no logarithm.
    hist = np.zeros(1002, np.uint64)
    hist[0], hist[10], hist[100], hist[1000] = 6, 5, 3, 2
    prob = oracle.mpd_rebin(hist, 10.0, 16, 4, 0.1, 1000.0)
    assert prob.tolist() == [0.0, 5 / 16, 3 / 16, 2 / 16]
    # a range that cuts the top off, and two bins per decade
    prob = oracle.mpd_rebin(hist, 10.0, 16, 4, 0.1, 10.0)  # bins of half a decade on [0.1, 10): mu = 1 -> bin 2; 10, 100 out
    assert prob.tolist() == [0.0, 0.0, 5 / 16, 0.0]


def test_packing_host_helpers_of_the_abi():
    from paper_1406_0559_b200 import build, mlens

    build.build_lib()
    L = mlens.lib()
    rows, need = _table_b6()
    for bits, max_printed, mb_printed, exact in rows:
        if exact:
            assert L.mlens_bits_needed(max_printed) == bits
        assert round(L.mlens_packed_words(10000 * 10000, bits) * 4 / 2**20) == mb_printed
    for value, bits in need:
        assert L.mlens_bits_needed(value) == bits
    assert L.mlens_packed_words(10, 0) == -1 and L.mlens_packed_words(10, 33) == -1 and L.mlens_packed_words(-1, 8) == -1
    assert L.mlens_packed_words(3, 20) == 2 and L.mlens_packed_words(0, 20) == 0
    assert L.mlens_pack_map(None, None, 32, 8, None, None) == mlens.EINVAL
    assert L.mlens_mpd_rebin(None, None, 10, 100, 0.1, 10.0, None, None) == mlens.EINVAL


# ---------------------------------------------------------------------------------------------------------------
# GPU parity
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("npix", [1, 7, 250, 1023])
def test_pack_unpack_match_the_oracle_bit_for_bit(oracle, npix):
    torch = pytest.importorskip("torch")
    from paper_1406_0559_b200 import mlens

    rng = np.random.default_rng(npix)
    with mlens.Mlens(0.3, 0.2, 0.0, 4.0, npix, 4.0 / npix / 2, np.zeros((1, 2), np.float32)) as h:
        for bits in (1, 3, 14, 16, 20, 24, 31, 32):
            vals = rng.integers(0, 2**bits, size=(npix, npix), dtype=np.uint64)
            src = torch.from_numpy(vals.astype(np.uint32).view(np.int32)).cuda()
            packed = h.pack_map(src, bits)
            ref = oracle.pack_bits(vals, bits)
            assert np.array_equal(packed.cpu().numpy().view(np.uint32), ref), bits
            back = h.unpack_map(packed, bits)
            assert torch.equal(back, src)
        for bits in (5, 11, 16):  # indexed maps are 16-bit
            vals = rng.integers(0, 2**bits, size=(npix, npix), dtype=np.uint64)
            src = torch.from_numpy(vals.astype(np.uint16)).cuda()
            packed = h.pack_map(src, bits)
            assert np.array_equal(packed.cpu().numpy().view(np.uint32), oracle.pack_bits(vals, bits)), bits
            assert torch.equal(h.unpack_map(packed, bits, dtype=torch.uint16), src)
        with pytest.raises(mlens.MlensError):
            h.pack_map(src, 17)  # wider than the 16-bit source


@pytest.mark.gpu
def test_indexed_map_packed_to_its_minimal_width_round_trips(oracle):
    # the whole storage chain of PAPER.md:700-712 on a shot map: count -> (index file, indexed map) -> minimal-width bit stream
    torch = pytest.importorskip("torch")
    import dataclasses

    from paper_1406_0559_b200 import fields, mlens

    cfg = dataclasses.replace(fields.CONFIGS[1], npix=200, sub=6)
    xy, m = fields.lens_field(cfg)
    with mlens.Mlens.from_config(cfg, xy, m) as h:
        count, _, st = h.shoot(want_mag=False)
        values, indexed = h.index_map(count)
        bits = oracle.bits_needed(int(values.numel()) - 1)
        assert bits == mlens.lib().mlens_bits_needed(int(values.numel()) - 1) and bits < 16
        packed = h.pack_map(indexed, bits)
        assert packed.numel() == (cfg.npix**2 * bits + 31) // 32
        assert np.array_equal(packed.cpu().numpy().view(np.uint32), oracle.pack_bits(indexed.cpu().numpy(), bits))
        back = h.unindex_map(h.unpack_map(packed, bits, dtype=torch.uint16), values.contiguous())
        assert torch.equal(back, count)
        # and the ray-count map itself at the width of its largest count
        bits_c = oracle.bits_needed(st["max_count"])
        assert torch.equal(h.unpack_map(h.pack_map(count, bits_c), bits_c), count)


@pytest.mark.gpu
def test_mpd_rebin_matches_the_oracle(oracle):
    torch = pytest.importorskip("torch")
    import dataclasses

    from paper_1406_0559_b200 import fields, mlens

    cfg = dataclasses.replace(fields.CONFIGS[3], npix=256, sub=6)
    xy, m = fields.lens_field(cfg)
    with mlens.Mlens.from_config(cfg, xy, m) as h:
        count, _, st = h.shoot(want_mag=False)
        n_bins = st["max_count"] + 2
        hist, _ = h.mpd(count, n_bins)
        hist_ref, _ = oracle.mpd(count.cpu().numpy(), n_bins, h.geometry.n_avg)
        for n_out, lo, hi in ((100, 0.1, 100.0), (400, 0.05, 300.0), (1, 0.5, 2.0), (7, 1.0, 3.0)):
            prob = h.mpd_rebin(hist, n_out, lo, hi).cpu().numpy()
            ref = oracle.mpd_rebin(hist_ref, h.geometry.n_avg, cfg.npix**2, n_out, lo, hi)
            assert np.array_equal(prob, ref)  # integer pixel counts per bin, one division: bit-exact and deterministic
            assert np.array_equal(h.mpd_rebin(hist, n_out, lo, hi).cpu().numpy(), prob)
            assert prob.sum() <= 1.0 + 1e-12
        # counts that sit EXACTLY on bin edges (N_avg = 36: c = 36, 360, 3600 are mu = 1, 10, 100): mu on an inner edge goes
        # to the upper bin, mu = mu_min is inside, mu = mu_max is outside — same side as the oracle in every case
        edge = np.zeros(4000, np.uint64)
        edge[[35, 36, 37, 359, 360, 361, 3599, 3600, 3601]] = [1, 2, 4, 8, 16, 32, 64, 128, 256]
        edge_dev = torch.from_numpy(edge.view(np.int64)).cuda()
        assert h.geometry.n_avg == 36.0
        for n_out, lo, hi in ((3, 0.1, 100.0), (2, 1.0, 100.0), (4, 1.0, 100.0), (400, 1.0, 10.0), (1, 10.0, 100.0), (6, 0.01, 10000.0)):
            prob = h.mpd_rebin(edge_dev, n_out, lo, hi).cpu().numpy()
            ref = oracle.mpd_rebin(edge, 36.0, cfg.npix**2, n_out, lo, hi)
            assert np.array_equal(prob, ref), (n_out, lo, hi)
        prob = h.mpd_rebin(edge_dev, 2, 1.0, 100.0).cpu().numpy() * cfg.npix**2  # [1,10) and [10,100)
        assert prob.tolist() == [2 + 4 + 8, 16 + 32 + 64]
        for bad in ((0, 0.1, 10.0), (401, 0.1, 10.0), (100, 0.0, 10.0), (100, 2.0, 1.0)):
            with pytest.raises(mlens.MlensError):
                h.mpd_rebin(hist, *bad)
