"""mlens_mpd_static — the MPD for callers that cannot allocate (include/mlens.h).

Who needs it: a process that handed all of its device memory to one allocator at start-up (or runs under a fixed memory
budget), and a loop that analyses finished maps while the next one is being shot on another stream — there a cudaMalloc
either fails or stalls every running kernel.  ``mlens_mpd`` allocates (handle, histogram slices, pinned statistics
block); ``mlens_mpd_static`` runs the same kernels with their scratch in a fixed 4.6 MiB array inside the library.

The file name sorts last on purpose: ``pytest -x`` stops at the first failure, and a failure here must not hide the
parity tests.  The GPU test passes alone in a fresh process (it then performs the once-per-device set-up itself) and after
the other tests (the library is then already loaded and other entry points have used the device).
"""
import ctypes

import numpy as np
import pytest

from paper_1406_0559_b200 import fields, mlens


def test_limits_are_checked_before_any_cuda_call():
    # no GPU needed: argument checks come first and name the limit (the scratch holds MLENS_MPD_STATIC_MAX_BINS bins)
    L = mlens.lib()
    one = ctypes.c_void_p(16)  # never dereferenced: the call fails on the size checks
    assert L.mlens_mpd_static(None, 4, 1.0, one, 16, None, None) == mlens.EINVAL
    assert L.mlens_mpd_static(one, 4, 1.0, None, 16, None, None) == mlens.EINVAL
    assert L.mlens_mpd_static(one, 0, 1.0, one, 16, None, None) == mlens.EINVAL
    assert L.mlens_mpd_static(one, 4, 1.0, one, 1, None, None) == mlens.EINVAL
    assert L.mlens_mpd_static(one, 4, 1.0, one, mlens.MPD_STATIC_MAX_BINS + 1, None, None) == mlens.ERANGE
    msg = L.mlens_last_error().decode()
    assert str(mlens.MPD_STATIC_MAX_BINS) in msg and "mlens_mpd" in msg
    ms = mlens.MapStats()
    assert L.mlens_mpd_static(one, 4, 0.0, one, 16, None, ctypes.byref(ms)) == mlens.EINVAL  # stats need N_avg > 0


def _synthetic_counts(npix, seed, hi):
    # the shape of a real count map: a smooth bulk, a caustic tail, empty pixels (as in tests/test_mpd.py)
    u = fields.uniform01(seed, 0, npix * npix)
    count = (200 + 30 * np.sin(np.arange(npix * npix) * 1e-3) + (u > 0.98) * u * hi).astype(np.int32)
    count[u < 0.01] = 0
    return count.reshape(npix, npix)


@pytest.mark.gpu
def test_mpd_static_equals_mlens_mpd_on_two_calls_in_a_row():
    """Two calls in a row share the static scratch: the second (fewer CTAs, fewer bins, different map) must not see
    anything of the first.  Integer work: the tolerance of the MPD tests is equality."""
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    # First the asynchronous form (stats = NULL), twice back to back on one stream without a host sync in between.  Run
    # alone in a fresh process this is the library's very first CUDA work: the once-per-device set-up happens here.
    a = torch.from_numpy(_synthetic_counts(700, 41, 3000)).cuda()
    b = torch.from_numpy(_synthetic_counts(64, 42, 100)).cuda()
    ha = torch.empty((4096,), dtype=torch.int64, device="cuda")
    hb = torch.empty((512,), dtype=torch.int64, device="cuda")
    mlens.mpd_static(a, 4096, 1.0, ha, sync=False)
    mlens.mpd_static(b, 512, 1.0, hb, sync=False)
    torch.cuda.synchronize()
    assert torch.equal(ha, torch.bincount(a.reshape(-1).clamp(max=4095).long(), minlength=4096))
    assert torch.equal(hb, torch.bincount(b.reshape(-1).clamp(max=511).long(), minlength=512))
    cases = [(1500, 8192, 9000, 31),   # 2.25 Mpx: all 148 CTAs, every static bin, counts clamped into the last bin
             (130, 300, 5000, 32),     # 16 900 px: 5 CTAs, 1024 shared bins, most of the tail clamped
             (1500, 8192, 9000, 31)]   # the first map again, after the small one
    stream = torch.cuda.Stream()
    for k, (npix, n_bins, hi, seed) in enumerate(cases):
        count = torch.from_numpy(_synthetic_counts(npix, seed, hi)).cuda()
        # the existing path needs a handle (of the same pixel count); its N_avg is passed to the static call
        cfg = fields.MapConfig("noalloc", npix, 4.0, 0.3, 0.1, 0.0, 5, "unit", 3)
        with mlens.Mlens.from_config(cfg, np.zeros((1, 2), np.float32), None) as h:
            hist_static = torch.full((n_bins,), -1, dtype=torch.int64, device="cuda")  # the call zeroes the bins itself
            torch.cuda.synchronize()
            _, st_static = mlens.mpd_static(count, n_bins, h.geometry.n_avg, hist_static, stream=stream)
            hist_ref, st_ref = h.mpd(count, n_bins)
            assert torch.equal(hist_static, hist_ref), f"call {k}: histograms differ"
            assert st_static == st_ref, (k, st_static, st_ref)
        assert int(hist_static.sum().item()) == npix * npix
