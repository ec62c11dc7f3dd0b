"""Finite-source convolution (Eq. 6).

CPU: the oracle (the circular convolution written out as its definition, FP64) is pinned to a hand-worked example,
closed forms and the convolution theorem evaluated by numpy's FFT.  GPU: mlens_profile_kernel / mlens_convolve
(cuFFT + the fused spectral-product kernel) against the oracle within the FP32 tolerance derived in DESIGN.md."""
import os

import numpy as np
import pytest

from paper_1406_0559_b200 import fields

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
# FP32 FFT round-off: ~eps * log2(N^2) relative to the rms of the data (eps = 6e-8, N = 10000 -> 1.6e-6); the spectral
# product and the 1/N^2 scale add O(eps).  Gate at 2e-5 of max|C|.
TOL_REL = 2e-5


def _read_golden():
    rows = {"M": [], "K": [], "C": []}
    for line in open(os.path.join(GOLDEN, "p12_convolution_hand.txt")):
        f = line.split()
        if f and f[0] in rows:
            rows[f[0]].append([float(v) for v in f[1:]])
    return (np.array(rows[k]) for k in ("M", "K", "C"))


# ---------------------------------------------------------------------------------------------------------------
# P12 — oracle pins
# ---------------------------------------------------------------------------------------------------------------
def test_p12_hand_worked_3x3(oracle):
    M, K, C = _read_golden()
    assert np.array_equal(oracle.convolve(M, K), C)  # all values are exact in binary
    assert np.array_equal(oracle.convolve(M, K, points=[[2, 0], [0, 2]]), [6.0, 3.5])


def test_p12_delta_shift_constant_and_flux(oracle):
    n = 12
    M = fields.uniform01(77, 0, n * n).reshape(n, n).astype(np.float32)
    K = np.zeros((n, n), np.float32); K[0, 0] = 1
    assert np.array_equal(oracle.convolve(M, K), M.astype(np.float64))          # delta at the origin: identity
    K = np.zeros((n, n), np.float32); K[2, n - 3] = 1
    assert np.array_equal(oracle.convolve(M, K), np.roll(M.astype(np.float64), (2, -3), axis=(0, 1)))  # shifted delta
    K = oracle.profile_kernel(1, 1.2, n)
    C = oracle.convolve(np.full((n, n), 3.0, np.float32), K)
    assert np.allclose(C, 3.0 * K.astype(np.float64).sum(), rtol=0, atol=1e-12)  # constant map -> constant * sum(K)
    C = oracle.convolve(M, K)
    assert abs(C.sum() - M.astype(np.float64).sum() * K.astype(np.float64).sum()) < 1e-9  # flux conservation
    # symmetric kernel => convolution commutes with a transpose of the map
    assert np.allclose(oracle.convolve(M.T.copy(), K), C.T, rtol=0, atol=1e-13)


def test_p12_convolution_theorem_with_numpy_fft(oracle):
    # Eq. 6 itself, evaluated by an independent library FFT in FP64 (non-power-of-two size, asymmetric kernel)
    n = 30
    M = (1 + 5 * fields.uniform01(5, 0, n * n)).reshape(n, n).astype(np.float32)
    K = np.zeros((n, n), np.float32)
    K[:4, :3] = fields.uniform01(6, 0, 12).reshape(4, 3); K[n - 2:, n - 5:] = fields.uniform01(7, 0, 10).reshape(2, 5)
    ref = np.fft.ifft2(np.fft.fft2(M.astype(np.float64)) * np.fft.fft2(K.astype(np.float64))).real
    assert np.allclose(oracle.convolve(M, K), ref, rtol=0, atol=1e-11)


@pytest.mark.parametrize("shape,size", [(0, 2.5), (1, 1.5), (0, 1.0), (1, 0.4)])
def test_p12_profile_kernel_properties(oracle, shape, size):
    n = 33
    K = oracle.profile_kernel(shape, size, n).astype(np.float64)
    assert abs(K.sum() - 1) < 1e-6 and (K >= 0).all()
    Kc = np.roll(K, (n // 2, n // 2), axis=(0, 1))  # centre the profile for geometric checks
    yy, xx = np.mgrid[:n, :n] - n // 2
    r = np.hypot(xx, yy)
    assert np.array_equal(Kc, Kc[::-1, :]) and np.array_equal(Kc, Kc[:, ::-1]) and np.array_equal(Kc, Kc.T)
    if shape == 0:  # uniform disc: equal weight 1/#pixels inside the radius, zero outside
        inside = r <= size
        assert np.allclose(Kc[inside], 1.0 / inside.sum(), rtol=1e-6) and not Kc[~inside].any()
    else:           # Gaussian: ratio to the central pixel follows exp(-r^2/2 sigma^2); cut at 4 sigma
        assert not Kc[r > 4 * size].any()
        sel = r <= 4 * size
        assert np.allclose(Kc[sel] / Kc[n // 2, n // 2], np.exp(-r[sel] ** 2 / (2 * size**2)), rtol=2e-6, atol=1e-9)


# ---------------------------------------------------------------------------------------------------------------
# GPU parity
# ---------------------------------------------------------------------------------------------------------------
def _gpu():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1406_0559_b200 import mlens

    return torch, mlens


def _handle(mlens, npix):
    cfg = fields.MapConfig("conv", npix, 4.0, 0.3, 0.1, 0.0, 5, "unit", 3)
    return mlens.Mlens.from_config(cfg, np.zeros((1, 2), np.float32), None)


@pytest.mark.gpu
@pytest.mark.parametrize("npix,shape,size", [(64, 1, 1.5), (250, 0, 6.3), (243, 1, 3.0), (1000, 0, 20.0), (17, 1, 0.5)])
def test_profile_kernel_and_convolution_match_the_oracle(oracle, npix, shape, size):
    torch, mlens = _gpu()
    # a map with the dynamic range of a magnification map: smooth background + sharp caustic-like ridges
    u = fields.uniform01(100 + npix, 0, npix * npix).reshape(npix, npix)
    yy, xx = np.mgrid[:npix, :npix]
    M = (1.0 + 0.3 * u + 40.0 / (1.0 + 0.5 * np.abs((xx * 0.7 + yy * 0.4) % 37 - 18))).astype(np.float32)
    with _handle(mlens, npix) as h:
        K_gpu = h.profile_kernel(shape, size)
        K_ref = oracle.profile_kernel(shape, size, npix)
        Kg = K_gpu.cpu().numpy()
        assert np.array_equal(Kg != 0, K_ref != 0)
        assert np.allclose(Kg, K_ref, rtol=1e-6, atol=0)
        C_gpu = h.convolve(torch.from_numpy(M).cuda(), K_gpu).cpu().numpy().astype(np.float64)
        C_gpu2 = h.convolve(torch.from_numpy(M).cuda(), K_gpu).cpu().numpy()  # plans and spectra are reused
        with pytest.raises(mlens.MlensError):
            h.convolve(torch.from_numpy(M).cuda(), None)  # nothing prepared yet
        h.convolve_prepare(K_gpu)  # the kernel's spectrum kept in the handle: two FFTs per map instead of three
        C_gpu3 = h.convolve(torch.from_numpy(M).cuda(), None).cpu().numpy()
        h.convolve(torch.from_numpy(M).cuda(), h.profile_kernel(0, 1.0))  # another kernel in between must not disturb it
        C_gpu4 = h.convolve(torch.from_numpy(M).cuda(), None).cpu().numpy()
        assert np.array_equal(C_gpu3, C_gpu2) and np.array_equal(C_gpu4, C_gpu2)
    if npix <= 250:
        C_ref = oracle.convolve(M, Kg)  # same kernel bytes on both sides: this compares the convolution alone
        err = np.abs(C_gpu - C_ref).max()
    else:
        pts = (fields.uniform01(9, 0, 4000) * npix).astype(np.int64).reshape(-1, 2)
        C_ref = oracle.convolve(M, Kg, points=pts)
        err = np.abs(C_gpu[pts[:, 0], pts[:, 1]] - C_ref).max()
    assert err <= TOL_REL * np.abs(C_ref).max(), (err, np.abs(C_ref).max())
    assert np.array_equal(C_gpu2.astype(np.float64), C_gpu)
    assert abs(C_gpu.sum() / M.astype(np.float64).sum() - 1) < 1e-5  # sum(K) = 1: flux is conserved


@pytest.mark.gpu
def test_convolution_rejects_bad_arguments():
    torch, mlens = _gpu()
    with _handle(mlens, 32) as h:
        for shape, size in [(2, 1.0), (0, 0.0), (0, float("nan")), (1, 5.0), (0, 16.0)]:  # 4 sigma = 20 > 32/2
            with pytest.raises(mlens.MlensError) as e:
                h.profile_kernel(shape, size)
            assert e.value.code == mlens.EINVAL
