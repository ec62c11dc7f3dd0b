"""Thin ctypes binding of ``libmlens.so`` (``include/mlens.h``): argument marshalling only.

PyTorch is used for device memory and streams; every step of the hot path runs in the CUDA kernels behind the C ABI.
There is no CPU fallback: if the library has not been built (``python -c "import __graft_entry__ as g; g.build()"``
or ``python -m paper_1406_0559_b200.build``) or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "lib", "libmlens.so")
LIB_PATH_ABLATIONS = os.path.join(_HERE, "lib", "libmlens_ablations.so")  # -DMLENS_ABLATIONS build: tests / profiling only
_libs: dict = {}

OK, EINVAL, ENOMEM, ECUDA, ERANGE = 0, -1, -2, -3, -4


class MlensError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"mlens error {code}: {msg}")
        self.code = code


class Stats(ctypes.Structure):
    _fields_ = [("rays_total", ctypes.c_longlong), ("rays_in_map", ctypes.c_longlong),
                ("rays_outside", ctypes.c_longlong), ("rays_lost", ctypes.c_longlong), ("n_lens", ctypes.c_longlong),
                ("max_count", ctypes.c_int), ("elapsed_ms", ctypes.c_float), ("kernel_ms", ctypes.c_float)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class Geometry(ctypes.Structure):
    _fields_ = [("n1", ctypes.c_longlong), ("n2", ctypes.c_longlong), ("a1", ctypes.c_double), ("a2", ctypes.c_double),
                ("p", ctypes.c_double), ("d", ctypes.c_double), ("kappa_s", ctypes.c_double),
                ("kappa_star", ctypes.c_double), ("n_avg", ctypes.c_double)]


class MapStats(ctypes.Structure):
    _fields_ = [("n_pixels", ctypes.c_longlong), ("sum_count", ctypes.c_longlong), ("n_clamped", ctypes.c_longlong),
                ("min_count", ctypes.c_int), ("max_count", ctypes.c_int), ("mean_count", ctypes.c_double),
                ("mean_mu", ctypes.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def lib(ablations: bool = False) -> ctypes.CDLL:
    """Load libmlens.so and declare the prototypes of every symbol in include/mlens.h.  Raises if it is not built.

    ``ablations=True`` loads libmlens_ablations.so instead: the same ABI compiled with -DMLENS_ABLATIONS, in which
    ``mlens_set_option`` can also select the debug / ablation / experimental kernels (tests and profiling only)."""
    key = bool(ablations)
    if key in _libs:
        return _libs[key]
    path = LIB_PATH_ABLATIONS if key else LIB_PATH
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it first (__graft_entry__.build()); there is no CPU fallback")
    L = ctypes.CDLL(path)
    vp, ll, dbl, ci = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_double, ctypes.c_int
    L.mlens_create.argtypes = [ctypes.POINTER(vp), dbl, dbl, dbl, dbl, ci, dbl, vp, vp, ll]
    L.mlens_shoot.argtypes = [vp, vp, vp, vp, ctypes.POINTER(Stats)]
    L.mlens_shoot_block.argtypes = [vp, ll, ll, ll, ll, vp, vp, vp, vp]
    L.mlens_shoot_host.argtypes = [vp, vp, vp, ctypes.POINTER(Stats)]
    L.mlens_magnification.argtypes = [vp, vp, vp, vp]
    L.mlens_mpd.argtypes = [vp, vp, vp, ci, vp, ctypes.POINTER(MapStats)]
    L.mlens_mpd_static.argtypes = [vp, ll, dbl, vp, ci, vp, ctypes.POINTER(MapStats)]
    L.mlens_index_map.argtypes = [vp, vp, vp, ci, vp, vp, ctypes.POINTER(ci)]
    L.mlens_unindex_map.argtypes = [vp, vp, vp, ci, vp, vp]
    L.mlens_bits_needed.argtypes = [ctypes.c_ulonglong]
    L.mlens_packed_words.argtypes = [ll, ci]
    L.mlens_packed_words.restype = ll
    L.mlens_pack_map.argtypes = [vp, vp, ci, ci, vp, vp]
    L.mlens_unpack_map.argtypes = [vp, vp, ci, vp, ci, vp]
    L.mlens_mpd_rebin.argtypes = [vp, vp, ci, ci, dbl, dbl, vp, vp]
    L.mlens_profile_kernel.argtypes = [vp, ci, dbl, vp, vp]
    L.mlens_convolve.argtypes = [vp, vp, vp, vp, vp]
    L.mlens_convolve_prepare.argtypes = [vp, vp, vp]
    L.mlens_get_geometry.argtypes = [vp, ctypes.POINTER(Geometry)]
    L.mlens_get_stats.argtypes = [vp, vp, ctypes.POINTER(Stats)]
    L.mlens_reset_stats.argtypes = [vp, vp]
    L.mlens_set_option.argtypes = [vp, ctypes.c_char_p, ll]
    L.mlens_last_error.argtypes = []
    L.mlens_last_error.restype = ctypes.c_char_p
    L.mlens_trim_memory.argtypes = []
    L.mlens_trim_memory.restype = ci
    L.mlens_destroy.argtypes = [vp]
    L.mlens_destroy.restype = None
    L.mlens_destroy_on_stream.argtypes = [vp, vp]
    L.mlens_destroy_on_stream.restype = None
    for name in ("mlens_create", "mlens_shoot", "mlens_shoot_block", "mlens_shoot_host", "mlens_magnification", "mlens_mpd",
                 "mlens_profile_kernel", "mlens_convolve", "mlens_index_map", "mlens_unindex_map",
                 "mlens_get_geometry", "mlens_get_stats", "mlens_reset_stats", "mlens_set_option", "mlens_bits_needed",
                 "mlens_pack_map", "mlens_unpack_map", "mlens_mpd_rebin", "mlens_convolve_prepare", "mlens_mpd_static"):
        getattr(L, name).restype = ci
    _libs[key] = L
    return L


def trim_memory(ablations: bool = False):
    """mlens_trim_memory: release the device blocks that destroyed handles left in the library's pool (current device)."""
    _check(lib(ablations).mlens_trim_memory(), lib(ablations))


def _check(rc: int, L=None):
    if rc != 0:
        raise MlensError(rc, (L or lib()).mlens_last_error().decode())


def _stream_ptr(stream=None):
    import torch

    s = stream if stream is not None else torch.cuda.current_stream()
    return ctypes.c_void_p(s.cuda_stream)


MPD_STATIC_MAX_BINS = 8192  # MLENS_MPD_STATIC_MAX_BINS of include/mlens.h


def mpd_static(count, n_bins, n_avg, hist, stream=None, sync=True, ablations=False):
    """mlens_mpd_static: the MPD histogram and map statistics of ``count`` without a handle and without any allocation
    inside the library — for programs that have no device memory left to give (everything reserved by one allocator, a
    fixed budget) or that must not pay an allocation's device-wide synchronisation while other streams are busy.

    ``hist`` is the caller's int64 [n_bins] device tensor (n_bins <= MPD_STATIC_MAX_BINS); this wrapper allocates nothing
    either.  All calls in the process share one scratch array per GPU: calls that could overlap on the GPU race, so keep
    them on one stream or order the streams.  Make the first call on a device before starting any stream capture.
    Returns (hist, stats dict or None when sync=False)."""
    import torch

    assert count.is_cuda and count.dtype == torch.int32 and count.is_contiguous()
    assert hist.is_cuda and hist.dtype == torch.int64 and hist.is_contiguous() and hist.numel() == int(n_bins)
    L = lib(ablations)
    ms = MapStats() if sync else None
    _check(L.mlens_mpd_static(ctypes.c_void_p(count.data_ptr()), int(count.numel()), float(n_avg),
                              ctypes.c_void_p(hist.data_ptr()), int(n_bins), _stream_ptr(stream),
                              ctypes.byref(ms) if sync else None), L)
    return hist, (ms.as_dict() if sync else None)


class Mlens:
    """A map context: mlens_create ... mlens_destroy.  Device tensors are torch tensors on the current CUDA device."""

    def __init__(self, kappa, gamma, s, map_side, npix, ray_spacing, lens_xy, lens_m=None, ablations=False):
        L = self._L = lib(ablations)
        xy = np.ascontiguousarray(np.asarray(lens_xy, dtype=np.float32).reshape(-1))
        m = None if lens_m is None else np.ascontiguousarray(np.asarray(lens_m, dtype=np.float32).reshape(-1))
        n = xy.size // 2
        if m is not None and m.size != n:
            raise ValueError("lens_m and lens_xy disagree on the number of lenses")
        self._h = ctypes.c_void_p()
        self.npix = int(npix)
        self._ck(L.mlens_create(ctypes.byref(self._h), kappa, gamma, s, map_side, int(npix), ray_spacing,
                              xy.ctypes.data_as(ctypes.c_void_p) if n else None,
                              m.ctypes.data_as(ctypes.c_void_p) if m is not None and n else None, n))
        g = Geometry()
        self._ck(L.mlens_get_geometry(self._h, ctypes.byref(g)))
        self.geometry = g
        self.n_lens = n

    @classmethod
    def from_config(cls, cfg, lens_xy, lens_m, ablations=False):
        return cls(cfg.kappa, cfg.gamma, cfg.s, cfg.map_side, cfg.npix, cfg.ray_spacing, lens_xy, lens_m, ablations)

    def _ck(self, rc: int):
        _check(rc, self._L)

    def close(self, stream=None):
        """mlens_destroy; with ``stream``: mlens_destroy_on_stream — waits for that stream only (every call on this handle
        must have been issued to it), so maps running on other streams are not waited for."""
        if getattr(self, "_h", None) is not None and self._h:
            if stream is None:
                self._L.mlens_destroy(self._h)
            else:
                self._L.mlens_destroy_on_stream(self._h, _stream_ptr(stream))
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:  # interpreter shutdown: module globals may already be gone
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def set_option(self, key: str, value: int):
        self._ck(self._L.mlens_set_option(self._h, key.encode(), int(value)))

    # -- step a1-a5: the whole map -----------------------------------------------------------------------------
    def shoot(self, count=None, mag=None, want_mag=True, stream=None, sync=True):
        """mlens_shoot.  Returns (count int32 [npix,npix], mag float32 [npix,npix] or None, stats dict or None)."""
        import torch

        if count is None:
            count = torch.empty((self.npix, self.npix), dtype=torch.int32, device="cuda")
        if mag is None and want_mag:
            mag = torch.empty((self.npix, self.npix), dtype=torch.float32, device="cuda")
        assert count.is_cuda and count.dtype == torch.int32 and count.is_contiguous() and count.numel() == self.npix**2
        assert mag is None or (mag.is_cuda and mag.dtype == torch.float32 and mag.is_contiguous() and mag.numel() == self.npix**2)
        st = Stats() if sync else None
        self._ck(self._L.mlens_shoot(self._h, ctypes.c_void_p(count.data_ptr()),
                                 ctypes.c_void_p(mag.data_ptr()) if mag is not None else None, _stream_ptr(stream),
                                 ctypes.byref(st) if sync else None))
        return count, mag, (st.as_dict() if sync else None)

    # -- verification / partial shooting ---------------------------------------------------------------------------
    def shoot_block(self, i0, j0, ni, nj, count=None, want_rays=False, stream=None):
        """mlens_shoot_block.  Returns dict(count, [y float64 (nj,ni,2), pix int32 (nj,ni)]); accumulates into count."""
        import torch

        y = pix = None
        if want_rays:
            y = torch.empty((nj, ni, 2), dtype=torch.float64, device="cuda")
            pix = torch.empty((nj, ni), dtype=torch.int32, device="cuda")
        if count is not None:
            assert count.is_cuda and count.dtype == torch.int32 and count.is_contiguous() and count.numel() == self.npix**2
        self._ck(self._L.mlens_shoot_block(self._h, int(i0), int(j0), int(ni), int(nj),
                                       ctypes.c_void_p(count.data_ptr()) if count is not None else None,
                                       ctypes.c_void_p(y.data_ptr()) if y is not None else None,
                                       ctypes.c_void_p(pix.data_ptr()) if pix is not None else None, _stream_ptr(stream)))
        return {"count": count, "y": y, "pix": pix}

    def shoot_host(self, want_mag=True, count=None, mag=None):
        """mlens_shoot_host: HOST numpy buffers in and out (the end-to-end call).  ``count`` / ``mag`` may be caller-owned
        C-contiguous int32 / float32 arrays of npix*npix elements (e.g. views of pinned memory, reused between maps)."""
        if count is None:
            count = np.empty((self.npix, self.npix), dtype=np.int32)
        if mag is None and want_mag:
            mag = np.empty((self.npix, self.npix), dtype=np.float32)
        assert count.dtype == np.int32 and count.flags.c_contiguous and count.size == self.npix**2
        assert mag is None or (mag.dtype == np.float32 and mag.flags.c_contiguous and mag.size == self.npix**2)
        st = Stats()
        self._ck(self._L.mlens_shoot_host(self._h, count.ctypes.data_as(ctypes.c_void_p),
                                          mag.ctypes.data_as(ctypes.c_void_p) if mag is not None else None, ctypes.byref(st)))
        return count, mag, st.as_dict()

    def magnification(self, count, mag=None, stream=None):
        import torch

        if mag is None:
            mag = torch.empty((self.npix, self.npix), dtype=torch.float32, device="cuda")
        self._ck(self._L.mlens_magnification(self._h, ctypes.c_void_p(count.data_ptr()), ctypes.c_void_p(mag.data_ptr()),
                                         _stream_ptr(stream)))
        return mag

    def mpd(self, count, n_bins, hist=None, stream=None, sync=True):
        """mlens_mpd: histogram of the counts = the full MPD.  Returns (hist int64 [n_bins] on the
        device — the library writes unsigned 64-bit bins, torch views them as int64 — and the map-stats dict or None)."""
        import torch

        if hist is None:
            hist = torch.empty((int(n_bins),), dtype=torch.int64, device="cuda")
        assert hist.is_cuda and hist.dtype == torch.int64 and hist.is_contiguous() and hist.numel() == int(n_bins)
        assert count.is_cuda and count.dtype == torch.int32 and count.is_contiguous() and count.numel() == self.npix**2
        ms = MapStats() if sync else None
        self._ck(self._L.mlens_mpd(self._h, ctypes.c_void_p(count.data_ptr()), ctypes.c_void_p(hist.data_ptr()), int(n_bins),
                               _stream_ptr(stream), ctypes.byref(ms) if sync else None))
        return hist, (ms.as_dict() if sync else None)

    def index_map(self, count, max_values=65536, stream=None):
        """mlens_index_map: (values int32 [n_distinct] ascending, indexed uint16 [npix,npix]) — PAPER.md:700-706."""
        import torch

        assert count.is_cuda and count.dtype == torch.int32 and count.is_contiguous() and count.numel() == self.npix**2
        values = torch.empty((int(max_values),), dtype=torch.int32, device="cuda")
        indexed = torch.empty((self.npix, self.npix), dtype=torch.uint16, device="cuda")
        nd = ctypes.c_int(0)
        self._ck(self._L.mlens_index_map(self._h, ctypes.c_void_p(count.data_ptr()), ctypes.c_void_p(values.data_ptr()),
                                     int(max_values), ctypes.c_void_p(indexed.data_ptr()), _stream_ptr(stream), ctypes.byref(nd)))
        return values[: nd.value], indexed

    def unindex_map(self, indexed, values, count=None, stream=None):
        """mlens_unindex_map: count[q] = values[indexed[q]]."""
        import torch

        if count is None:
            count = torch.empty((self.npix, self.npix), dtype=torch.int32, device="cuda")
        assert indexed.is_cuda and indexed.dtype == torch.uint16 and indexed.is_contiguous() and indexed.numel() == self.npix**2
        assert values.is_cuda and values.dtype == torch.int32 and values.is_contiguous()
        self._ck(self._L.mlens_unindex_map(self._h, ctypes.c_void_p(indexed.data_ptr()), ctypes.c_void_p(values.data_ptr()),
                                       int(values.numel()), ctypes.c_void_p(count.data_ptr()), _stream_ptr(stream)))
        return count

    def pack_map(self, src, bits: int, stream=None):
        """mlens_pack_map: int32 or uint16 map -> uint32 words of the `bits`-per-value bit stream."""
        import torch

        assert src.is_cuda and src.is_contiguous() and src.numel() == self.npix**2 and src.dtype in (torch.int32, torch.uint16)
        n_words = int(self._L.mlens_packed_words(self.npix**2, int(bits)))
        if n_words < 0:
            raise MlensError(EINVAL, "bits must be 1..32")
        packed = torch.empty((n_words,), dtype=torch.int32, device="cuda")  # 32-bit words (torch views them as int32)
        self._ck(self._L.mlens_pack_map(self._h, ctypes.c_void_p(src.data_ptr()), 32 if src.dtype == torch.int32 else 16, int(bits),
                                        ctypes.c_void_p(packed.data_ptr()), _stream_ptr(stream)))
        return packed

    def unpack_map(self, packed, bits: int, dtype=None, stream=None):
        """mlens_unpack_map: the inverse of pack_map, into int32 (default) or uint16."""
        import torch

        dtype = dtype or torch.int32
        assert packed.is_cuda and packed.is_contiguous() and packed.dtype == torch.int32 and dtype in (torch.int32, torch.uint16)
        n_words = int(self._L.mlens_packed_words(self.npix**2, int(bits)))
        if n_words < 0 or packed.numel() < n_words:  # a short buffer would be read out of bounds on the device
            raise MlensError(EINVAL, f"packed holds {packed.numel()} words, a {self.npix}^2 map at {bits} bits needs {n_words}")
        dst = torch.empty((self.npix, self.npix), dtype=dtype, device="cuda")
        self._ck(self._L.mlens_unpack_map(self._h, ctypes.c_void_p(packed.data_ptr()), int(bits), ctypes.c_void_p(dst.data_ptr()),
                                          32 if dtype == torch.int32 else 16, _stream_ptr(stream)))
        return dst

    def mpd_rebin(self, hist, n_out: int, mu_min: float, mu_max: float, stream=None):
        """mlens_mpd_rebin: the exact MPD histogram -> n_out (<= 400) bins of equal width in log10(mu); float64 [n_out]."""
        import torch

        assert hist.is_cuda and hist.dtype == torch.int64 and hist.is_contiguous() and hist.numel() >= 2
        prob = torch.empty((int(n_out),), dtype=torch.float64, device="cuda")
        self._ck(self._L.mlens_mpd_rebin(self._h, ctypes.c_void_p(hist.data_ptr()), int(hist.numel()), int(n_out), float(mu_min),
                                         float(mu_max), ctypes.c_void_p(prob.data_ptr()), _stream_ptr(stream)))
        return prob

    def profile_kernel(self, shape: int, size_pixels: float, kernel=None, stream=None):
        """mlens_profile_kernel: convolution kernel of a source profile (0 uniform disc, 1 Gaussian), float32 [npix,npix]."""
        import torch

        if kernel is None:
            kernel = torch.empty((self.npix, self.npix), dtype=torch.float32, device="cuda")
        assert kernel.is_cuda and kernel.dtype == torch.float32 and kernel.is_contiguous() and kernel.numel() == self.npix**2
        self._ck(self._L.mlens_profile_kernel(self._h, int(shape), float(size_pixels), ctypes.c_void_p(kernel.data_ptr()),
                                          _stream_ptr(stream)))
        return kernel

    def convolve_prepare(self, kernel, stream=None):
        """mlens_convolve_prepare: transform a kernel once; later ``convolve(mag, None)`` calls reuse its spectrum."""
        import torch

        assert kernel.is_cuda and kernel.dtype == torch.float32 and kernel.is_contiguous() and kernel.numel() == self.npix**2
        self._ck(self._L.mlens_convolve_prepare(self._h, ctypes.c_void_p(kernel.data_ptr()), _stream_ptr(stream)))

    def convolve(self, mag, kernel, out=None, stream=None):
        """mlens_convolve: out = F^-1[F(mag) F(kernel)] (Eq. 6), the circular convolution; float32 [npix,npix].
        ``kernel=None`` uses the spectrum kept by ``convolve_prepare``."""
        import torch

        if out is None:
            out = torch.empty((self.npix, self.npix), dtype=torch.float32, device="cuda")
        for t in (mag, kernel, out):
            assert t is None or (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.numel() == self.npix**2)
        assert out.data_ptr() != mag.data_ptr() and (kernel is None or out.data_ptr() != kernel.data_ptr())
        self._ck(self._L.mlens_convolve(self._h, ctypes.c_void_p(mag.data_ptr()),
                                        ctypes.c_void_p(kernel.data_ptr()) if kernel is not None else None,
                                        ctypes.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def stats(self, stream=None):
        st = Stats()
        self._ck(self._L.mlens_get_stats(self._h, _stream_ptr(stream), ctypes.byref(st)))
        return st.as_dict()

    def reset_stats(self, stream=None):
        self._ck(self._L.mlens_reset_stats(self._h, _stream_ptr(stream)))
