"""ORACLE — TEST INFRASTRUCTURE ONLY (ctypes loader for oracle/oracle.cpp).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import
this package.  It shares no code with ``paper_1406_0559_b200`` and does not import it.  See the header of
``oracle.cpp`` for the passages of PAPER.md each function follows and for the pins.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


class Geometry(ctypes.Structure):
    _fields_ = [("n1", ctypes.c_longlong), ("n2", ctypes.c_longlong), ("a1", ctypes.c_double), ("a2", ctypes.c_double),
                ("p", ctypes.c_double), ("d", ctypes.c_double), ("kappa_s", ctypes.c_double),
                ("kappa_star", ctypes.c_double), ("n_avg", ctypes.c_double)]


class Stats(ctypes.Structure):
    _fields_ = [("rays_total", ctypes.c_longlong), ("rays_in_map", ctypes.c_longlong),
                ("rays_outside", ctypes.c_longlong), ("rays_lost", ctypes.c_longlong)]


def build(force: bool = False) -> str:
    """Compile oracle.cpp with g++ (-O3 -march=native -fopenmp, no fast-math) if the .so is missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O3", "-march=native", "-fopenmp", "-shared", "-fPIC", "-Wall", _SRC, "-o", _LIB])
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        try:
            _lib = ctypes.CDLL(build())
        except OSError:  # built on another host with a different -march=native
            _lib = ctypes.CDLL(build(force=True))
    return _lib


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ct))


def _lens(lens_xy, lens_m):
    xy = np.ascontiguousarray(np.asarray(lens_xy, dtype=np.float32).reshape(-1))
    m = None if lens_m is None else np.ascontiguousarray(np.asarray(lens_m, dtype=np.float32).reshape(-1))
    n = xy.size // 2
    assert m is None or m.size == n
    return xy, m, n


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def geometry(kappa, gamma, s, L, npix, d) -> Geometry:
    g = Geometry()
    rc = lib().oracle_derive_geometry(ctypes.c_double(kappa), ctypes.c_double(gamma), ctypes.c_double(s),
                                      ctypes.c_double(L), ctypes.c_int(npix), ctypes.c_double(d), ctypes.byref(g))
    if rc != 0:
        raise ValueError("oracle_derive_geometry: invalid parameters")
    return g


def shoot_block(kappa, gamma, s, L, npix, d, lens_xy, lens_m, block=None, count=None, want_rays=False, n_threads=0):
    """Shoot a ray sub-block (default: the whole lattice).  Returns dict(count, stats, [y, alpha, scale, pix])."""
    g = geometry(kappa, gamma, s, L, npix, d)
    i0, j0, ni, nj = block if block is not None else (0, 0, g.n1, g.n2)
    xy, m, n = _lens(lens_xy, lens_m)
    if count is None:
        count = np.zeros((npix, npix), dtype=np.int32)
    assert count.dtype == np.int32 and count.flags.c_contiguous and count.size == npix * npix
    y = al = sc = pix = None
    if want_rays:
        y = np.empty((nj, ni, 2), dtype=np.float64)
        al = np.empty((nj, ni, 2), dtype=np.float64)
        sc = np.empty((nj, ni), dtype=np.float64)
        pix = np.empty((nj, ni), dtype=np.int32)
    st = Stats()
    rc = lib().oracle_shoot_block(
        ctypes.c_double(kappa), ctypes.c_double(gamma), ctypes.c_double(s), ctypes.c_double(L), ctypes.c_int(npix),
        ctypes.c_double(d), _p(xy, ctypes.c_float), _p(m, ctypes.c_float), ctypes.c_longlong(n),
        ctypes.c_longlong(i0), ctypes.c_longlong(j0), ctypes.c_longlong(ni), ctypes.c_longlong(nj),
        _p(count, ctypes.c_int), _p(y, ctypes.c_double), _p(al, ctypes.c_double), _p(sc, ctypes.c_double),
        _p(pix, ctypes.c_int), ctypes.byref(st), ctypes.c_int(n_threads))
    if rc != 0:
        raise ValueError("oracle_shoot_block: invalid parameters or block")
    out = {"count": count, "geometry": g,
           "stats": {k: int(getattr(st, k)) for k in ("rays_total", "rays_in_map", "rays_outside", "rays_lost")}}
    if want_rays:
        out.update(y=y, alpha=al, scale=sc, pix=pix)
    return out


def shoot_rays(kappa, gamma, s, L, npix, d, lens_xy, lens_m, ray_ij, n_threads=0):
    """Individual lattice rays (ray_ij int64 (n, 2) = (i, j)).  Returns dict(y, alpha, scale, pix)."""
    xy, m, n = _lens(lens_xy, lens_m)
    ij = np.ascontiguousarray(np.asarray(ray_ij, dtype=np.int64).reshape(-1, 2))
    nr = ij.shape[0]
    y = np.empty((nr, 2)); al = np.empty((nr, 2)); sc = np.empty((nr,)); pix = np.empty((nr,), dtype=np.int32)
    rc = lib().oracle_shoot_rays(
        ctypes.c_double(kappa), ctypes.c_double(gamma), ctypes.c_double(s), ctypes.c_double(L), ctypes.c_int(npix),
        ctypes.c_double(d), _p(xy, ctypes.c_float), _p(m, ctypes.c_float), ctypes.c_longlong(n),
        _p(ij, ctypes.c_longlong), ctypes.c_longlong(nr), _p(y, ctypes.c_double), _p(al, ctypes.c_double),
        _p(sc, ctypes.c_double), _p(pix, ctypes.c_int), ctypes.c_int(n_threads))
    if rc != 0:
        raise ValueError("oracle_shoot_rays: invalid parameters")
    return {"y": y, "alpha": al, "scale": sc, "pix": pix}


def map_points(kappa, gamma, s, lens_xy, lens_m, x, want_scale=False):
    """Eq. (1) at arbitrary image-plane positions x (n, 2) float64.  Returns (y, alpha) or, with ``want_scale``,
    (y, alpha, scale) where scale = sum_i m_i/|x - x_i| (the north_star's deflection-tolerance scale)."""
    xy, m, n = _lens(lens_xy, lens_m)
    x = np.ascontiguousarray(np.asarray(x, dtype=np.float64).reshape(-1, 2))
    y = np.empty_like(x); al = np.empty_like(x)
    sc = np.empty((x.shape[0],), dtype=np.float64) if want_scale else None
    lib().oracle_map_points(ctypes.c_double(kappa), ctypes.c_double(gamma), ctypes.c_double(s), _p(xy, ctypes.c_float),
                            _p(m, ctypes.c_float), ctypes.c_longlong(n), _p(x, ctypes.c_double),
                            ctypes.c_longlong(x.shape[0]), _p(y, ctypes.c_double), _p(al, ctypes.c_double),
                            _p(sc, ctypes.c_double))
    return (y, al, sc) if want_scale else (y, al)


def pixels_of(y, L, npix):
    y = np.ascontiguousarray(np.asarray(y, dtype=np.float64).reshape(-1, 2))
    pix = np.empty((y.shape[0],), dtype=np.int32)
    lib().oracle_pixels_of(_p(y, ctypes.c_double), ctypes.c_longlong(y.shape[0]), ctypes.c_double(L), ctypes.c_int(npix),
                           _p(pix, ctypes.c_int))
    return pix


def magnification(count, n_avg):
    c = np.ascontiguousarray(count, dtype=np.int32)
    mag = np.empty(c.shape, dtype=np.float32)
    lib().oracle_magnification(_p(c, ctypes.c_int), ctypes.c_longlong(c.size), ctypes.c_double(n_avg),
                               _p(mag, ctypes.c_float))
    return mag


def mpd(count, n_bins, n_avg):
    """Full MPD as the histogram of the integer counts + map means.  Returns
    (hist uint64 [n_bins], dict(n_pixels, sum_count, n_clamped, min_count, max_count, mean_count, mean_mu))."""
    c = np.ascontiguousarray(count, dtype=np.int32).reshape(-1)
    hist = np.empty((int(n_bins),), dtype=np.uint64)
    out = np.zeros((4,), dtype=np.int64)
    lib().oracle_mpd(_p(c, ctypes.c_int), ctypes.c_longlong(c.size), _p(hist, ctypes.c_ulonglong), ctypes.c_int(int(n_bins)),
                     _p(out, ctypes.c_longlong))
    mean = float(out[0]) / float(c.size)
    return hist, {"n_pixels": int(c.size), "sum_count": int(out[0]), "n_clamped": int(out[1]), "min_count": int(out[2]),
                  "max_count": int(out[3]), "mean_count": mean, "mean_mu": mean / float(n_avg)}


def profile_kernel(shape, size, npix):
    """Source-profile convolution kernel K (reading S19): float32 [npix, npix], sum 1, centre on (0,0)."""
    K = np.empty((int(npix), int(npix)), dtype=np.float32)
    lib().oracle_profile_kernel(ctypes.c_int(int(shape)), ctypes.c_double(float(size)), ctypes.c_int(int(npix)),
                                _p(K, ctypes.c_float))
    return K


def convolve(M, K, points=None):
    """Eq. 6 as its definition: circular convolution of float32 maps M and K in FP64.  points=None: the whole map
    (float64 [npix, npix]); else an (n, 2) integer array of (y, x) output pixels -> float64 [n]."""
    M = np.ascontiguousarray(M, dtype=np.float32)
    K = np.ascontiguousarray(K, dtype=np.float32)
    npix = M.shape[0]
    assert M.shape == (npix, npix) == K.shape
    if points is None:
        out = np.empty((npix, npix), dtype=np.float64)
        lib().oracle_convolve_at(_p(M, ctypes.c_float), _p(K, ctypes.c_float), ctypes.c_int(npix), None, ctypes.c_longlong(-1),
                                 _p(out, ctypes.c_double))
        return out
    pts = np.ascontiguousarray(points, dtype=np.int64).reshape(-1, 2)
    out = np.empty((pts.shape[0],), dtype=np.float64)
    lib().oracle_convolve_at(_p(M, ctypes.c_float), _p(K, ctypes.c_float), ctypes.c_int(npix), _p(pts, ctypes.c_longlong),
                             ctypes.c_longlong(pts.shape[0]), _p(out, ctypes.c_double))
    return out


def index_map(count):
    """Indexed map + index file.  Returns (values int32 [n_distinct] ascending, indexed int32 map)."""
    c = np.ascontiguousarray(count, dtype=np.int32)
    values = np.empty((c.size,), dtype=np.int32)
    indexed = np.empty(c.shape, dtype=np.int32)
    f = lib().oracle_index_map
    f.restype = ctypes.c_longlong
    n = f(_p(c, ctypes.c_int), ctypes.c_longlong(c.size), _p(values, ctypes.c_int), _p(indexed, ctypes.c_int))
    return values[:n].copy(), indexed


def bits_needed(max_value: int) -> int:
    """Smallest b >= 1 with max_value < 2**b (PAPER.md Table B.6)."""
    f = lib().oracle_bits_needed
    f.argtypes = [ctypes.c_ulonglong]
    return int(f(int(max_value)))


def pack_bits(values, bits: int):
    """Minimal-bit-width bit stream of non-negative integers < 2**bits: uint32 words."""
    v = np.ascontiguousarray(np.asarray(values).reshape(-1).astype(np.uint32))
    n_words = (v.size * int(bits) + 31) // 32
    packed = np.empty((n_words,), dtype=np.uint32)
    lib().oracle_pack_bits(_p(v, ctypes.c_uint), ctypes.c_longlong(v.size), ctypes.c_int(int(bits)), _p(packed, ctypes.c_uint),
                           ctypes.c_longlong(n_words))
    return packed


def unpack_bits(packed, n: int, bits: int):
    pk = np.ascontiguousarray(np.asarray(packed, dtype=np.uint32).reshape(-1))
    out = np.empty((int(n),), dtype=np.uint32)
    lib().oracle_unpack_bits(_p(pk, ctypes.c_uint), ctypes.c_longlong(int(n)), ctypes.c_int(int(bits)), _p(out, ctypes.c_uint))
    return out


def mpd_rebin(hist, n_avg, n_pixels, n_out, mu_min, mu_max):
    """Re-binned MPD (reading S20): float64 [n_out] probabilities in equal-width log10(mu) bins."""
    h = np.ascontiguousarray(np.asarray(hist, dtype=np.uint64).reshape(-1))
    prob = np.empty((int(n_out),), dtype=np.float64)
    lib().oracle_mpd_rebin(_p(h, ctypes.c_ulonglong), ctypes.c_int(h.size), ctypes.c_double(float(n_avg)),
                           ctypes.c_double(float(n_pixels)), ctypes.c_int(int(n_out)), ctypes.c_double(float(mu_min)),
                           ctypes.c_double(float(mu_max)), _p(prob, ctypes.c_double))
    return prob
