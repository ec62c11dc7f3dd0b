"""Seeded synthetic lens fields and the five workload configurations.

This module is the ONE piece shared by the FP64 oracle's tests and the CUDA path: it only *generates inputs*
(configuration parameters, lens positions, lens masses).  It contains none of the method's arithmetic — no lens
equation, no ray lattice, no binning.  The lattice (n1, n2) is derived independently inside ``oracle/`` and inside
``libmlens.so``.

What the paper fixes (Eq. 3; Fig. 1 caption PAPER.md:103): N* = kappa_* A / (pi <M>) lenses
"distributed in a circle of area A", random positions, mass spectrum a parameter.  Everything else
(rectangle margin 1.2, disc radius R* = 1.2 x half-diagonal, Salpeter slope) is BASELINE.json's construction rule.

The paper's own lens files (``lenspos.dat``) and map sets are not available; these seeded fields stand
in for them ("Input recipe").

Generator: splitmix64 used as a counter-based generator (value k = mix(seed + (k+1)*GOLDEN)), 53-bit uniforms,
rejection sampling from the square for the disc (no libm trig => reproducible bit for bit across hosts).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, start: int, count: int) -> np.ndarray:
    """Values start..start+count-1 of the splitmix64 stream seeded with ``seed`` (uint64 array)."""
    with np.errstate(over="ignore"):
        k = np.arange(start + 1, start + count + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + k * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, start: int, count: int) -> np.ndarray:
    """53-bit uniforms in [0, 1) from the splitmix64 stream (float64 array)."""
    return (splitmix64(seed, start, count) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


@dataclasses.dataclass(frozen=True)
class MapConfig:
    """One workload: the arguments of ``mlens_create`` minus the lens arrays, plus the field recipe."""

    name: str
    npix: int
    map_side: float  # L, in Einstein radii of the mean mass
    kappa: float
    gamma: float
    s: float  # smooth-matter fraction kappa_s / kappa (Eq. 2)
    sub: int  # pixel / ray_spacing
    masses: str  # "unit" | "salpeter"
    seed: int
    margin: float = 1.2

    @property
    def pixel(self) -> float:
        return self.map_side / self.npix

    @property
    def ray_spacing(self) -> float:
        return self.map_side / self.npix / self.sub

    @property
    def kappa_star(self) -> float:
        return (1.0 - self.s) * self.kappa

    @property
    def half_widths(self) -> tuple[float, float]:
        """Half-widths (a1, a2) of the image-plane shooting rectangle (BASELINE.json config rule)."""
        h = self.margin * (self.map_side / 2.0)
        return (h / abs(1.0 - self.kappa - self.gamma), h / abs(1.0 - self.kappa + self.gamma))

    @property
    def map_half_image(self) -> tuple[float, float]:
        """Half-widths of the map's pre-image under the macro-model alone: (L/2)/|1-kappa-+gamma| = half_widths/margin."""
        a1, a2 = self.half_widths
        return (a1 / self.margin, a2 / self.margin)

    @property
    def disc_radius(self) -> float:
        a1, a2 = self.half_widths
        return self.margin * math.sqrt(a1 * a1 + a2 * a2)

    @property
    def n_lens(self) -> int:
        """Eq. 3 with A = pi R*^2 and <M> = 1."""
        r = self.disc_radius
        return int(round(self.kappa_star * r * r))

    @property
    def mu_th(self) -> float:
        """Macro-magnification 1/|(1-kappa)^2 - gamma^2|."""
        return 1.0 / abs((1.0 - self.kappa) ** 2 - self.gamma**2)


# BASELINE.json "configs" (1-based numbering as in SURVEY.md §8(d)); seeds 1000*cfg + 1.
CONFIGS: dict[int, MapConfig] = {
    1: MapConfig("cfg1_tiny", 256, 4.0, 0.3, 0.2, 0.0, 10, "unit", 1001),
    2: MapConfig("cfg2_dense_2048", 2048, 25.0, 0.6, 0.3, 0.0, 10, "unit", 2001),
    3: MapConfig("cfg3_smooth_4096", 4096, 25.0, 0.5, 0.3, 0.9, 8, "unit", 3001),
    4: MapConfig("cfg4_nearcritical_1024", 1024, 5.0, 0.9, 0.0, 0.0, 10, "salpeter", 4001),
    5: MapConfig("cfg5_production_10000", 10000, 25.0, 0.3, 0.3, 0.0, 8, "unit", 5001),
}


def disc_positions(n: int, radius: float, seed: int) -> np.ndarray:
    """n points uniform in the disc of ``radius`` centred on the origin; float64 array (n, 2).

    Rejection from the enclosing square: candidate c uses stream values 2c and 2c+1; the first n accepted
    candidates are returned in stream order.
    """
    if n == 0:
        return np.zeros((0, 2), dtype=np.float64)
    out = np.empty((n, 2), dtype=np.float64)
    got, start = 0, 0
    while got < n:
        m = max(64, int((n - got) * 1.4) + 16)
        u = uniform01(seed, 2 * start, 2 * m)
        cx = 2.0 * u[0::2] - 1.0
        cy = 2.0 * u[1::2] - 1.0
        ok = cx * cx + cy * cy < 1.0
        take = min(n - got, int(ok.sum()))
        out[got : got + take, 0] = cx[ok][:take]
        out[got : got + take, 1] = cy[ok][:take]
        got += take
        start += m
    return out * radius


def salpeter_masses(n: int, seed: int, slope: float = 2.35, m_lo: float = 0.01, m_hi: float = 1.0) -> np.ndarray:
    """n masses from dN/dm ~ m^-slope on [m_lo, m_hi] by inverse CDF, divided by the SAMPLE mean (float64)."""
    if n == 0:
        return np.zeros((0,), dtype=np.float64)
    u = uniform01(seed ^ 0x5A17E7E5, 0, n)
    e = 1.0 - slope
    lo, hi = m_lo**e, m_hi**e
    m = (lo + u * (hi - lo)) ** (1.0 / e)
    return m / m.mean()


def lens_field(cfg: MapConfig) -> tuple[np.ndarray, np.ndarray]:
    """(lens_xy float32 (N*, 2) interleaved x,y ; lens_m float32 (N*,)) — the canonical FP32 inputs of BOTH sides."""
    n = cfg.n_lens
    xy = disc_positions(n, cfg.disc_radius, cfg.seed).astype(np.float32)
    if cfg.masses == "unit":
        m = np.ones((n,), dtype=np.float32)
    elif cfg.masses == "salpeter":
        m = salpeter_masses(n, cfg.seed).astype(np.float32)
    else:
        raise ValueError(f"unknown mass spectrum {cfg.masses!r}")
    return np.ascontiguousarray(xy), np.ascontiguousarray(m)


def random_field(n: int, radius: float, seed: int, masses: str = "unit") -> tuple[np.ndarray, np.ndarray]:
    """Free-form seeded field for tests (same generators, arbitrary n / radius)."""
    xy = disc_positions(n, radius, seed).astype(np.float32)
    m = np.ones((n,), np.float32) if masses == "unit" else salpeter_masses(n, seed).astype(np.float32)
    return np.ascontiguousarray(xy), np.ascontiguousarray(m)


def block_plan(n1: int, n2: int, lens_xy: np.ndarray, half_widths: tuple[float, float], d: float, seed: int,
               n_random: int = 32, n_lens_centred: int = 16, n_border: int = 8, size: int = 256,
               n_straddle: int = 0, n_inside: int = 0, map_half_image: tuple[float, float] | None = None
               ) -> list[tuple[int, int, int, int]]:
    """Seeded (i0, j0, ni, nj) ray sub-blocks for parity at the large configs (SURVEY.md §8(d) sub-block plan).

    Random unaligned blocks, blocks centred on lenses (near-lens path), blocks touching the lattice border, and — when
    ``map_half_image`` = (b1, b2) is given — blocks that straddle / lie inside the image-plane rectangle |x1| < b1,
    |x2| < b2 (the caller passes the pre-image of the map under the macro-model, b = (L/2)/|1-kappa-+gamma| =
    half_width/margin: the region whose rays the macro-model alone would send into the map, so that the compared sample
    holds in-map rays).  Pure index bookkeeping: which rays to compare, not how they are shot.
    """
    sx, sy = min(size, n1), min(size, n2)
    u = uniform01(seed ^ 0xB10C, 0, 4 * (n_random + n_lens_centred + n_border) + 8)
    blocks: list[tuple[int, int, int, int]] = []
    k = 0
    for _ in range(n_random):
        blocks.append((int(u[k] * (n1 - sx + 1)), int(u[k + 1] * (n2 - sy + 1)), sx, sy))
        k += 2
    a1, a2 = half_widths
    inside = [q for q in range(len(lens_xy)) if abs(lens_xy[q, 0]) < a1 and abs(lens_xy[q, 1]) < a2]
    for t in range(n_lens_centred):
        if not inside:
            break
        q = inside[int(u[k] * len(inside))]
        k += 1
        ic = int(math.floor(float(lens_xy[q, 0]) / d + n1 / 2.0))
        jc = int(math.floor(float(lens_xy[q, 1]) / d + n2 / 2.0))
        i0 = min(max(ic - sx // 2 + (t % 7), 0), n1 - sx)
        j0 = min(max(jc - sy // 2 + (t % 5), 0), n2 - sy)
        blocks.append((i0, j0, sx, sy))
    for t in range(n_border):
        r = int(u[k] * max(1, (n2 - sy if t % 2 == 0 else n1 - sx)))
        k += 1
        if t % 4 == 0:
            blocks.append((0, r, sx, sy))
        elif t % 4 == 1:
            blocks.append((r, 0, sx, sy))
        elif t % 4 == 2:
            blocks.append((n1 - sx, r, sx, sy))
        else:
            blocks.append((r, n2 - sy, sx, sy))
    if (n_straddle or n_inside) and map_half_image is not None:
        b1, b2 = map_half_image
        v = uniform01(seed ^ 0x57AD, 0, 2 * (n_straddle + n_inside) + 2)
        # lattice index of image-plane position x along an axis with n rays: x = (i + 1/2 - n/2) d
        def idx(x, n):
            return int(math.floor(x / d + n / 2.0))

        def clamp(i0, n, sz):
            return min(max(i0, 0), n - sz)

        k = 0
        for t in range(n_straddle):  # block centred on one of the four edges of the map's macro pre-image
            r = 2.0 * v[k] - 1.0
            k += 1
            side = -1.0 if (t // 2) % 2 == 0 else 1.0
            if t % 2 == 0:   # an edge x1 = +-b1, anywhere along it
                ic, jc = idx(side * b1, n1), idx(0.9 * r * b2, n2)
            else:            # an edge x2 = +-b2
                ic, jc = idx(0.9 * r * b1, n1), idx(side * b2, n2)
            blocks.append((clamp(ic - sx // 2, n1, sx), clamp(jc - sy // 2, n2, sy), sx, sy))
        for t in range(n_inside):    # block well inside the pre-image (central 80 %)
            ic, jc = idx(0.8 * (2.0 * v[k] - 1.0) * b1, n1), idx(0.8 * (2.0 * v[k + 1] - 1.0) * b2, n2)
            k += 2
            blocks.append((clamp(ic - sx // 2, n1, sx), clamp(jc - sy // 2, n2, sy), sx, sy))
    return blocks
