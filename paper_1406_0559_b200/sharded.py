"""One map on several GPUs: row-band sharding of the ray lattice + ONE integer all-reduce.

Rays are independent and the only shared state is the additive int32 count map ("accumulated on a gridded
source plane"), so the lattice rows j are cut into contiguous bands, one per rank.  Every rank holds the full lens list
(<= 320 KB) and a private count map; after shooting its band through ``mlens_shoot_block`` the maps are summed with one
``all_reduce`` (NCCL over NVLink on GPUs; gloo in the CPU tests).  Bands start on multiples of the kernel's 64-ray tile,
so every ray sees exactly the tile centre it sees in the single-GPU launch: the summed map is BIT-IDENTICAL to the
1-GPU map for any number of ranks (integer sums commute).

The collective is one 4*Npix^2-byte message per map (4 MB ... 381.5 MB, i.e. ~ms on NVLink 5) after seconds of
shooting, so it is not fused into the shooting kernel: there is nothing to overlap it with.  The paper itself scales
differently — one independent map per GPU through a batch queue — which is what
``bench.py --gpus N`` does by default; ``bench.py --gpus N --shard`` times this module instead.

This module is host logic only (band plan + the reduction); every ray is shot by the CUDA kernels behind the C ABI.
"""
from __future__ import annotations

TILE = 64  # rays per tile side of shoot_fp32_kernel (csrc/shoot_kernel.cuh: kTile); bands are aligned to it


def row_bands(n2: int, world: int, tile: int = TILE) -> list[tuple[int, int]]:
    """Contiguous (j0, nj) bands covering [0, n2), one per rank, each starting on a multiple of ``tile``.

    Tiles (not rows) are dealt out as evenly as possible: the first ``n_tiles % world`` ranks get one tile more.  A rank
    can get an empty band (nj = 0) when there are fewer tiles than ranks."""
    if n2 < 0 or world < 1 or tile < 1:
        raise ValueError("row_bands: n2 >= 0, world >= 1, tile >= 1 required")
    n_tiles = (n2 + tile - 1) // tile
    base, extra = divmod(n_tiles, world)
    bands, t0 = [], 0
    for r in range(world):
        nt = base + (1 if r < extra else 0)
        j0 = min(t0 * tile, n2)
        j1 = min((t0 + nt) * tile, n2)
        bands.append((j0, j1 - j0))
        t0 += nt
    return bands


def allreduce_map(count, counters, group=None):
    """Sum the per-rank count maps (int32 tensor, in place) and the 4 ray counters (int64 tensor: in_map, outside,
    lost, total) over ``group``.  Works on whatever backend the tensors' device needs (nccl for CUDA, gloo for CPU)."""
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(count, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(counters, op=dist.ReduceOp.SUM, group=group)
    return count, counters


def shoot_sharded(h, rank: int, world: int, count=None, mag=None, want_mag=True, group=None, stream=None, device="cuda"):
    """Shoot rank ``rank``'s row band of ``h``'s lattice, all-reduce the maps, then Eq. 4 on the summed map.

    ``h`` is a ``mlens.Mlens`` created with the SAME parameters and lens arrays on every rank.  Returns
    (count, mag or None, stats dict) — identical on every rank.  ``stats['band']`` is this rank's (j0, nj).

    Only five members of ``h`` are used — ``geometry`` (n1, n2), ``npix``, ``reset_stats``, ``shoot_block``, ``stats`` and
    ``magnification`` — so the multi-process CPU test (tests/test_sharded.py, gloo, world_size 2) drives THIS function
    with a stand-in handle whose band shooter is the oracle and ``device="cpu"``; the product always passes a
    ``mlens.Mlens`` and CUDA tensors."""
    import torch

    g = h.geometry
    if count is None:
        count = torch.empty((h.npix, h.npix), dtype=torch.int32, device=device)
    count.zero_()
    h.reset_stats(stream)
    j0, nj = row_bands(g.n2, world)[rank]
    if nj > 0:
        h.shoot_block(0, j0, g.n1, nj, count=count, stream=stream)
    st = h.stats(stream)  # synchronises the stream
    counters = torch.tensor([st["rays_in_map"], st["rays_outside"], st["rays_lost"], st["rays_total"]],
                            dtype=torch.int64, device=count.device)
    allreduce_map(count, counters, group)
    if want_mag:
        mag = h.magnification(count, mag, stream)  # also refreshes max_count on the summed map
    c = [int(v) for v in counters.tolist()]
    out = dict(st, rays_in_map=c[0], rays_outside=c[1], rays_lost=c[2], rays_total=c[3], band=(j0, nj))
    if want_mag:
        out["max_count"] = h.stats(stream)["max_count"]
    return count, (mag if want_mag else None), out
