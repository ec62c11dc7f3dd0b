"""Many maps on one GPU: the way the paper actually scales.

GERLUMPH is ~70 000 independent maps "grouped in batches and submitted to the gSTAR job queue" (datasets
PAPER.md:221-233), one map per GPU at a time.  On a B200 a smooth-matter-dominated map (s = 0.9 ... 0.99: a few dozen
lenses, PAPER.md:111 puts the saturation point at N* ~ 300) is a sub-millisecond to sub-second kernel, so the per-map
host work — mlens_create, the launch, the device-to-host copy, mlens_destroy — is a visible share of a map.  This driver
hides it: K worker threads, each with its own CUDA stream, handle and device buffers, pull jobs from one queue; while one
thread creates or destroys a handle or waits for its copy, the other streams keep the GPU busy.  Results land in
caller-owned (pinned) host buffers.

One process drives one GPU; a node runs one such process per GPU (``bench.py --gpus N``: independent maps per rank, no
collective — weak scaling).  Host logic only: every ray is shot by the CUDA kernels behind the C ABI.
"""
from __future__ import annotations

import dataclasses
import queue
import threading
import time

import numpy as np

from . import fields, mlens


@dataclasses.dataclass
class MapJob:
    """One map of a survey: the arguments of mlens_create.  ``lens_xy`` / ``lens_m`` are the host arrays of the field."""

    cfg: fields.MapConfig
    lens_xy: np.ndarray
    lens_m: np.ndarray | None

    @classmethod
    def from_config(cls, cfg: fields.MapConfig) -> "MapJob":
        xy, m = fields.lens_field(cfg)
        return cls(cfg, xy, m)


def parameter_grid(base: fields.MapConfig, kappas, gammas, s_values, seed0: int | None = None) -> list[MapJob]:
    """Jobs over a (kappa, gamma, s) grid — the shape of the paper's parameter-space survey — with
    the map size, resolution and mass recipe of ``base``; seeds count up from ``seed0`` (default: base.seed)."""
    jobs, seed = [], base.seed if seed0 is None else seed0
    for k in kappas:
        for g in gammas:
            for s in s_values:
                jobs.append(MapJob.from_config(dataclasses.replace(base, kappa=float(k), gamma=float(g), s=float(s), seed=seed)))
                seed += 1
    return jobs


def run_survey(jobs: list[MapJob], n_streams: int = 2, want_mag: bool = True, out_count=None, out_mag=None) -> dict:
    """Shoot every job on the current CUDA device, ``n_streams`` maps in flight.

    ``out_count[i]`` / ``out_mag[i]``: caller-owned host arrays (int32 / float32, npix*npix of job i; pinned memory
    makes the copies asynchronous); allocated here as pinned tensors when None.  Returns ``{"stats": [per-job dict],
    "count": [...], "mag": [...], "seconds": wall time of the whole batch, "maps_per_s": ...}``.  Raises the first
    worker error.  Each worker issues ALL of a handle's work to its own stream and destroys it with
    mlens_destroy_on_stream, so no worker waits for another worker's map."""
    import torch

    if not torch.cuda.is_available():
        raise RuntimeError("run_survey needs a CUDA device; there is no CPU fallback")
    if n_streams < 1:
        raise ValueError("n_streams must be >= 1")
    mlens.lib()
    n = len(jobs)
    if out_count is None:
        out_count = [torch.empty((j.cfg.npix, j.cfg.npix), dtype=torch.int32, pin_memory=True) for j in jobs]
    if out_mag is None and want_mag:
        out_mag = [torch.empty((j.cfg.npix, j.cfg.npix), dtype=torch.float32, pin_memory=True) for j in jobs]
    as_tensor = lambda a: a if isinstance(a, torch.Tensor) else torch.from_numpy(a)  # noqa: E731
    host_count = [as_tensor(a) for a in out_count]
    host_mag = [as_tensor(a) for a in out_mag] if want_mag else None
    stats: list = [None] * n
    todo: queue.SimpleQueue = queue.SimpleQueue()
    for i in range(n):
        todo.put(i)
    errors: list = []
    device = torch.cuda.current_device()

    def worker():
        try:
            torch.cuda.set_device(device)
            stream = torch.cuda.Stream()
            dev_count = dev_mag = None
            with torch.cuda.stream(stream):
                while not errors:
                    try:
                        i = todo.get_nowait()
                    except queue.Empty:
                        break
                    job = jobs[i]
                    npix = job.cfg.npix
                    if dev_count is None or dev_count.shape[0] != npix:  # device buffers are reused from map to map
                        dev_count = torch.empty((npix, npix), dtype=torch.int32, device="cuda")
                        dev_mag = torch.empty((npix, npix), dtype=torch.float32, device="cuda") if want_mag else None
                    h = mlens.Mlens.from_config(job.cfg, job.lens_xy, job.lens_m)
                    try:
                        h.shoot(count=dev_count, mag=dev_mag, want_mag=want_mag, stream=stream, sync=False)
                        host_count[i].copy_(dev_count, non_blocking=True)
                        if want_mag:
                            host_mag[i].copy_(dev_mag, non_blocking=True)
                        stats[i] = h.stats(stream)  # synchronises THIS stream: the map and its copies are done
                    finally:
                        h.close(stream)
        except BaseException as exc:  # noqa: BLE001 — handed to the caller's thread
            errors.append(exc)

    torch.cuda.synchronize()
    t0 = time.perf_counter()
    threads = [threading.Thread(target=worker, name=f"mlens-survey-{k}") for k in range(min(n_streams, max(1, n)))]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    if errors:
        raise errors[0]
    return {"stats": stats, "count": out_count, "mag": out_mag, "seconds": dt, "maps_per_s": n / dt if dt > 0 else float("inf"),
            "n_streams": len(threads)}
