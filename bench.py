#!/usr/bin/env python
"""bench.py — throughput of the direct inverse ray-shooting hot path (BASELINE.json metric) on B200.

A "step" is one pass of the whole hot path (lattice, deflection sum over all N* lenses,
source position, binning, count -> magnification) over one synthetic map.  The default workload is BASELINE.json's
config 4 (`configs[3]`, the near-critical 1024^2 field the north_star quotes its FP32 target on); `--config` selects
another.  One JSON line is printed by rank 0.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

* `value`      ray-lens interactions/s, all ranks, device-timed (CUDA events on the launching stream), max over ranks.
* `e2e`        the same metric through `mlens_create` + `mlens_shoot_host` + `mlens_destroy` with HOST buffers (lens
               arrays in, count + magnification maps out into pinned host memory), copies inside the timed region.
* `roofline`   the shooting kernel alone: 11 flops x interactions / kernel time (events inside libmlens around the
               kernel launch) against the FP32 peak SMs x 128 x 2 x f_max; bound = "alu".
               `peak_measured` / `frac_of_measured`: the scalar-FFMA rate measured on this box just before the timed
               region by bench/alu_microbench --fp32-peak (MEASURED_PEAKS.json holds no FP32 figure), with the SM clock
               observed inside that kernel.  `traffic`: DRAM bytes of one launch from the tracked ncu capture named in
               `traffic_source` (null when no capture of the committed kernel exists for the workload).
* `cpu_baseline` the FP64 oracle (oracle/) on the box's host cores on a bounded block of the same lattice.
* N > 1        weak scaling: every rank shoots an independent map of the same config (seed + rank), the way the paper
               scales (one map per GPU); no data-path collective.
* `--impl reference`  times the oracle, as it stands, on the host cores (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1406_0559_b200 import fields  # noqa: E402

METRIC = "ray_lens_interactions_per_s"
UNIT = "interactions/s"
FLOPS_PER_INTERACTION = 11  # 2 sub, mul+fma (r^2), rcp, mass mul, 2 fma (10 when all m_i = 1)
FP32_LANES_PER_SM = 128


def flops_per_interaction(cfg) -> int:
    return FLOPS_PER_INTERACTION if cfg.masses != "unit" else FLOPS_PER_INTERACTION - 1


def workload_name(cfg_id: int, cfg, n_lens: int, n1: int, n2: int) -> str:
    return (f"BASELINE.json config {cfg_id} ({cfg.name}): {cfg.npix}^2 px, side {cfg.map_side:g} R_E, kappa={cfg.kappa:g}, "
            f"gamma={cfg.gamma:g}, s={cfg.s:g}, spacing=pixel/{cfg.sub}, masses={cfg.masses}, N*={n_lens}, "
            f"lattice {n1}x{n2}")


# -----------------------------------------------------------------------------------------------------------------
# clocks
# -----------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi sampled every 200 ms during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, smax, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_min_mhz": min(sm), "sm_max_mhz": max(smax), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


# -----------------------------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline and --impl reference): the ONLY places bench.py touches oracle/
# -----------------------------------------------------------------------------------------------------------------
def oracle_block_for(cfg, n1, n2, n_lens, target_s, rate_guess):
    """A centred ni x nj block of the config's lattice holding about target_s seconds of oracle work."""
    rays = max(4096.0, target_s * rate_guess / max(1, n_lens))
    side = int(max(64, min(min(n1, n2), round(rays**0.5))))
    return ((n1 - side) // 2, (n2 - side) // 2, side, side)


_ORACLE_THREADS = 0  # 0 = OpenMP's own choice; the reference arm under a multi-rank launcher sets it (see run_reference)


def oracle_time_block(oracle, cfg, xy, m, block):
    t0 = time.perf_counter()
    r = oracle.shoot_block(cfg.kappa, cfg.gamma, cfg.s, cfg.map_side, cfg.npix, cfg.ray_spacing, xy, m, block=block,
                           n_threads=_ORACLE_THREADS)
    dt = time.perf_counter() - t0
    return dt, r["stats"]["rays_total"]


def oracle_calibrate(oracle, cfg, xy, m, n1, n2):
    """Rate (interactions/s) from a short run, used only to SIZE the timed sample."""
    n_lens = max(1, len(m))
    blk = oracle_block_for(cfg, n1, n2, n_lens, 1.0, 2.0e9)
    dt, rays = oracle_time_block(oracle, cfg, xy, m, blk)
    return rays * n_lens / max(dt, 1e-6)


def run_cpu_baseline(cfg, xy, m, target_s=15.0):
    import oracle

    oracle.lib()
    g = oracle.geometry(cfg.kappa, cfg.gamma, cfg.s, cfg.map_side, cfg.npix, cfg.ray_spacing)
    n_lens = max(1, len(m))
    rate0 = oracle_calibrate(oracle, cfg, xy, m, g.n1, g.n2)
    blk = oracle_block_for(cfg, g.n1, g.n2, n_lens, target_s, rate0)
    dt, rays = oracle_time_block(oracle, cfg, xy, m, blk)
    return {"value": rays * n_lens / dt, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
            "rays_per_s": rays / dt, "seconds": dt,
            "sample": f"centred {blk[2]}x{blk[3]}-ray block of the same lattice ({rays} rays x {n_lens} lenses = "
                      f"{rays * n_lens:.3e} interactions), FP64 C++ -O3 -march=native, OpenMP, oracle/oracle.cpp as it stands"}


def run_reference(args):
    """--impl reference: the oracle on the host cores, K timed steps of a bounded sample each (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        print(f"bench.py: rank {os.environ['RANK']} of {os.environ.get('WORLD_SIZE', '?')}: idle (the reference arm runs on rank 0 only)",
              file=sys.stderr, flush=True)
        return
    import oracle

    oracle.lib()
    global _ORACLE_THREADS
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        # torch.distributed.run exports OMP_NUM_THREADS=1 to every rank; here the other ranks idle, so rank 0 takes the
        # host cores this process may run on — the same machine share the N = 1 reference run gets
        _ORACLE_THREADS = len(os.sched_getaffinity(0))
    cfg = fields.CONFIGS[args.config]
    xy, m = fields.lens_field(cfg)
    g = oracle.geometry(cfg.kappa, cfg.gamma, cfg.s, cfg.map_side, cfg.npix, cfg.ray_spacing)
    n_lens = max(1, len(m))
    rate0 = oracle_calibrate(oracle, cfg, xy, m, g.n1, g.n2)
    per_step = min(8.0, 120.0 / max(1, args.steps + args.warmup))
    blk = oracle_block_for(cfg, g.n1, g.n2, n_lens, per_step, rate0)
    for _ in range(args.warmup):
        oracle_time_block(oracle, cfg, xy, m, blk)
    t0 = time.perf_counter()
    rays = 0
    for _ in range(args.steps):
        _, r = oracle_time_block(oracle, cfg, xy, m, blk)
        rays += r
    dt = time.perf_counter() - t0
    value = rays * n_lens / dt
    sample = (f"each step: centred {blk[2]}x{blk[3]}-ray block of the config's lattice ({blk[2] * blk[3] * n_lens:.3e} "
              f"interactions), FP64 oracle on host cores")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, cfg, len(m), g.n1, g.n2), "sample": sample},
            "rays_per_s": rays / dt,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": _ORACLE_THREADS or oracle.max_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# -----------------------------------------------------------------------------------------------------------------
# roofline inputs that are measured, not derived
# -----------------------------------------------------------------------------------------------------------------
def measure_fp32_peak(device_index: int):
    """Scalar-FFMA rate of this GPU, measured now (bench/alu_microbench --fp32-peak, ~0.1 s).  None if it is not built."""
    exe = os.path.join(ROOT, "bench", "alu_microbench")
    if not os.path.exists(exe):
        return None
    try:
        r = subprocess.run([exe, "--fp32-peak", str(device_index)], capture_output=True, text=True, timeout=120)
        return json.loads(r.stdout.strip().splitlines()[-1]) if r.returncode == 0 else None
    except (OSError, ValueError, IndexError, subprocess.TimeoutExpired):
        return None


def load_traffic(cfg_id: int, shard: bool):
    """DRAM bytes (read + write) of ONE shooting-kernel launch of this workload from the tracked ncu capture of the
    committed kernel, profiles/traffic_shoot_cfg<N>.json ({"dram_bytes_read", "dram_bytes_write", "command", ...}), or
    (None, reason).  Never a literal in this file: the number and the command that produced it live under profiles/."""
    if shard:
        return None, "not captured for the sharded launch"
    path = os.path.join(ROOT, "profiles", f"traffic_shoot_cfg{cfg_id}.json")
    if not os.path.exists(path):
        return None, f"no ncu capture of the committed kernel for config {cfg_id} under profiles/"
    t = json.load(open(path))
    return int(t["dram_bytes_read"]) + int(t["dram_bytes_write"]), f"profiles/traffic_shoot_cfg{cfg_id}.json ({t.get('command', '')})"


def make_line(*, cfg_id, cfg, n_lens, n1, n2, world, shard, steps, warmup, ms_total, kern_ms, in_map, clocks, sms,
              e2e_s, e2e_steps, h2d_bytes, d2h_bytes, peak_meas=None, traffic=None, traffic_source=None):
    """The bench JSON line from the measured numbers (pure function: tests/test_bench_contract.py checks the contract)."""
    rays = n1 * n2
    inter = rays * max(1, n_lens)
    f_max_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak = sms * FP32_LANES_PER_SM * 2 * f_max_mhz * 1e6 / 1e12  # TFLOP/s at the maximum SM clock
    fpi = flops_per_interaction(cfg)
    # shard mode: each rank's kernel covers 1/world of the interactions (kern_ms then also holds the all-reduce)
    achieved = fpi * (inter / (world if shard else 1)) / (kern_ms * 1e-3) / 1e12
    maps = 1 if shard else world
    roof = {"bound": "alu", "kernel": "shoot_fp32_kernel", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
            "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_source,
            "algorithmic_bytes": 4 * cfg.npix**2 + 16 * n_lens,  # the count map written once + the lens list read once
            "flops_per_interaction": fpi, "kernel_ms": kern_ms,
            "peak_source": f"derived: {sms} SMs x 128 FP32 lanes x 2 x {f_max_mhz:.0f} MHz (clocks.max.sm); "
                           "no FP32 figure in MEASURED_PEAKS.json",
            "mufu_ceiling_frac": 16.0 * fpi / (FP32_LANES_PER_SM * 2)}
    if peak_meas:
        roof.update(peak_measured=peak_meas["fp32_tflops"], frac_of_measured=achieved / peak_meas["fp32_tflops"],
                    peak_measured_sm_mhz=peak_meas.get("sm_mhz_observed"),
                    peak_measured_source="bench/alu_microbench --fp32-peak on this GPU just before the timed region: "
                                         + peak_meas.get("how", ""))
    return {
        "metric": METRIC, "value": maps * inter * steps / (ms_total * 1e-3), "unit": UNIT, "n_gpus": world, "steps": steps,
        "warmup": warmup, "ms_per_step": ms_total / max(1, steps), "higher_is_better": True,
        "scaling": "strong" if shard else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg_id, cfg, n_lens, n1, n2), "rays_per_map": rays,
                   "interactions_per_map": inter, "rays_in_map": in_map,
                   "mean_mu_over_mu_th": in_map / (cfg.npix**2 * cfg.sub**2) / cfg.mu_th,
                   "l2": "256 MiB device write between steps (inputs are smaller than L2)",
                   "parallelism": (f"one map, {world} row bands + one int32 all-reduce" if shard else
                                   f"{world} independent map(s), one per GPU (seed + rank)")},
        "rays_per_s": maps * rays * steps / (ms_total * 1e-3),
        "clocks": clocks,
        "e2e": {"value": maps * inter * e2e_steps / e2e_s, "unit": UNIT, "steps": e2e_steps,
                "h2d_bytes_per_step": int(h2d_bytes), "d2h_bytes_per_step": int(d2h_bytes)},
        # our kernels launched inside the timed region, by construction of mlens_shoot: one shooting kernel and one
        # magnification kernel per step (the memsets are driver operations; the L2 flush is torch's fill)
        "gpu_launches": 2 * steps,
        "roofline": roof,
    }


# -----------------------------------------------------------------------------------------------------------------
# our arm
# -----------------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_1406_0559_b200 import mlens, sharded

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    mlens.lib()  # fail loudly if libmlens.so is missing
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    import dataclasses

    cfg0 = fields.CONFIGS[args.config]
    shard = bool(args.shard) and world > 1
    # default N > 1: weak scaling, an independent map per rank (the paper's way); --shard: ONE map, row bands per rank
    cfg = cfg0 if shard else dataclasses.replace(cfg0, seed=cfg0.seed + rank)
    xy, m = fields.lens_field(cfg)
    n_lens = len(m)
    h = mlens.Mlens.from_config(cfg, xy, m)
    g = h.geometry
    rays = g.n1 * g.n2
    inter = rays * max(1, n_lens)
    count = torch.empty((cfg.npix, cfg.npix), dtype=torch.int32, device="cuda")
    mag = torch.empty((cfg.npix, cfg.npix), dtype=torch.float32, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    def step(sync_stats=False):
        flush.fill_(1)  # evict the count map and lens list from L2 between steps
        if shard:
            t0k, t1k = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0k.record()
            st_ = sharded.shoot_sharded(h, rank, world, count=count, mag=mag)[2]
            t1k.record()
            torch.cuda.synchronize()
            st_["kernel_ms"] = t0k.elapsed_time(t1k)  # band kernel + all-reduce + Eq. 4
            return st_
        return h.shoot(count=count, mag=mag, sync=sync_stats)[2]

    for _ in range(args.warmup):
        step()
    barrier()
    # measured FP32 peak of THIS box, taken after the warm-up (clocks ramped) and before the timed region (rank 0's GPU)
    peak_meas = measure_fp32_peak(local_rank) if rank == 0 else None
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    kernel_ms = []
    for _ in range(args.steps):
        st = step(sync_stats=True)  # stats pointer => libmlens brackets the shooting kernel with its own events
        kernel_ms.append(st["kernel_ms"])
    ev1.record()
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if rank == 0 else None
    t = torch.tensor([ms_total, sum(kernel_ms) / max(1, len(kernel_ms))], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total, kern_ms = float(t[0]), float(t[1])
    assert st["rays_total"] == rays and st["rays_in_map"] + st["rays_outside"] + st["rays_lost"] == rays
    in_map = st["rays_in_map"]

    # end to end through the C ABI with host buffers: create (H2D lens list) + shoot + D2H maps + destroy
    # maps of seconds: two end-to-end maps; maps shorter than a second: as many as --steps (capped), a usable statistic
    e2e_steps = max(1, min(args.steps, 2 if ms_total / max(1, args.steps) >= 1000.0 else 50))
    h.close()
    barrier()
    e2e_kernel_ms = []
    # the caller's result buffers: pinned host memory, allocated once and reused for every map (as a survey would)
    c_pin = torch.empty((cfg.npix, cfg.npix), dtype=torch.int32, pin_memory=True)
    m_pin = torch.empty((cfg.npix, cfg.npix), dtype=torch.float32, pin_memory=True)
    e2e_phase_ms = []  # host clock per step: [mlens_create (H2D of the lens list), shoot + D2H, mlens_destroy]
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ta = time.perf_counter()
        h2 = mlens.Mlens.from_config(cfg, xy, m)
        tb = time.perf_counter()
        if shard:
            c_dev, m_dev, st2 = sharded.shoot_sharded(h2, rank, world)
            c_host, m_host = c_dev.cpu().numpy(), m_dev.cpu().numpy()
        else:
            c_host, m_host, st2 = h2.shoot_host(count=c_pin.numpy(), mag=m_pin.numpy())
        tc = time.perf_counter()
        h2.close()
        td = time.perf_counter()
        e2e_kernel_ms.append(st2.get("kernel_ms"))
        e2e_phase_ms.append([round(1e3 * (tb - ta), 3), round(1e3 * (tc - tb), 3), round(1e3 * (td - tc), 3)])
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_s = float(t[0])
    assert int(c_host.sum(dtype=np.int64)) == st2["rays_in_map"] == in_map

    if rank == 0:
        prop = torch.cuda.get_device_properties(local_rank)
        traffic, traffic_source = load_traffic(args.config, shard)
        line = make_line(cfg_id=args.config, cfg=cfg0, n_lens=n_lens, n1=g.n1, n2=g.n2, world=world, shard=shard,
                         steps=args.steps, warmup=args.warmup, ms_total=ms_total, kern_ms=kern_ms, in_map=in_map,
                         clocks=clocks, sms=prop.multi_processor_count, e2e_s=e2e_s, e2e_steps=e2e_steps,
                         h2d_bytes=xy.nbytes + m.nbytes, d2h_bytes=c_host.nbytes + m_host.nbytes, peak_meas=peak_meas,
                         traffic=traffic, traffic_source=traffic_source)
        line["e2e"]["kernel_ms_per_step"] = e2e_kernel_ms  # of which: the shooting kernel (events inside libmlens)
        line["e2e"]["host_ms_per_step_create_shoot_destroy"] = e2e_phase_ms
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = run_cpu_baseline(cfg, xy, m)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_block(args):
    """--block S: K launches of mlens_shoot_block on a centred S x S-ray block (the short launch ncu profiles)."""
    import torch

    from paper_1406_0559_b200 import mlens

    torch.cuda.set_device(0)
    cfg = fields.CONFIGS[args.config]
    xy, m = fields.lens_field(cfg)
    with mlens.Mlens.from_config(cfg, xy, m, ablations=args.ablations) as h:
        for k, v in (args.option or []):
            h.set_option(k, int(v))
        g = h.geometry
        si, sj = min(args.block, g.n1), min(args.block, g.n2)
        blk = ((g.n1 - si) // 2, (g.n2 - sj) // 2, si, sj)
        count = torch.zeros((cfg.npix, cfg.npix), dtype=torch.int32, device="cuda")
        for _ in range(args.warmup):
            h.shoot_block(*blk, count=count)
        torch.cuda.synchronize()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
        ev[0].record()
        for k in range(args.steps):
            h.shoot_block(*blk, count=count)
            ev[k + 1].record()
        torch.cuda.synchronize()
        ms = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
        st = h.stats()
    inter = si * sj * max(1, len(m))
    med = statistics.median(ms)
    fpi = flops_per_interaction(cfg)
    print(json.dumps({"mode": "block", "config": args.config, "block": blk, "options": args.option, "ms": ms, "ms_median": med,
                      "interactions_per_s": inter / (med * 1e-3), "rays_per_s": si * sj / (med * 1e-3),
                      "tflops": fpi * inter / (med * 1e-3) / 1e12,
                      "frac_fp32_peak_1965": fpi * inter / (med * 1e-3) / (148 * 128 * 2 * 1.965e9),
                      "rays_in_map_frac": st["rays_in_map"] / max(1, st["rays_total"])}), flush=True)


def run_mpd(args):
    """--mpd: K launches of mlens_mpd (row f1: MPD histogram + map means) on the config's shot map; HBM roofline."""
    import torch

    from paper_1406_0559_b200 import mlens

    torch.cuda.set_device(0)
    cfg = fields.CONFIGS[args.config]
    xy, m = fields.lens_field(cfg)
    with mlens.Mlens.from_config(cfg, xy, m) as h:
        count, _, st = h.shoot(want_mag=False)
        n_bins = st["max_count"] + 2
        hist = torch.empty((n_bins,), dtype=torch.int64, device="cuda")
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        for _ in range(args.warmup):
            h.mpd(count, n_bins, hist=hist, sync=False)
        torch.cuda.synchronize()
        ms = []
        for _ in range(args.steps):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            h.mpd(count, n_bins, hist=hist, sync=False)
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        _, mst = h.mpd(count, n_bins, hist=hist)
        # row f5 on the same map: mlens_index_map (max reduction + MPD + compaction + 16-bit map; synchronous) and decode
        ims, dms = [], []
        for _ in range(args.steps):
            flush.fill_(1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            values, indexed = h.index_map(count)
            ims.append(1e3 * (time.perf_counter() - t0))
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            back = h.unindex_map(indexed, values.contiguous())
            e1.record()
            torch.cuda.synchronize()
            dms.append(e0.elapsed_time(e1))
        assert torch.equal(back, count)
        # minimal-bit-width storage: the indexed map at the width of its largest index, and back
        bits = int(mlens.lib().mlens_bits_needed(int(values.numel()) - 1))
        pms, ums = [], []
        for _ in range(args.steps):
            flush.fill_(1)
            e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            e0.record()
            packed = h.pack_map(indexed, bits)
            e1.record()
            unpacked = h.unpack_map(packed, bits, dtype=torch.uint16)
            e2.record()
            torch.cuda.synchronize()
            pms.append(e0.elapsed_time(e1)); ums.append(e1.elapsed_time(e2))
        assert torch.equal(unpacked, indexed)
    med = statistics.median(ms)
    nbytes = 4 * cfg.npix**2
    peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("hbm_gbs") if os.path.exists(
        os.path.join(ROOT, "MEASURED_PEAKS.json")) else None
    gbs = nbytes / (med * 1e-3) / 1e9
    print(json.dumps({"mode": "mpd", "config": args.config, "npix": cfg.npix, "n_bins": n_bins, "ms": ms, "ms_median": med,
                      "algorithmic_bytes": nbytes, "achieved_gbs": gbs, "peak_gbs": peak, "frac": gbs / peak if peak else None,
                      "note": "includes the memset of the bins and of the stats struct (stream-ordered, same events)",
                      "map_stats": mst,
                      "index_map": {"n_distinct": int(values.numel()), "ms_median_host_clock": statistics.median(ims),
                                    "unindex_ms_median": statistics.median(dms),
                                    "algorithmic_bytes": 10 * cfg.npix**2,  # MPD pass 4 B + apply 4 B in + 2 B out per pixel
                                    "unindex_gbs": 6 * cfg.npix**2 / (statistics.median(dms) * 1e-3) / 1e9},
                      "pack_indexed_map": {"bits": bits, "pack_ms_median": statistics.median(pms), "unpack_ms_median": statistics.median(ums),
                                           "algorithmic_bytes": (2 + bits / 8) * cfg.npix**2,
                                           "pack_gbs": (2 + bits / 8) * cfg.npix**2 / (statistics.median(pms) * 1e-3) / 1e9,
                                           "unpack_gbs": (2 + bits / 8) * cfg.npix**2 / (statistics.median(ums) * 1e-3) / 1e9}}),
          flush=True)


def run_survey_mode(args):
    """--survey: maps per second of the many-maps driver (paper_1406_0559_b200/survey.py, row f3) on ONE GPU: M independent
    maps of the config's class (seeds differ), with 1, 2 and 4 maps in flight.  Timed region per K: create (H2D lens
    list) + shoot + Eq. 4 + D2H of both maps into pinned host buffers + destroy, for all M maps; host clock around the
    batch with a device synchronize on both sides.  The lens fields are generated before the clock starts."""
    import dataclasses

    import torch

    from paper_1406_0559_b200 import survey

    torch.cuda.set_device(0)
    cfg0 = fields.CONFIGS[args.config]
    jobs = [survey.MapJob.from_config(dataclasses.replace(cfg0, seed=cfg0.seed + 17 * k)) for k in range(args.maps)]
    out_c = [torch.empty((cfg0.npix, cfg0.npix), dtype=torch.int32, pin_memory=True) for _ in jobs]
    out_m = [torch.empty((cfg0.npix, cfg0.npix), dtype=torch.float32, pin_memory=True) for _ in jobs]
    inter = None
    rows = []
    for k in [int(v) for v in args.streams.split(",")]:
        best = None
        for rep in range(max(1, args.warmup) + max(1, args.steps)):  # first repetitions are warm-up
            r = survey.run_survey(jobs, n_streams=k, out_count=out_c, out_mag=out_m)
            for j, st, c in zip(jobs, r["stats"], out_c):
                assert st["rays_in_map"] + st["rays_outside"] + st["rays_lost"] == st["rays_total"]
                assert int(c.sum(dtype=torch.int64)) == st["rays_in_map"]
            inter = sum(st["rays_total"] * max(1, len(j.lens_m)) for j, st in zip(jobs, r["stats"]))
            if rep >= max(1, args.warmup) and (best is None or r["seconds"] < best):
                best = r["seconds"]
        rows.append({"streams": k, "seconds": best, "maps_per_s": len(jobs) / best, "interactions_per_s": inter / best})
    print(json.dumps({"mode": "survey", "config": args.config, "workload": f"{len(jobs)} maps of config {args.config}'s class "
                      f"({cfg0.npix}^2 px, seeds {cfg0.seed}+17k), one GPU, create + shoot + D2H (count and mag) + destroy per map",
                      "maps": len(jobs), "d2h_bytes_per_map": 8 * cfg0.npix**2, "rows": rows}), flush=True)


def run_convolve(args):
    """--convolve: K launches of mlens_convolve (row f2, Eq. 6) on a map of the config's size (synthetic magnification
    values: the convolution's cost does not depend on them); HBM roofline on the minimum traffic of the method."""
    import torch

    from paper_1406_0559_b200 import mlens

    torch.cuda.set_device(0)
    cfg = fields.CONFIGS[args.config]
    n = cfg.npix
    with mlens.Mlens.from_config(cfg, np.zeros((1, 2), np.float32), None) as h:
        mag = torch.rand((n, n), dtype=torch.float32, device="cuda") * 4 + 0.5
        ker = h.profile_kernel(1, max(1.0, n / 400.0))
        out = torch.empty_like(mag)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        for _ in range(args.warmup):
            h.convolve(mag, ker, out=out)
        torch.cuda.synchronize()
        ms = []
        for _ in range(args.steps):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            h.convolve(mag, ker, out=out)
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        flux = float(out.sum(dtype=torch.float64) / mag.sum(dtype=torch.float64))
        # the survey case: one profile, many maps — the kernel's spectrum is prepared once (two FFTs per map)
        h.convolve_prepare(ker)
        ms_prep = []
        for _ in range(args.steps):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            h.convolve(mag, None, out=out)
            e1.record()
            torch.cuda.synchronize()
            ms_prep.append(e0.elapsed_time(e1))
    med = statistics.median(ms)
    nc = n * (n // 2 + 1)
    # minimum HBM traffic of the method as built (each array touched once per stage): 2 R2C (read 4 B/pixel, write 8 B per
    # complex) + product (read 2 x 8, write 8 per complex) + C2R (read 8 per complex, write 4 B/pixel)
    nbytes = 2 * (4 * n * n + 8 * nc) + 24 * nc + (8 * nc + 4 * n * n)
    peak_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    peak = json.load(open(peak_path)).get("hbm_gbs") if os.path.exists(peak_path) else None
    gbs = nbytes / (med * 1e-3) / 1e9
    print(json.dumps({"mode": "convolve", "config": args.config, "npix": n, "ms": ms, "ms_median": med,
                      "min_stage_bytes": nbytes, "achieved_gbs": gbs, "peak_gbs": peak, "frac": gbs / peak if peak else None,
                      "flux_ratio": flux, "ms_median_prepared_kernel": statistics.median(ms_prep), "paper_context": "~3 s per 10000^2 map with cuFFT on the paper's GPU (PAPER.md:152)"}),
          flush=True)


# -----------------------------------------------------------------------------------------------------------------
# N > 1: one process per GPU.  The driver starts the ranks itself (torch.distributed.run); called plainly as
# `python bench.py --gpus N`, bench.py re-executes itself under the same launcher so that N ranks really run.
# -----------------------------------------------------------------------------------------------------------------
def _free_port() -> int:
    import socket

    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        return sock.getsockname()[1]


def launch_ranks(args) -> int:
    """`--gpus N` (N > 1) without a launcher's environment: start N ranks of this very command line under
    `python -m torch.distributed.run` on 127.0.0.1 and a free port.  Never falls back to one rank: the GPU arms fail
    loudly when fewer than N devices are visible (the reference arm and --dry-run need no device)."""
    if args.impl == "ours" and not args.dry_run:
        import torch

        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but only {have} CUDA device(s) visible; refusing to run fewer ranks")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.abspath(__file__), *sys.argv[1:]]
    print(f"bench.py: starting {args.gpus} ranks: {' '.join(cmd)}", file=sys.stderr, flush=True)
    return subprocess.run(cmd).returncode


def run_dry(args):
    """--dry-run: the multi-rank plumbing without a GPU — every rank joins a gloo group on CPU, takes its row band of
    the config's lattice (sharded.row_bands, as --shard does) or its own map seed (weak mode), and the ranks all-reduce
    the number of lattice rows they own.  Rank 0 prints one JSON line.  No kernel runs and no throughput is reported."""
    import torch
    import torch.distributed as dist

    from paper_1406_0559_b200 import sharded

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29531")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = fields.CONFIGS[args.config]
    import math

    a1, a2 = cfg.half_widths  # DESIGN.md reading S2: n = 2 ceil(a/d - 1e-9) rays per axis
    n1, n2 = (2 * math.ceil(a / cfg.ray_spacing - 1e-9) for a in (a1, a2))
    band = sharded.row_bands(n2, world)[rank] if args.shard else (0, n2)
    rows = torch.tensor([band[1], 1], dtype=torch.int64)
    dist.all_reduce(rows, op=dist.ReduceOp.SUM)
    gathered = [None] * world
    dist.all_gather_object(gathered, {"rank": rank, "band": list(band), "seed": cfg.seed + (0 if args.shard else rank)})
    if rank == 0:
        print(json.dumps({"dry_run": True, "backend": "gloo", "n_gpus": world, "ranks_joined": int(rows[1]),
                          "scaling": "strong" if args.shard else "weak", "lattice": [n1, n2], "rows_total": int(rows[0]),
                          "ranks": gathered}), flush=True)
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=sorted(fields.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--shard", action="store_true", help="N > 1: shoot ONE map in row bands + one all-reduce (strong scaling)")
    ap.add_argument("--block", type=int, default=0, help="profile mode: shoot a centred SxS-ray block K times")
    ap.add_argument("--mpd", action="store_true", help="profile mode: time mlens_mpd on the config's shot map")
    ap.add_argument("--convolve", action="store_true", help="profile mode: time mlens_convolve on a map of the config's size")
    ap.add_argument("--ablations", action="store_true", help="block mode: load libmlens_ablations.so (kernel / loop variants)")
    ap.add_argument("--option", nargs=2, action="append", metavar=("KEY", "VALUE"), help="mlens_set_option (block mode)")
    ap.add_argument("--survey", action="store_true", help="profile mode: maps/s of the many-maps driver at 1, 2, 4 maps in flight")
    ap.add_argument("--maps", type=int, default=32, help="--survey: maps per batch")
    ap.add_argument("--streams", default="1,2,4", help="--survey: comma-separated numbers of maps in flight")
    ap.add_argument("--dry-run", action="store_true", help="N ranks on CPU over gloo: rank start-up, band plan, one all-reduce; no kernels")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is None and args.gpus > 1:
        raise SystemExit(launch_ranks(args))  # N ranks of this command line; rank 0 prints the line
    if world_env is not None and int(world_env) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={world_env} ranks")
    if args.dry_run:
        run_dry(args)
    elif args.survey:
        run_survey_mode(args)
    elif args.mpd:
        run_mpd(args)
    elif args.convolve:
        run_convolve(args)
    elif args.block:
        run_block(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
