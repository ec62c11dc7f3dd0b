"""bench.py's reference arm (the oracle on host cores) runs without a GPU: check the JSON contract of its line, and that
ranks other than 0 stay silent.  (The GPU arm is exercised on the B200 box by the driver and by `bench.py` itself.)"""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(env_extra, extra_args=()):
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    env.update(env_extra)
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "1",
                           "--warmup", "0", *extra_args], capture_output=True, text=True, env=env, timeout=600)


def test_reference_arm_prints_one_contract_line():
    r = _run({"RANK": "0", "WORLD_SIZE": "1"})
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "ray_lens_interactions_per_s" and d["unit"] == "interactions/s"
    assert d["higher_is_better"] is True and d["vs_baseline"] is None and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["steps"] == 1 and d["warmup"] == 0 and d["gpu_launches"] == 0
    assert "workload" in d["config"] and "config 1" in d["config"]["workload"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_reference_arm_other_ranks_are_silent():
    r = _run({"RANK": "1", "WORLD_SIZE": "2"}, ["--gpus", "2"])
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_gpus_n_starts_n_ranks_itself():
    # `python bench.py --gpus 2` with no launcher environment: bench.py must start two ranks (torch.distributed.run on
    # 127.0.0.1), rank 0 prints the one line with n_gpus = 2, rank 1 reports in on stderr.  The reference arm needs no GPU.
    r = _run({}, ["--gpus", "2"])
    assert r.returncode == 0, r.stderr
    assert "starting 2 ranks" in r.stderr and "--nproc-per-node=2" in r.stderr
    assert "rank 1 of 2: idle" in r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["cores"] == len(os.sched_getaffinity(0))  # not the launcher's OMP_NUM_THREADS=1


def test_gpus_n_dry_run_of_the_sharded_launch_over_gloo():
    # the --shard plumbing without a GPU: two ranks join a gloo group, take their row bands, all-reduce once
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--shard", "--dry-run", "--config", "3"],
                       capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["dry_run"] is True and d["n_gpus"] == 2 and d["ranks_joined"] == 2 and d["scaling"] == "strong"
    assert d["lattice"] == [196608, 49152] and d["rows_total"] == 49152
    bands = [tuple(x["band"]) for x in sorted(d["ranks"], key=lambda x: x["rank"])]
    assert bands == [(0, 24576), (24576, 24576)]


def test_gpus_n_never_falls_back_to_fewer_ranks():
    # a launcher that started a different number of ranks than --gpus says: refuse
    r = _run({"RANK": "0", "WORLD_SIZE": "1"}, ["--gpus", "2"])
    assert r.returncode != 0 and "WORLD_SIZE=1" in r.stderr
    import torch

    if not torch.cuda.is_available():  # the GPU arm with no (or too few) devices: refuse, do not run one rank
        env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--config", "1"], capture_output=True,
                           text=True, env=env, timeout=300)
        assert r.returncode != 0 and "refusing to run fewer ranks" in r.stderr and r.stdout.strip() == ""


def test_gpu_arm_line_contract_from_measured_numbers():
    # bench.make_line is the pure function that assembles the GPU arm's JSON line; fed here with made-up measurements
    # for a 2-rank sharded run and a 1-rank run (the timing itself needs the B200 box)
    sys.path.insert(0, ROOT)
    import bench
    from paper_1406_0559_b200 import fields

    cfg = fields.CONFIGS[4]
    kw = dict(cfg_id=4, cfg=cfg, n_lens=2333, n1=122880, n2=122880, steps=3, warmup=3, ms_total=3 * 8000.0, kern_ms=7990.0,
              in_map=1_820_000_000, clocks={"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": []}, sms=148, e2e_s=16.2,
              e2e_steps=2, h2d_bytes=28000, d2h_bytes=8 << 20)
    one = bench.make_line(world=1, shard=False, peak_meas={"fp32_tflops": 71.8, "sm_mhz_observed": 1965.0, "how": "x"},
                          traffic=4_500_000, traffic_source="profiles/x.json", **kw)
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline"):
        assert key in one, key
    inter = 122880 * 122880 * 2333
    assert one["metric"] == "ray_lens_interactions_per_s" and one["scaling"] == "weak" and one["n_gpus"] == 1
    assert abs(one["value"] / (inter / 8.0) - 1) < 1e-12 and one["ms_per_step"] == 8000.0 and one["vs_baseline"] is None
    assert "workload" in one["config"] and "model" not in one["config"] and one["dtype"] == "f32"
    r = one["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-15
    assert abs(r["achieved"] - 11 * inter / 7.99 / 1e12) < 1e-9 and abs(r["peak"] - 148 * 128 * 2 * 1.965e9 / 1e12) < 1e-9
    assert r["peak_measured"] == 71.8 and abs(r["frac_of_measured"] - r["achieved"] / 71.8) < 1e-15
    assert r["traffic"] == 4_500_000 and r["traffic_source"] == "profiles/x.json"
    assert one["e2e"]["h2d_bytes_per_step"] == 28000 and one["e2e"]["d2h_bytes_per_step"] == 8 << 20
    two = bench.make_line(world=2, shard=True, **kw)
    assert two["scaling"] == "strong" and two["n_gpus"] == 2 and "row bands" in two["config"]["parallelism"]
    assert abs(two["value"] - one["value"]) < 1e-3  # ONE map on two GPUs: the job is the same map
    assert abs(two["roofline"]["achieved"] * 2 - one["roofline"]["achieved"]) < 1e-9  # each rank shoots half of it
    assert two["roofline"]["traffic"] is None and "peak_measured" not in two["roofline"]
