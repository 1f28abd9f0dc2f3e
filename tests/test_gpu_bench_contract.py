"""The bench.py output contract on a GPU box: one JSON line with the keys the driver reads, for our
arm (small step count) and for the reference arm."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(*args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                       timeout=900, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]
    return json.loads(lines[0])


def test_our_arm_json_line():
    d = run("--steps", "6", "--warmup", "3", "--check-every", "3", "--workload", "cfg2", "--extra-workloads", "cfg1",
            "--extra-steps", "4")
    assert d["metric"] == "su3_landau_or_site_updates_per_s" and d["unit"] == "site-updates/s"
    assert d["n_gpus"] == 1 and d["steps"] == 6 and d["warmup"] >= 3 and d["higher_is_better"] is True
    assert d["scaling"] == "weak" and d["vs_baseline"] is None and d["dtype"] == "f32" and d["data"] == "synthetic"
    assert d["value"] > 0 and d["ms_per_step"] > 0
    assert d["gpu_launches"] == 2 * 6 + 2 * 2          # half-sweeps + (partial, final) per check
    assert "workload" in d["config"] and "model" not in d["config"]
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["peak"] > 1000
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert r["bytes_per_launch"] == 2 * 4 * 16 ** 4 * 48
    e = d["e2e"]
    assert e["unit"] == d["unit"] and e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    assert e["value"] != d["value"]
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["unit"] == d["unit"] and c["sample"]
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert d["clocks"]["samples"] >= 3 and d["clocks"]["window_ms"] >= 50     # never a single NVML sample
    # the DRAM-side figures come from a committed ncu capture stamped with the kernel it was taken on
    assert r["kernel"].startswith("or_sweep_su3_staged_kernel<f32-12") and "traffic_capture" in r
    assert r["traffic"] is None and "stale" in r["traffic_capture"]           # no capture exists for cfg2
    # the other kernels of the path, the other workloads and the driver loop ride on the same line
    for k in ("theta_F", "pack", "unpack", "gauge_transform"):
        assert d["kernels"][k]["us"] > 0 and 0 < d["kernels"][k]["frac"] < 2
    for k in ("coulomb", "series_order_4", "microcanonical", "annealing_T_0.1", "annealing_T_2"):
        assert d["sweep_variants"][k]["half_sweep_us"] > 0 and d["sweep_variants"][k]["value"] > 0
    (x,) = d["extra_workloads"]
    assert x["workload"].startswith("cfg1") and x["value"] > 0 and x["launch_us"] > 0 and x["steps"] == 4
    assert x["roofline"]["frac"] == x["roofline"]["achieved"] / x["roofline"]["peak"] and "clocks" in x
    for name in ("cfg0", "cfg1", "cfg2"):
        loop = d["driver_loop"][name]
        a, b = loop["host_sync_every_check"], loop["device_stop_flag"]
        assert a["sweeps"] == b["sweeps"] and a["wall_ms"] > 0 and b["wall_ms"] > 0
        assert abs(b["theta"] - a["theta"]) <= 1e-9 * a["theta"] + 1e-29      # the same loop (sums grouped differently)
    assert d["value"] > 20 * c["value"]               # the GPU path, not a CPU fallback


def test_reference_arm_json_line():
    d = run("--impl", "reference", "--steps", "2", "--warmup", "1", "--workload", "cfg2")
    assert d["impl"] == "reference" and d["metric"] == "su3_landau_or_site_updates_per_s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_sharded_arm_json_line():
    """`bench.py --sharded` (time-slab decomposition, one slab per rank over NCCL) with one rank: the
    contract keys, strong scaling, and the same theta/F as the replica arm's field would give."""
    d = run("--sharded", "--steps", "6", "--warmup", "3", "--check-every", "3", "--workload", "cfg2")
    assert d["metric"] == "su3_landau_or_site_updates_per_s" and d["n_gpus"] == 1 and d["scaling"] == "strong"
    assert d["value"] > 0 and d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0
    assert "time-slab split: 1 slab(s) of 16 time-slices" in d["config"]["parallelism"]
    assert d["halo_bytes_per_step_per_rank"] == 4 * (16 ** 3 // 2) * 48
    assert d["roofline"]["frac"] == d["roofline"]["achieved"] / d["roofline"]["peak"]
    assert 0 < d["final"]["F"] < 1 and d["final"]["theta"] > 0
