"""The N > 1 path of bench.py on CPU: two gloo ranks ("replicas only").

The method has no exchange step, so the only multi-rank logic is (a) one independent seeded
configuration per rank, (b) MAX over ranks of the per-rank elapsed time, (c) whole-job value =
units of all ranks / that time, (d) the reference arm runs on rank 0 only.  All of it is host
logic and runs here without a GPU.
"""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402
import lattice_inputs as li  # noqa: E402


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        elapsed_s = 0.25 + 0.5 * rank                  # rank 1 is the slow one
        worst = bench.max_over_ranks(elapsed_s, world, "cpu")
        value = bench.whole_job_value(world, 4096, 10, worst)
        seed = bench.rank_seed(1003, rank)
        u = li.make_config((2, 2, 2, 2), 3, "haar", seed)
        out[rank] = (worst, value, seed, float(abs(u).sum()))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_max_time_and_whole_job_value():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert r0[0] == r1[0] == 0.75                        # MAX over ranks, seen by both
    assert r0[1] == r1[1] == 2 * 4096 * 10 / 0.75        # units of ALL ranks / slowest time
    assert r0[2] != r1[2] and r0[3] != r1[3]             # independent configurations


def test_single_rank_needs_no_process_group():
    assert bench.max_over_ranks(1.5, 1) == 1.5
    assert bench.whole_job_value(1, 100, 3, 0.5) == 600.0


def test_reference_arm_prints_on_rank0_only():
    """`bench.py --impl reference` (the oracle on the host cores): rank 0 prints the JSON line,
    every other rank exits 0 without work."""
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg0",
           "--steps", "2", "--warmup", "1", "--gpus", "2"]
    env = dict(os.environ, WORLD_SIZE="2", RANK="1", LOCAL_RANK="1")
    r1 = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    env = dict(os.environ, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0")
    r0 = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == bench.METRIC and line["unit"] == bench.UNIT
    assert line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["n_gpus"] == 2 and line["steps"] == 2


def test_committed_traffic_rows_are_stamped_and_stale_rows_are_refused():
    """roofline.traffic* comes from committed ncu captures (profiles/roofline_traffic.csv), which cannot
    be measured live: every row carries the commit and the kernel instantiation it was taken on, and
    bench.py uses a row only for the kernel it names."""
    rows = [l.strip().split(";") for l in open(os.path.join(ROOT, "profiles", "roofline_traffic.csv")) if l.strip()]
    assert rows[0] == ["workload", "capture", "dram_read_bytes", "dram_write_bytes", "commit", "kernel", "source"]
    for r in rows[1:]:
        assert len(r) == 7 and int(r[2]) > 0 and int(r[3]) > 0 and len(r[4]) >= 7
        assert os.path.exists(os.path.join(ROOT, r[6]))
    import paper_1412_3655_b200 as culgt
    kernel = culgt.culgt_sweep_kernel_name(culgt.Lattice((32, 32, 32, 32), 3, 32, 12))
    total, info = bench.committed_traffic("cfg3_fp32", "steady_state", kernel)
    assert total is not None and 3.0e8 < total < 4.1e8 and info["kernel"] == kernel and "stale" not in info
    # the steady-state DRAM traffic never exceeds the algorithmic bytes of a half-sweep (no re-reads)
    assert total <= 2 * 4 * 32 ** 4 * 48
    total, info = bench.committed_traffic("cfg3_fp32", "steady_state", "some_other_kernel<...>")
    assert total is None and "stale" in info
    total, info = bench.committed_traffic("cfg2", "steady_state", kernel)
    assert total is None and "stale" in info
