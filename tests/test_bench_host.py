"""CPU tier for bench.py's host logic: the JSON contract of the reference arm, the paper's
timing protocol, and the N>1 aggregation (max over ranks, summed units, one shard per rank) on
a world_size-2 gloo group."""
import json
import os
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_trimmed_mean_follows_the_papers_protocol():
    # discard warm-up, remove the slowest 5 %, average the rest
    xs = [100.0] * 10 + [1.0] * 38 + [50.0, 60.0]
    assert bench.trimmed_mean(xs, drop_first=10) == 1.0          # 40 left, slowest 2 (50, 60) dropped
    assert bench.trimmed_mean([1.0] * 19 + [21.0]) == 1.0        # 20 values: the slowest one dropped
    assert bench.trimmed_mean([2.0, 4.0]) == 3.0                 # fewer than 20: nothing to drop


def test_roofline_inputs_come_from_committed_files():
    assert bench.committed_traffic("c2") == 6521582080
    assert bench.committed_traffic("nope") is None
    peak, src = bench.measured_peaks()
    assert 3000 < peak < 9000 and ("measured" in src or "fallback" in src)
    assert bench.BYTES_PER_ELEM == 14 + 26


def test_reference_arm_prints_one_valid_json_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                        "--warmup", "1", "--cpu-sample", "200000"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == bench.METRIC and d["unit"] == "GB/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"] > 0
    assert d["config"]["workload"].startswith("c3") and d["steps"] == 2      # the headline config (largest single-GPU)
    # the oracle runs the WHOLE step of that config: a1 (clip) + a3 => 42 algorithmic bytes per element
    assert d["cpu_baseline"]["bytes_per_element"] == 42 and d["cpu_baseline"]["sample_elements"] == 200000
    assert d["cpu_baseline"]["value"] == d["value"]


def test_plain_launch_with_gpus_2_starts_two_ranks_and_prints_one_line():
    """`python bench.py --gpus 2` launched PLAINLY (no torchrun) must start 2 ranks by itself and
    yield exactly one line with n_gpus = 2 (reference arm: rank 0 alone works, the other rank exits 0)."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--steps", "1",
                        "--warmup", "1", "--cpu-sample", "100000"], capture_output=True, text=True, timeout=900, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["impl"] == "reference"


def test_plain_launch_refuses_more_gpus_than_the_box_has():
    if torch.cuda.is_available() and torch.cuda.device_count() >= 64:
        pytest.skip("a box with 64 GPUs")
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "64"], capture_output=True, text=True,
                       timeout=300, env=env)
    assert r.returncode != 0 and "CUDA device" in (r.stderr + r.stdout)
    assert not [l for l in r.stdout.splitlines() if l.strip().startswith("{")]        # no line, no silent 1-GPU run


def test_step_bytes_per_element_counts_the_clip_pass():
    import argparse
    a = argparse.Namespace(precision="bf16", decay_groups=False)
    assert bench.step_bytes_per_elem(bench.workload_of(a, "c3")) == 42          # a1 (2) + a3 (40)
    assert bench.step_bytes_per_elem(bench.workload_of(a, "c2")) == 40
    assert bench.step_bytes_per_elem(bench.workload_of(a, "c3"), clip_pass=False) == 40
    assert bench.step_bytes_per_elem(bench.workload_of(a, "c2"), source="direct") == 28
    a32 = argparse.Namespace(precision="fp32", decay_groups=False)
    assert bench.step_bytes_per_elem(bench.workload_of(a32, "c3")) == 44        # fp32 gradients: 4-byte a1 read


def test_clock_log_cuts_samples_into_legs(tmp_path):
    f = tmp_path / "smi.csv"
    f.write_text("2026/11/04 10:00:00.000, 1965, 1965, 400.1, Not Active, Not Active, Not Active, Not Active\n"
                 "2026/11/04 10:00:00.050, 1700, 1965, 900.5, Not Active, Not Active, Not Active, Active\n"
                 "garbage line\n"
                 "2026/11/04 10:00:01.000, 1500, 1965, 950.0, Active, Not Active, Not Active, Not Active\n")
    rows = bench.ClockLog._parse(str(f))
    assert len(rows) == 3 and rows[1][1] == 1700.0 and rows[1][4] == [False, False, False, True]
    s = bench.ClockLog._summary(rows[:2])
    assert s["samples"] == 2 and s["reasons"] == ["sw_power_cap"] and s["sm_max_mhz"] == 1965.0 and s["sm_min_mhz"] == 1700.0
    assert bench.ClockLog._summary([])["samples"] == 0


def test_reference_arm_under_two_ranks_only_rank0_prints():
    outs = []
    for rank in (0, 1):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank))
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--steps", "1", "--warmup", "1", "--cpu-sample", "100000"],
                           capture_output=True, text=True, timeout=600, env=env)
        assert r.returncode == 0, r.stderr
        outs.append([l for l in r.stdout.splitlines() if l.strip()])
    assert len(outs[0]) == 1 and outs[1] == []


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    bench.dist_init(world, use_cuda=False)          # gloo on CPU
    dev = torch.device("cpu")
    t = bench.max_over_ranks(10.0 + rank, world, dev)      # the slowest rank defines the time
    u = bench.sum_over_ranks(1000.0 * (rank + 1), world, dev)
    bench.barrier(world)
    # one DP shard per rank: same layout, its own dp_rank, disjoint ranges (weak scaling, no exchange)
    import dataclasses
    from oracle import oracle as O
    from paper_2607_01646_b200 import workloads as W
    base = W.tiny_workload([1000, 333, 64], dp_size=2)
    wl = dataclasses.replace(base, dp_rank=bench.rank_env()[0] % base.dp_size)
    d = O.define_shard(wl.layout(), wl.dp_size, wl.dp_rank)
    q.put((rank, t, u, d["shard_begin"], d["n"]))
    dist.destroy_process_group()


def test_world_size_two_aggregation_on_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29600 + os.getpid() % 200
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [11.0, 11.0]      # max over ranks
    assert [r[2] for r in res] == [3000.0, 3000.0]  # units summed over ranks
    (b0, n0), (b1, n1) = (res[0][3], res[0][4]), (res[1][3], res[1][4])
    assert b0 == 0 and b1 >= n0 and n0 + n1 == 1397  # disjoint ranges that cover the tensors
