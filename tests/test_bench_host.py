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


def _canned_full_record():
    """A full phx-arm record shaped like run_headline's (all five configs, every sub-record, full-precision floats and
    the long prose strings the 39 KB line of round 2 carried)."""
    import math
    x = math.pi * 1000.0
    prose = "a long explanatory sentence that belongs in DESIGN.md and not in the line; " * 4
    recs = []
    for key in bench.ALL_CONFIGS:
        win = {"rule": prose, "gemms_per_iter": 4096, "compute_window_ms": x, "flush_ms": x / 7, "iter_ms_off": x,
               "exposed_ms_eager": x / 900, "exposed_pct_eager": x / 2500, "iter_ms_on_eager": x, "iters_per_arm": 30,
               "exposed_pct_graph_step": x / 4100, "exposed_ms_graph_step": x / 1300,
               "exposed_decomposition_ms": {"kernel_delta_isolated": x / 9000, "rest_eager": x / 7000}}
        r = {"config": key, "workload": prose[:80], "elements": 421150976, "state_bytes": 12 * 421150976, "clip": prose[:40],
             "step_ms": x / 1180, "step_bytes_per_element": 42, "step_gbs": x * 2.1, "step_frac_of_measured_peak": x / 3100,
             "kernel_ms": x / 1230, "kernel_gbs": x * 2.11, "kernel_frac_of_measured_peak": x / 3120,
             "e2e": {"ms_per_step": x / 30, "steps": 15, "h2d_bytes_per_step": 842301952, "d2h_bytes_per_step": 5053811968,
                     "link_gbs": x / 57, "metric_gbs": x / 18},
             "flush": {"ms": x / 34, "gbs": x / 57, "frac_of_d2h_peak": x / 3170, "chunk_mib": 32, "bytes": 5053811968},
             "overlap": {"headline_window": dict(win), "tight_window": dict(win)},
             "exposed_ckpt_ms_per_iter": x / 900, "exposed_pct": x / 2500,
             "restore": {"restore_ms": x / 34, "recompute_ms": x / 1180, "mode": "copy", "two_phase": {"note": prose}}}
        if key in ("c4a", "c4b"):
            r["hotswap"] = {"restore_ms": x / 70, "trajectory_bit_exact_vs_uninterrupted": True, "note": prose,
                            "two_phase": {"params_ready_ms": x / 200, "trajectory_bit_exact_vs_uninterrupted": True}}
        if key == "c5":
            r["chunk_depth_grid"] = [{"chunk_mib": c, "depth": d, "exposed_pct": x / 2000, "note": prose}
                                     for c in (4, 16, 64, 256) for d in (1, 2, 3, 4)]
        recs.append(r)
    legs = {f"{k}.{leg}": {"sm_mhz": 1965.0, "sm_min_mhz": 1500.0, "sm_max_mhz": 1965.0, "power_w_max": 989.2,
                           "reasons": ["sw_power_cap"], "samples": 609, "seconds": 1.334}
            for k in bench.ALL_CONFIGS for leg in ("step", "kernel", "e2e", "flush", "overlap.headline_window.eager",
                                                   "overlap.tight_window.graph_step", "restore")}
    return {
        "metric": bench.METRIC, "value": x * 2.1, "unit": bench.UNIT, "n_gpus": 1, "steps": 20, "warmup": 5,
        "ms_per_step": x / 1180, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": "c3: LLaMA-7B-style shard: 32L h4096 ffn11008 V32000, TP1 PP1 dp16 rank0, clip 1.0 — " + prose,
                   "configs_measured": bench.ALL_CONFIGS, "elements_per_shard": 421150976, "state_bytes": 12 * 421150976,
                   "staging_depth": 2, "chunk_mib": 32, "sync_mode": "strict", "snapshot_source": "staged",
                   "bytes_per_element": 42, "bytes_per_element_note": prose, "precision": prose, "decay_groups": False,
                   "l2": prose, "timed_region": prose, "host_payload": prose,
                   "parallelism": "dp1 independent shards, no data-path collective in the timed region"},
        "elements_per_s": x * 5e7, "exposed_ckpt_ms_per_iter": x / 900,
        "exposed_pct_worst_config": {"config": "c5", "exposed_pct": x / 2100, "exposed_ms": x / 800},
        "roofline": {"bound": "hbm", "achieved": x * 2.11, "peak": 6551.7, "unit": "GB/s", "frac": x * 2.11 / 6551.7,
                     "traffic": 16788000000, "peak_source": "MEASURED_PEAKS.json:hbm_gbs (measured)",
                     "frac_of_nominal_8TBps": x / 3800, "kernel": "phx::k_step8<true,0,false>", "kernel_ms": x / 1230,
                     "step_ms": x / 1180, "algorithmic_bytes_per_launch": 40 * 421150976, "bytes_per_element": 40,
                     "note": prose, "mix_ceiling_gbs": {"step_mix_3r6w": x * 2.13, "off_mix_3r3w": x * 2.2},
                     "frac_of_mix_ceiling": x / 3180},
        "host_link": {"bound": "host_link", "achieved": x / 57, "peak": x / 56, "unit": "GB/s", "frac": x / 3170,
                      "flush_ms": x / 34, "chunk_mib": 32, "h2d_peak_gbs": x / 56},
        "e2e": {"value": x / 18, "unit": bench.UNIT, "h2d_bytes_per_step": 842301952, "d2h_bytes_per_step": 5053811968,
                "ms_per_step": x / 30, "steps": 15, "link_gbs": x / 57, "note": prose},
        "configs": recs,
        "cpu_baseline": {"value": x / 90, "unit": bench.UNIT, "cores": 16, "kind": "oracle", "sample": prose,
                         "sample_elements": 1 << 26, "ms_per_step": x / 40, "a1_ms": x / 52, "a1_threads": 1,
                         "a3_ms": x / 170, "a3_threads": 16, "elements_per_s": x * 3e5, "bytes_per_element": 42},
        "gpu_launches": 60,
        "clocks": {"sm_mhz": 1965.0, "sm_min_mhz": 1965.0, "sm_max_mhz": 1965.0, "power_w_max": 989.2, "reasons": [],
                   "samples": 26, "seconds": 0.06, "sampler": "nvml, 2 ms period"},
        "clocks_all_legs": {"sm_mhz": 1545.0, "reasons": ["sw_power_cap"], "samples": 100000}, "clocks_legs": legs,
        "step_ms_min_max": [x / 1190, x / 1170],
    }


def test_phx_arm_line_is_compact_strict_json_with_every_contract_key():
    """ADVICE r2 (high) / VERDICT r2 item 1: the round-2 line was 39 KB and the driver parsed nothing.  The line the
    phx arm prints is built by compact_line from the full record and must stay under MAX_LINE_BYTES whatever the full
    record holds; the full record goes to a side file the line names."""
    full = _canned_full_record()
    assert len(json.dumps(full)) > 20000                      # the canned record is as bulky as the real one
    text = bench.compact_line(full, "gpurun_out/bench_full.json")
    assert "\n" not in text and len(text.encode()) <= bench.MAX_LINE_BYTES <= 3000, len(text)
    d = json.loads(text, parse_constant=lambda c: pytest.fail(f"non-strict JSON constant {c}"))
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert k in d, k
    assert d["value"] > 0 and d["config"]["workload"].startswith("c3:") and "model" not in d["config"]
    assert set(d["roofline"]) >= {"bound", "achieved", "peak", "unit", "frac", "traffic", "kernel", "kernel_ms"}
    assert abs(d["roofline"]["frac"] - d["roofline"]["achieved"] / d["roofline"]["peak"]) < 1e-3
    assert set(d["cpu_baseline"]) >= {"value", "unit", "cores", "kind", "sample", "a1_ms", "a3_ms"}
    assert set(d["e2e"]) >= {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"} and d["e2e"]["h2d_bytes_per_step"] > 0
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons", "samples"}
    assert list(d["configs"]) == bench.ALL_CONFIGS and all(len(v) == len(d["configs_cols"]) for v in d["configs"].values())
    assert d["configs"]["c4a"][-1] is True and d["configs"]["c2"][-1] is None
    assert d["full_record"] == "gpurun_out/bench_full.json"
    # a record even bulkier than any real one still yields a line under the limit (optional parts are shed)
    full["config"]["workload"] = "c3: " + "x" * 5000
    full["roofline"]["kernel"] = "k" * 2000
    assert len(bench.compact_line(full)) <= bench.MAX_LINE_BYTES


def test_phx_arm_prints_exactly_one_line():
    import inspect
    src = inspect.getsource(bench.run_headline)
    assert src.count("print(") == 1 and "print(compact_line(" in src


def test_cpu_baseline_reports_a1_and_a3_separately():
    import argparse
    wl = bench.workload_of(argparse.Namespace(precision="bf16", decay_groups=False), "c3")
    cb = bench.cpu_baseline(wl, 100000, 2, 1)
    assert cb["a1_ms"] > 0 and cb["a3_ms"] > 0 and abs(cb["a1_ms"] + cb["a3_ms"] - cb["ms_per_step"]) < 1e-6
    assert cb["a1_threads"] == 1 and cb["a3_threads"] == cb["cores"]
