#!/usr/bin/env python
"""bench.py — measures the phx hot path on B200 and prints ONE JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--configs c2,c3,c4a,c4b,c5] [--impl phx|reference]

`--gpus N` with N > 1 starts N ranks BY ITSELF (re-exec through torch.distributed.run on 127.0.0.1) when it
was not launched under torchrun already; it fails loudly when the box has fewer than N GPUs.

The one line covers EVERY bandwidth-sized config of BASELINE.json (c2, c3, c4a, c4b, c5) in one process:
  value      fused AdamW+snapshot HBM GB/s of the HEADLINE config — c3, the largest single-GPU configuration —
             K back-to-back passes of the whole device-side hot path (a1 clip pass where the config has one, a2
             sync-point wait, a3 ONE fused kernel writing live state + bf16 copy + packed snapshot) with the
             gradients resident in HBM; the step's TRUE algorithmic bytes (42 B/element with the a1 pass, 40
             without) / device time (CUDA events on the launching stream).  Working set >> L2.
  roofline   the dominant kernel (the fused step) alone, 40 B/element, against the measured HBM peak.
  configs    per config: step / kernel / snapshot-off ms and GB/s, flush GB/s against the pinned-copy peak measured
             in the same run, exposed checkpoint ms/iteration at T_c >= 4 T_D2H and at the tight 1.25 T_D2H window,
             with eagerly launched iterations and with the whole iteration captured in a CUDA graph (the
             graph-capturable form of the step), e2e through host buffers, restore + recompute (one phase, and the
             two-phase restore beside the recomputed iteration), the c4 hot-swap scenario (bit-exact trajectory
             flag), the c5 chunk x depth grid, the c3 producer-side clip.
  e2e        the headline config through the same C-ABI calls with HOST buffers (H2D grads, D2H snapshot + commit).
  cpu_baseline  the oracle as it stands on the box's host cores, on the SAME bounded sample `--impl reference` times.
  clocks     NVML (what nvidia-smi prints from) sampled over the whole run every 2 ms, reported per timed leg.
`--impl reference` times the oracle instead (the reference arm of this tier).
"""
from __future__ import annotations

import argparse
import contextlib
import datetime
import json
import math
import os
import socket
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fused_adamw_snapshot_hbm_gbs"
UNIT = "GB/s"
BYTES_PER_ELEM = 40          # a3: 14 read + 26 written
BYTES_PER_ELEM_OFF = 28      # a3 with snapshots off / direct source
BYTES_A1 = 2                 # a1: one read of the bf16 gradients (4 in the all-FP32 precision)
NOMINAL_HBM_GBS = 8000.0     # north_star "~8 TB/s"
FALLBACK_HBM_GBS = 6650.0    # /opt/skills/guides/B200_PROFILING.md, only if MEASURED_PEAKS.json is absent
ALL_CONFIGS = ["c2", "c3", "c4a", "c4b", "c5"]
HEADLINE = "c3"              # the largest single-GPU configuration of BASELINE.json:configs
ORACLE_SAMPLE = 1 << 26      # elements of the shard the oracle is timed on (both arms): ~10-30 s of CPU work


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="phx", choices=["phx", "reference"])
    ap.add_argument("--configs", default="", help="comma list of workload keys (default: c2,c3,c4a,c4b,c5 at one GPU, "
                                                  "the headline config at N > 1)")
    ap.add_argument("--config", default="", help="shorthand for --configs X --headline X")
    ap.add_argument("--headline", default=HEADLINE, help="config `value` / `roofline` / `e2e` are quoted on")
    ap.add_argument("--depth", type=int, default=2)
    ap.add_argument("--chunk-mib", type=int, default=32)
    ap.add_argument("--sync", default="strict", choices=["strict", "relaxed"])
    ap.add_argument("--gemms", type=int, default=0, help="GEMMs per overlapped iteration (0 = auto: T_c >= 4 T_D2H)")
    ap.add_argument("--overlap-secs", type=float, default=4.5, help="time budget per overlap arm (sets the iteration count)")
    ap.add_argument("--overlap-iters", type=int, default=0, help="iterations per overlap arm (0 = from --overlap-secs, 8..30)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="0 = auto (>= 1.5 s)")
    ap.add_argument("--no-overlap", action="store_true")
    ap.add_argument("--no-graph-step", action="store_true", help="skip the CUDA-graph-captured iteration arms")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-mix-ceiling", action="store_true", help="skip the no-arithmetic HBM mix-ceiling probe")
    ap.add_argument("--no-grid", action="store_true", help="skip the c5 chunk x depth grid")
    ap.add_argument("--no-direct", action="store_true", help="skip the PHX_SNAPSHOT_DIRECT repeat on the headline config")
    ap.add_argument("--cpu-sample", type=int, default=0, help="elements the oracle is timed on (0 = %d)" % ORACLE_SAMPLE)
    ap.add_argument("--mode", default="headline", choices=["headline", "overlap-curve", "sweep", "timeline", "probe"],
                    help="headline: the ONE contract line (default).  The others print one JSON line per measurement: "
                         "overlap-curve = exposed ms vs G; sweep = the full chunk x depth x sync-mode grid "
                         "(BASELINE.json:configs[4]); timeline = copy/compute overlap from CUDA events")
    ap.add_argument("--source", default="staged", choices=["staged", "direct"],
                    help="snapshot source: staged = fused kernel also writes the staging slot (40 B/elem, north_star); "
                         "direct = flush DMAs the live planes under the strict sync point (28 B/elem)")
    ap.add_argument("--restore-mode", default="copy", choices=["bulk", "copy"])
    ap.add_argument("--peers", type=int, default=-1,
                    help="k ring peers (SURVEY 8(f1)); -1 = auto: k = 1 and 2 over the real CUDA-IPC ring when --gpus > 1, "
                         "none at one GPU; k > 0 at one GPU measures a loopback stand-in (same device)")
    ap.add_argument("--publish", default="auto", choices=["auto", "none", "fused", "copy", "both"],
                    help="SURVEY 8(f3) model-parameter publication: auto = both at N > 1, none at one GPU")
    ap.add_argument("--precision", default="bf16", choices=["bf16", "fp32"])
    ap.add_argument("--decay-groups", action="store_true")
    ap.add_argument("--payload", default="optimizer", choices=["optimizer", "full"])
    ap.add_argument("--clip-scope", default="auto", choices=["auto", "local", "global"],
                    help="configs with a clip (c3): local = the shard's own norm; global = SURVEY 8(e) all-gather of one "
                         "double per rank; auto = local at one GPU, both at N > 1")
    ap.add_argument("--chunks", default="4,8,16,32,64,128,256", help="chunk sizes (MiB) of --mode sweep")
    ap.add_argument("--depths", default="1,2,3,4", help="staging depths of --mode sweep")
    ap.add_argument("--syncs", default="strict,relaxed", help="sync modes of --mode sweep")
    ap.add_argument("--debug-shared-gpu", action="store_true",
                    help="N > 1 ranks all on cuda:0 with a gloo control plane — a functional check of the N-rank code "
                         "path on a one-GPU box; the numbers it prints are NOT multi-GPU numbers and say so")
    a = ap.parse_args(argv)
    if a.config:
        a.configs, a.headline = a.config, a.config
    return a


# ----------------------------------------------------------------------------------------------
# helpers
# ----------------------------------------------------------------------------------------------


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return float(d["hbm_gbs"]), "MEASURED_PEAKS.json:hbm_gbs (measured)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "B200_PROFILING.md fallback"


def committed_traffic(config):
    """dram bytes/launch of the fused kernel from the committed ncu --set full capture, or None."""
    path = os.path.join(ROOT, "profiles", "traffic.txt")
    try:
        for line in open(path):
            w = line.split()
            if w and w[0] == config:
                return int(w[1])
    except Exception:
        pass
    return None


# the sampler process: NVML (the library nvidia-smi prints from) polled every ~2 ms, one CSV row per sample in the
# same columns as the nvidia-smi query below, so that even a K = 20 step leg (tens of ms) gets >= 10 samples
_NVML_SAMPLER = r"""
import sys, time
import pynvml as N
N.nvmlInit()
uuid, index, period = sys.argv[1], int(sys.argv[2]), float(sys.argv[3])
h = None
if uuid:
    for u in (uuid, uuid.encode()):
        try:
            h = N.nvmlDeviceGetHandleByUUID(u); break
        except Exception:
            pass
if h is None:
    h = N.nvmlDeviceGetHandleByIndex(index)
reasons = getattr(N, "nvmlDeviceGetCurrentClocksEventReasons", None) or N.nvmlDeviceGetCurrentClocksThrottleReasons
mx = N.nvmlDeviceGetMaxClockInfo(h, N.NVML_CLOCK_SM)
out = sys.stdout
while True:
    t = time.time()
    r = reasons(h)
    out.write("%.6f,%d,%d,%.2f,%d,%d,%d,%d\n" % (t, N.nvmlDeviceGetClockInfo(h, N.NVML_CLOCK_SM), mx,
              N.nvmlDeviceGetPowerUsage(h) / 1000.0, bool(r & 0x8), bool(r & 0x40), bool(r & 0x20), bool(r & 0x4)))
    out.flush()
    time.sleep(period)
"""


class ClockLog:
    """SM clocks / throttle reasons sampled over the WHOLE run with timestamps by ONE side process, cut into the
    timed legs afterwards — every leg gets its own record (B200_PROFILING.md clocks line).  The sampler polls NVML
    (what nvidia-smi itself reads) every ~2 ms; if pynvml is missing it falls back to `nvidia-smi -lms 50`."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index=0, period_ms=2, uuid=""):
        self.legs = []
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        self.source = None
        try:
            import pynvml  # noqa: F401  (only to learn whether the sampler can run)
            self.p = subprocess.Popen([sys.executable, "-c", _NVML_SAMPLER, uuid, str(index), str(period_ms / 1e3)],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
            time.sleep(0.3)
            if self.p.poll() is not None:
                self.p = None
            else:
                self.source = f"nvml, {period_ms} ms period"
        except Exception:
            self.p = None
        if self.p is None:
            try:
                self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                           "--format=csv,noheader,nounits", "-lms", "50"],
                                          stdout=self.f, stderr=subprocess.DEVNULL)
                self.source = "nvidia-smi -lms 50"
            except Exception:
                self.p = None

    @contextlib.contextmanager
    def leg(self, name):
        t0 = time.time()
        try:
            yield
        finally:
            self.legs.append((name, t0, time.time()))

    @staticmethod
    def _parse(path):
        rows = []
        for r in open(path):
            w = [x.strip() for x in r.strip().split(",")]
            if len(w) < 8:
                continue
            try:
                ts = float(w[0]) if "/" not in w[0] else datetime.datetime.strptime(w[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                rows.append((ts, float(w[1]), float(w[2]), float(w[3]),
                             [x == "1" or x.lower().startswith("active") for x in w[4:8]]))
            except Exception:
                continue
        return rows

    @classmethod
    def _summary(cls, rows):
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        reasons = sorted({cls.NAMES[k] for r in rows for k in range(4) if r[4][k]})
        return {"sm_mhz": statistics.median(r[1] for r in rows), "sm_min_mhz": min(r[1] for r in rows),
                "sm_max_mhz": max(r[2] for r in rows), "power_w_max": max(r[3] for r in rows),
                "reasons": reasons, "samples": len(rows)}

    def stop(self):
        """-> (summary over all legs, {leg name: summary})"""
        if self.p is None:
            return self._summary([]), {}
        time.sleep(0.12)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = self._parse(self.f.name)
        os.unlink(self.f.name)
        per = {}
        for name, t0, t1 in self.legs:
            per[name] = self._summary([r for r in rows if t0 <= r[0] <= t1])
            per[name]["seconds"] = round(t1 - t0, 3)
        inside = [r for r in rows if any(t0 <= r[0] <= t1 for _, t0, t1 in self.legs)]
        return self._summary(inside), per


def trimmed_mean(xs, drop_first=0, drop_slowest_frac=0.05):
    """The paper's protocol: discard warm-up iterations, remove the slowest 5 %, average."""
    xs = list(xs)[drop_first:]
    k = int(len(xs) * drop_slowest_frac)
    xs = sorted(xs)[:len(xs) - k] if k else xs
    return sum(xs) / len(xs)


def rank_env():
    return (int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)),
            int(os.environ.get("LOCAL_RANK", 0)))


def dist_init(world, use_cuda):
    import torch.distributed as dist
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group("nccl" if use_cuda else "gloo")
    return dist


def _reduce(x: float, world, device, op):
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    dev = device if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=op)
    return float(t.item())


def max_over_ranks(x: float, world, device) -> float:
    """The slowest rank defines the step time (max over ranks)."""
    if world == 1:
        return x
    import torch.distributed as dist
    return _reduce(x, world, device, dist.ReduceOp.MAX)


def sum_over_ranks(x: float, world, device) -> float:
    if world == 1:
        return x
    import torch.distributed as dist
    return _reduce(x, world, device, dist.ReduceOp.SUM)


def barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def self_spawn(args):
    """`python bench.py --gpus N` launched plainly: start N ranks (one per GPU) through torch.distributed.run."""
    if args.impl == "phx" and not args.debug_shared_gpu:
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            raise SystemExit(f"bench.py --gpus {args.gpus}: this box has {have} CUDA device(s); refusing to time fewer "
                             f"ranks than asked for (there is no CPU fallback)")
    env = dict(os.environ)
    if args.impl == "phx":
        # leave NCCL's own init lines visible, on stderr so that stdout stays ONE JSON line
        env.setdefault("NCCL_DEBUG", "INFO")
        env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        env.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


# ----------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the oracle on the host cores — ONE sample definition for both
# ----------------------------------------------------------------------------------------------


def workload_of(args, key):
    """BASELINE.json config `key`, in the precision / decay-group variant the flags ask for."""
    import dataclasses
    from paper_2607_01646_b200 import workloads as W
    return dataclasses.replace(W.CONFIGS[key], precision=args.precision, decay_groups=bool(args.decay_groups))


def shard_elements(args, key):
    """n_padded of a config's shard from the library's own a0 (host-only call, no GPU work)."""
    from paper_2607_01646_b200 import binding as B
    wl = workload_of(args, key)
    h = B.phx_shard_create(wl.layout(), wl.dp_size, wl.dp_rank, tp=(wl.tp_size, wl.tp_rank), pp=(wl.pp_size, wl.pp_rank),
                           flags=wl.flags())
    n = int(B.phx_shard_info(h).n_padded)
    B.phx_shard_destroy(h)
    return n


def step_bytes_per_elem(wl, source="staged", clip_pass=True):
    """Algorithmic bytes per element of one pass of the device-side hot path."""
    fp32 = wl.precision == "fp32"
    b = BYTES_PER_ELEM_OFF if source == "direct" else BYTES_PER_ELEM
    if clip_pass and wl.hyper.max_grad_norm > 0:
        b += 4 if fp32 else BYTES_A1
    return b


def time_oracle(wl, sample, steps, warmup, nthreads):
    """Oracle hot path (phx_oracle.c as it stands: a1 sum of squares + clip where the config has one, a3 AdamW
    step) on the first `sample` elements of the shard.  Inputs generated on the CPU from the workload's seed."""
    import numpy as np
    import torch
    from oracle import oracle as O
    from paper_2607_01646_b200 import workloads as W
    fp32 = wl.precision == "fp32"
    d = O.define_shard(wl.layout(), wl.dp_size, wl.dp_rank, (wl.tp_size, wl.tp_rank), (wl.pp_size, wl.pp_rank), wl.flags())
    n = min(sample, d["n_padded"])
    segs = []
    for tid, _, off, ln in d["segments"]:
        if off < n:
            segs.append((tid, off, min(ln, n - off)))
    p = W.init_params(n, n, wl.seed).numpy()
    m = np.zeros(n, np.float32)
    v = np.zeros(n, np.float32)
    p16 = np.zeros(n, np.uint16)
    if fp32:
        g = W.gen_grads(wl, segs, n, 1, wl.seed, dtype=torch.float32).numpy()
    else:
        g = W.gen_grads(wl, segs, n, 1, wl.seed).view(torch.int16).numpy().view(np.uint16)
    mask = None
    if any(wl.flags()):
        mask = np.zeros(n, np.uint8)
        fl = wl.flags()
        for tid, off, ln in segs:
            if fl[tid] & 1:
                mask[off:off + ln] = 1
    h = wl.hyper
    times, a1_times = [], []
    for t in range(1, warmup + steps + 1):
        coef = 1.0
        t0 = time.perf_counter()
        if h.max_grad_norm > 0:
            coef = float(O.clip_coef(O.sumsq(g), h.max_grad_norm))
        t1 = time.perf_counter()
        if fp32 or mask is not None:
            O.adamw_step_ex(p, m, v, g, None if fp32 else p16, mask, h.lr, h.beta1, h.beta2, h.eps, h.wd, t, coef, nthreads)
        else:
            O.adamw_step(p, m, v, g, p16, h.lr, h.beta1, h.beta2, h.eps, h.wd, t, coef, nthreads)
        dt = time.perf_counter() - t0
        if t > warmup:
            times.append(dt)
            a1_times.append(t1 - t0)
    return n, times, a1_times


def oracle_sample_desc(n, wl, steps, warmup):
    return (f"first {n} of {wl.n_expected} elements of the {wl.key} shard, {steps} steps after {warmup} warm-up; "
            f"a1 sum of squares (single thread) + a3 AdamW step (all cores)" if wl.hyper.max_grad_norm > 0 else
            f"first {n} of {wl.n_expected} elements of the {wl.key} shard, {steps} steps after {warmup} warm-up; a3 AdamW step")


def cpu_baseline(wl, sample, steps, warmup):
    """The record both arms print for the oracle on the host cores: same workload, same sample, same byte count."""
    cores = len(os.sched_getaffinity(0))
    n, times, a1_times = time_oracle(wl, sample, steps, warmup, cores)
    t = sum(times) / len(times)
    a1 = sum(a1_times) / len(a1_times)
    bpe = step_bytes_per_elem(wl)
    # a1_ms: the oracle's sum of squares as it stands (ONE thread, long double); a3_ms: its AdamW step on `cores`
    # threads.  `value` is their sum at the step's byte count; the two passes differ ~4x in elements/s.
    return {"value": bpe * n / t / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": oracle_sample_desc(n, wl, steps, warmup), "sample_elements": n, "ms_per_step": t * 1e3,
            "a1_ms": a1 * 1e3, "a1_threads": 1 if wl.hyper.max_grad_norm > 0 else 0, "a3_ms": (t - a1) * 1e3,
            "a3_threads": cores, "elements_per_s": n / t, "bytes_per_element": bpe}


def run_reference(args):
    rank, world, _ = rank_env()
    if rank != 0:
        return 0
    wl = workload_of(args, args.headline)
    cb = cpu_baseline(wl, args.cpu_sample or ORACLE_SAMPLE, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": cb["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{wl.key}: {wl.title}", "sample_elements": cb["sample_elements"],
                   "bytes_per_element": cb["bytes_per_element"],
                   "note": "oracle/phx_oracle.c as it stands on the host cores; the same bounded sample the phx arm's "
                           "cpu_baseline times"},
        "cpu_baseline": cb,
        "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------------------------
# the contract line: a compact headline record; the full record goes to a side file
# ----------------------------------------------------------------------------------------------

MAX_LINE_BYTES = 2900        # the driver keeps ~3 KB of stdout tail; a 39 KB line was not parsed (BENCH_r02: parsed null)
FULL_RECORD = os.path.join("gpurun_out", "bench_full.json")
CONFIG_COLS = ["step_gbs", "kernel_frac_of_peak", "flush_frac_of_d2h_peak", "exposed_pct_eager_4x", "exposed_pct_graph_4x",
               "exposed_pct_eager_1.25x", "exposed_pct_graph_1.25x", "restore_ms", "hotswap_bit_exact"]


def _r(x, sig=5):
    """Floats to `sig` significant digits, strings cut at 100 characters, everything else untouched."""
    if isinstance(x, str):
        return x[:100]
    if isinstance(x, bool) or not isinstance(x, float):
        return x
    if x != x or x in (float("inf"), float("-inf")):
        return None
    return float(f"{x:.{sig}g}")


def _pick(d, keys, sig=5):
    return {k: _r(d[k], sig) for k in keys if d is not None and k in d}


def compact_line(full, full_record=FULL_RECORD):
    """The ONE stdout line of the phx arm: every key of the bench contract plus a 9-number summary per config, at most
    MAX_LINE_BYTES bytes.  `full` is the complete record run_headline assembles (written to `full_record`)."""
    cfg = full["config"]
    line = {k: full[k] for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                                 "scaling", "vs_baseline", "dtype", "data", "gpu_launches") if k in full}
    line["value"], line["ms_per_step"] = _r(full["value"], 7), _r(full["ms_per_step"], 7)
    line["config"] = {"workload": cfg["workload"].split(" — ")[0][:100], "elements_per_shard": cfg["elements_per_shard"],
                      "staging_depth": cfg["staging_depth"], "chunk_mib": cfg["chunk_mib"], "sync_mode": cfg["sync_mode"],
                      "snapshot_source": cfg["snapshot_source"], "bytes_per_element": cfg["bytes_per_element"],
                      "l2": "inputs > L2", "parallelism": cfg["parallelism"].split(",")[0][:40]}
    rf = full["roofline"]
    line["roofline"] = _pick(rf, ("bound", "achieved", "peak", "unit", "frac", "traffic", "kernel", "kernel_ms", "step_ms",
                                  "algorithmic_bytes_per_launch", "frac_of_nominal_8TBps", "frac_of_mix_ceiling"))
    line["roofline"]["peak_source"] = "measured" if "measured" in rf.get("peak_source", "") else "fallback"
    if full.get("host_link"):
        line["host_link"] = _pick(full["host_link"], ("achieved", "peak", "frac"))
    if full.get("cpu_baseline"):
        cb = full["cpu_baseline"]
        line["cpu_baseline"] = _pick(cb, ("value", "unit", "cores", "kind", "sample_elements", "ms_per_step", "a1_ms", "a3_ms"))
        line["cpu_baseline"]["sample"] = "first %d elements of the %s shard; a1 one thread, a3 all cores" % (
            cb["sample_elements"], cfg["workload"].split(":")[0])
    else:
        line["cpu_baseline"] = None
    line["e2e"] = _pick(full["e2e"], ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step", "steps",
                                      "link_gbs"))
    line["exposed_ckpt_ms_per_iter"] = _r(full.get("exposed_ckpt_ms_per_iter"), 4)
    w = full.get("exposed_pct_worst_config")
    line["exposed_pct_worst_config"] = _pick(w, ("config", "exposed_pct"), 4) if w else None
    line["clocks"] = _pick(full.get("clocks") or {}, ("sm_mhz", "sm_max_mhz", "reasons", "samples"))
    rows = {}
    for r in full.get("configs", []):
        ov = r.get("overlap", {})
        hw, tw = ov.get("headline_window", {}), ov.get("tight_window", {})
        hs = r.get("hotswap")
        ok = None
        if hs is not None:
            ok = bool(hs.get("trajectory_bit_exact_vs_uninterrupted")) and all(
                bool(v.get("trajectory_bit_exact_vs_uninterrupted")) for v in hs.values() if isinstance(v, dict))
        rows[r["config"]] = [_r(v, 4) if isinstance(v, float) else v for v in (
            r.get("step_gbs"), r.get("kernel_frac_of_measured_peak"), r.get("flush", {}).get("frac_of_d2h_peak"),
            hw.get("exposed_pct_eager"), hw.get("exposed_pct_graph_step"), tw.get("exposed_pct_eager"),
            tw.get("exposed_pct_graph_step"), r.get("restore", {}).get("restore_ms"), ok)]
    line["configs_cols"] = CONFIG_COLS
    line["configs"] = rows
    line["full_record"] = full_record
    for k in ("process_group",):
        if k in full:
            line[k] = full[k]
    text = json.dumps(line, separators=(",", ":"))
    if len(text) > MAX_LINE_BYTES:           # never let an oversized line out again: shed the optional parts
        for k in ("configs_cols", "configs", "host_link", "exposed_pct_worst_config"):
            line.pop(k, None)
            text = json.dumps(line, separators=(",", ":"))
            if len(text) <= MAX_LINE_BYTES:
                break
    return text


def write_full_record(full, path=FULL_RECORD):
    """The complete record (every config's overlap / restore / hot-swap / grid sub-records, per-leg clocks)."""
    for target in (os.path.join(ROOT, path), os.path.join(tempfile.gettempdir(), os.path.basename(path))):
        try:
            os.makedirs(os.path.dirname(target), exist_ok=True)
            with open(target, "w") as f:
                json.dump(full, f, indent=1)
            return os.path.relpath(target, ROOT) if target.startswith(ROOT) else target
        except OSError:
            continue
    return None


# ----------------------------------------------------------------------------------------------
# phx arm
# ----------------------------------------------------------------------------------------------


class Rig:
    """One shard on one GPU plus everything the measurements need around it: gradients resident in HBM
    and in pinned host memory, a flush stream, the GEMM operands of the stand-in compute window."""

    def __init__(self, args, key, rank=0, world=1, local_rank=0, depth=None, chunk_mib=None, sync=None,
                 replica=None, host_grads=True, restore_mode=None, source=None, clip_scope="local"):
        import dataclasses
        import torch
        from paper_2607_01646_b200 import binding as B
        from paper_2607_01646_b200 import workloads as W
        from paper_2607_01646_b200.shard import Shard
        self.torch, self.B, self.W, self.Shard, self.args = torch, B, W, Shard, args
        self.device = torch.device(f"cuda:{local_rank}")
        base = workload_of(args, key)
        # weak scaling: every rank owns one DP shard of the same model (its own dp_rank); no data-path collective
        self.wl = dataclasses.replace(base, dp_rank=rank % base.dp_size)
        self.depth = depth or args.depth
        self.chunk_mib = chunk_mib or args.chunk_mib
        self.sync_name = sync or args.sync
        self.sync_mode = B.PHX_SYNC_STRICT if self.sync_name == "strict" else B.PHX_SYNC_RELAXED
        self.source_name = source or args.source
        self.source = B.PHX_SNAPSHOT_DIRECT if self.source_name == "direct" else B.PHX_SNAPSHOT_STAGED
        self.bytes_per_elem = BYTES_PER_ELEM_OFF if self.source_name == "direct" else BYTES_PER_ELEM
        if restore_mode is None:
            restore_mode = B.PHX_RESTORE_COPY_ENGINE if args.restore_mode == "copy" else B.PHX_RESTORE_BULK_KERNEL
        self.restore_mode_name = "copy_engine" if restore_mode == B.PHX_RESTORE_COPY_ENGINE else "bulk_kernel"
        self.full = getattr(args, "payload", "optimizer") == "full"
        self.s = Shard(self.wl, device=self.device, staging_depth=self.depth, sync_mode=self.sync_mode,
                       chunk_bytes=self.chunk_mib << 20, replica=replica, restore_mode=restore_mode,
                       snapshot_source=self.source,
                       payload=B.PHX_PAYLOAD_FULL_RANK_STATE if self.full else B.PHX_PAYLOAD_OPTIMIZER)
        self.N = self.s.n_padded
        self.s.p.copy_(W.init_params(self.s.n, self.N, self.wl.seed, device=self.device))
        self.s.set_state(0)
        self.fp32 = self.wl.precision == "fp32"
        self.grad_bytes = 4 if self.fp32 else 2
        gdt = torch.float32 if self.fp32 else torch.bfloat16
        self.grads = [W.gen_grads(self.wl, self.s.segments, self.N, t, self.wl.seed, device=self.device, dtype=gdt)
                      for t in (1, 2)]
        self.hgrads = [g.cpu().pin_memory() for g in self.grads] if host_grads else None
        torch.cuda.synchronize()
        self.cur = torch.cuda.current_stream(self.device)
        self.side = torch.cuda.Stream(device=self.device)
        self.step = 0
        self.s_off = None
        self.off_step = 0
        self._gemm = None
        self._fault_stream = None
        self.gemm_ms = None
        self.k_peers = 0
        self.peers_in_overlap = False
        self.gclip = None
        self.clip = self.wl.hyper.max_grad_norm > 0
        if clip_scope == "global" and self.clip:
            from paper_2607_01646_b200.clip import GlobalClip
            self.gclip = GlobalClip(self.s)     # default process group = the DP group of this bench

    # -- §8(f1): peer replication ----------------------------------------------------------------------
    def setup_peers(self, k, rank, world):
        """Bind k ring peers: a real CUDA-IPC ring over the `world` processes, or, on one GPU, received buffers
        on the same device (loopback stand-in).  Returns a description; raises on failure (all ranks agree)."""
        from paper_2607_01646_b200 import ring as PR
        self.peer_stream = self.torch.cuda.Stream(device=self.device)
        self.k_peers = k
        if world > 1:
            self.ring = PR.PeerRing(self.s, k, ring_size=world, ring_rank=rank)
            return "P2P into the ring successors' HBM, received buffers mapped over CUDA IPC"
        self.recv = PR.ReceivedBuffers(self.s.info.slot_stride, k)
        self.B.phx_shard_bind_peers(self.s.h, self.recv.ptrs)
        return "loopback stand-in: received buffers on the SAME GPU (device-to-device copy engine, not NVLink)"

    def time_peer_flush(self):
        """One replication of the newest snapshot to all k peers, alone, timed on the peer stream."""
        torch = self.torch
        self.do_step()
        torch.cuda.synchronize()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record(self.peer_stream)
        self.B.phx_snapshot_flush_peers_async(self.s.h, self.peer_stream)
        f1.record(self.peer_stream)
        self.B.phx_snapshot_wait_peers(self.s.h, self.step)
        torch.cuda.synchronize()
        return f0.elapsed_time(f1)

    def close_peers(self):
        if getattr(self, "ring", None) is not None:
            self.ring.close()
            self.ring = None
        if getattr(self, "recv", None) is not None:
            self.B.phx_shard_bind_peers(self.s.h, [])
            self.recv.free()
            self.recv = None
        self.k_peers = 0

    def precision_code(self):
        return self.B.PHX_PRECISION_FP32 if self.fp32 else self.B.PHX_PRECISION_BF16_GRADS

    def kernel_name(self):
        mode = (1 if self.fp32 else 0) | (2 if any(self.wl.flags()) else 0)
        return "phx::k_step8<%s,%d,false>" % ("true" if self.source_name == "staged" else "false", mode)

    # -- the hot path -------------------------------------------------------------------------------
    def do_step(self):
        self.step += 1
        if self.gclip is not None:
            self.gclip.step_and_snapshot(self.grads[self.step & 1], self.step, stream=self.cur)
        else:
            self.s.step_and_snapshot(self.grads[self.step & 1], self.step)

    def time_steps(self, K, Wm):
        """K back-to-back a1..a3 passes after Wm warm-ups; CUDA events on the launching stream."""
        torch, B = self.torch, self.B
        for _ in range(Wm):
            self.do_step()
        torch.cuda.synchronize()
        l0 = B.phx_kernel_launches(self.s.h)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
        ev[0].record(self.cur)
        h0 = time.perf_counter()
        kh = min(K, 48)          # host cost of the calls: a short burst, before the driver's launch queue can fill up
        for k in range(K):
            self.do_step()
            ev[k + 1].record(self.cur)
            if k + 1 == kh:
                self.host_enqueue_us = (time.perf_counter() - h0) * 1e6 / kh   # the calls only enqueue
        torch.cuda.synchronize()
        per = [ev[k].elapsed_time(ev[k + 1]) for k in range(K)]
        return ev[0].elapsed_time(ev[K]), per, B.phx_kernel_launches(self.s.h) - l0

    def _aux_handle(self, **kw):
        B, wl = self.B, self.wl
        h = B.phx_shard_create(wl.layout(), wl.dp_size, wl.dp_rank, tp=(wl.tp_size, wl.tp_rank),
                               pp=(wl.pp_size, wl.pp_rank), flags=wl.flags(), precision=self.precision_code(), **kw)
        return h

    def time_fused_kernel_alone(self, K):
        """The dominant kernel without the clip kernels: a second handle with clipping off bound to the same memory."""
        torch, B = self.torch, self.B
        h0 = self._aux_handle(staging_depth=self.depth, max_grad_norm=0.0, snapshot_source=self.source)
        B.phx_shard_bind(h0, self.s.p, self.s.m, self.s.v, self.s.p16, self.s.staging, self.s.replica)
        B.phx_shard_set_state(h0, 0, self.cur)
        hp = self.wl.hyper
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for k in range(3 + K):
            if k == 3:
                e0.record(self.cur)
            B.phx_step_and_snapshot(h0, self.grads[k & 1], hp.lr, hp.beta1, hp.beta2, hp.eps, hp.wd, k + 1, self.cur)
        e1.record(self.cur)
        torch.cuda.synchronize()
        B.phx_shard_destroy(h0)
        return e0.elapsed_time(e1) / K

    def time_producer_clip(self, K):
        """the gradients come out of the producer's epilogue (fp32 main gradients -> bf16 + sum of
        squares, one pass) and the step takes the sum: no a1 pass.  Returns (finalize ms, step ms)."""
        torch, B = self.torch, self.B
        g32 = self.W.gen_grads(self.wl, self.s.segments, self.N, 3, self.wl.seed, device=self.device, dtype=torch.float32)
        g16 = torch.empty(self.N, dtype=torch.bfloat16, device=self.device)
        S = torch.zeros(1, dtype=torch.float64, device=self.device)
        for _ in range(2):
            self.s.grads_finalize(g32, 1.0, g16, S)
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        nf = max(5, K // 2)
        f0.record(self.cur)
        for _ in range(nf):
            self.s.grads_finalize(g32, 1.0, g16, S)
        f1.record(self.cur)
        for _ in range(3):
            self.step += 1
            B.phx_set_clip_partials(self.s.h, S, 1)
            self.s.step_and_snapshot(g16, self.step)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = B.phx_kernel_launches(self.s.h)
        e0.record(self.cur)
        for _ in range(K):
            self.step += 1
            B.phx_set_clip_partials(self.s.h, S, 1)
            self.s.step_and_snapshot(g16, self.step)
        e1.record(self.cur)
        torch.cuda.synchronize()
        launches = B.phx_kernel_launches(self.s.h) - l0
        del g32, g16
        return f0.elapsed_time(f1) / nf, e0.elapsed_time(e1) / K, launches / K

    def off_shard(self):
        """Snapshot-disabled handle (the paper's 'mechanism disabled' baseline) bound to the same live arrays."""
        if self.s_off is None:
            B = self.B
            h = self._aux_handle(snapshot_disabled=True, max_grad_norm=self.wl.hyper.max_grad_norm)
            B.phx_shard_bind(h, self.s.p, self.s.m, self.s.v, self.s.p16, None, None)
            B.phx_shard_set_state(h, 0, self.cur)
            self.s_off = h
        return self.s_off

    def do_step_off(self):
        hp = self.wl.hyper
        self.off_step += 1
        self.B.phx_step_and_snapshot(self.off_shard(), self.grads[self.off_step & 1], hp.lr, hp.beta1, hp.beta2,
                                     hp.eps, hp.wd, self.off_step, self.cur)

    def time_steps_off(self, K, Wm=3):
        torch = self.torch
        for _ in range(Wm):
            self.do_step_off()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(self.cur)
        for _ in range(K):
            self.do_step_off()
        e1.record(self.cur)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / K

    def flush(self):
        """a4+a5 of the newest snapshot on the side stream.  Full rank state (8(f4)): the caller first declares, in
        compute-stream order, that W holds every rank's parameters of this step (here only the own range changes)."""
        if self.full:
            self.s.params_ready(self.cur)
        self.s.flush_async(self.side)

    def time_flush(self):
        """One a4+a5 flush alone, timed on the side stream."""
        torch = self.torch
        self.do_step()
        torch.cuda.synchronize()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record(self.side)
        self.flush()
        f1.record(self.side)
        self.s.wait(self.step)
        torch.cuda.synchronize()
        return f0.elapsed_time(f1)

    def e2e(self, Ke, world=1):
        """Host buffers in, host replica out, through the same C-ABI calls."""
        torch = self.torch

        def loop(k_steps):
            for _ in range(k_steps):
                self.step += 1
                g = self.grads[self.step & 1]
                g.copy_(self.hgrads[self.step & 1], non_blocking=True)   # H2D of this step's inputs
                self.s.step_and_snapshot(g, self.step)
                self.flush()                                             # D2H of this step's result (a4 + a5)
            self.s.wait(self.step)
        loop(2)
        torch.cuda.synchronize()
        barrier(world)
        t0 = time.perf_counter()
        loop(Ke)
        torch.cuda.synchronize()
        barrier(world)
        return (time.perf_counter() - t0) * 1e3 / Ke

    def restore_timing(self):
        """Drop the live shard, restore from the host replica, recompute the in-flight step."""
        torch = self.torch
        torch.cuda.synchronize()
        self.s.drop_live()
        torch.cuda.synchronize()
        r0, r1, r2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        r0.record(self.cur)
        back = self.s.restore()
        r1.record(self.cur)
        self.step = back
        self.do_step()
        r2.record(self.cur)
        torch.cuda.synchronize()
        return back, r0.elapsed_time(r1), r1.elapsed_time(r2)

    def restore_two_phase(self, G, reps=3):
        """a6 in two phases (phx_restore_async, R37) and what it buys: the recomputed iteration (G GEMMs of
        forward/backward + the optimizer step) after a fault, three arms on the same stream —
          no_fault   : G GEMMs -> step                                   (the iteration itself)
          serial     : phx_restore -> G GEMMs -> step                     (one-phase restore, everything exposed)
          overlapped : phx_restore_async on the side stream, the compute stream waits for "parameters ready" only,
                       G GEMMs -> step (the step waits for the moments by itself).
        Exposed recovery time = arm - no_fault; median of `reps`."""
        torch = self.torch
        self.gemm_setup()

        def fresh_fault():
            self.do_step()
            self.flush()
            self.s.wait(self.step)
            torch.cuda.synchronize()
            self.s.drop_live()
            torch.cuda.synchronize()

        def timed(body):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(self.cur)
            body()
            e1.record(self.cur)
            torch.cuda.synchronize()
            return e0.elapsed_time(e1)

        def iteration():
            self.gemm_window(G)
            self.do_step()

        def serial():
            self.step = self.s.restore()
            iteration()

        def overlapped():
            self.side.wait_stream(self.cur)
            self.step = self.s.restore_async(self.side)
            self.s.restore_wait_params(self.cur)
            iteration()

        pr, sr = [], []
        for _ in range(reps):                      # latency to "parameters ready" / "state ready", nothing else running
            fresh_fault()
            r0, r1, r2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            r0.record(self.cur)
            self.side.wait_stream(self.cur)
            self.step = self.s.restore_async(self.side)
            r2.record(self.side)
            self.s.restore_wait_params(self.cur)
            r1.record(self.cur)
            torch.cuda.synchronize()
            pr.append(r0.elapsed_time(r1))
            sr.append(r0.elapsed_time(r2))
        arms = {"no_fault": [], "serial": [], "overlapped": []}
        for _ in range(reps):
            self.do_step()
            torch.cuda.synchronize()
            arms["no_fault"].append(timed(iteration))
            fresh_fault()
            arms["serial"].append(timed(serial))
            fresh_fault()
            arms["overlapped"].append(timed(overlapped))
        med = {k: sorted(v)[len(v) // 2] for k, v in arms.items()}
        return {"params_ready_ms": sorted(pr)[len(pr) // 2], "state_ready_ms": sorted(sr)[len(sr) // 2],
                "recomputed_iteration": {"gemms_per_iter": G, "compute_window_ms": G * self.gemm_ms,
                                         "no_fault_ms": med["no_fault"], "serial_restore_ms": med["serial"],
                                         "two_phase_restore_ms": med["overlapped"]},
                "exposed_recovery_ms_serial": med["serial"] - med["no_fault"],
                "exposed_recovery_ms_two_phase": med["overlapped"] - med["no_fault"], "repeats": reps,
                "note": "phx_restore_async: the parameters first on the side stream (p + bf16 copy; W alone for a full "
                        "rank state), the rest behind the recomputed iteration's forward/backward (stand-in GEMMs); the "
                        "step waits for it by itself"}

    def hotswap(self, G, two_phase=False):
        """BASELINE.json:configs[3]: 20 steps with snapshots (overlapped with G GEMMs each), the live shard is dropped
        while step 21 is in flight, restore from the pinned host replica, recompute 21, run 22..25; timed, and the
        trajectory compared bit for bit with an uninterrupted run (GPU vs GPU; GPU vs oracle is in tests/).
        two_phase: the recovery is phx_restore_async (parameters first, moments behind the recomputed iteration's G
        GEMMs of forward/backward); the timed region then holds that compute window too."""
        torch, W, wl, N = self.torch, self.W, self.wl, self.N
        torch.cuda.synchronize()
        self.s.p.copy_(W.init_params(self.s.n, N, wl.seed, device=self.device))
        self.s.m.zero_(); self.s.v.zero_()
        self.s.set_state(0)
        self.step = 0
        ref = self.Shard(wl, device=self.device, snapshot=False)
        ref.p.copy_(self.s.p); ref.set_state(0)
        for t in range(1, 26):
            ref.step_and_snapshot(self.grads[t & 1], t)
        torch.cuda.synchronize()
        self.gemm_setup()
        after_20 = torch.cuda.Event()
        for t in range(1, 21):
            self.gemm_window(G)
            self.do_step()
            if t == 20:
                after_20.record(self.cur)
            self.s.flush_async(self.side)
        self.do_step()                                # step 21 launched: in flight when the fault hits
        # The fault lands from a SECOND stream that waits for step 20's kernel only, with no host synchronisation
        # (the scenario of tests/test_gpu_fullsize.py): flush(20) is being DMA'd and step 21 is queued
        # behind the sync point / running while the live planes are zeroed and step 21's staging slot is scribbled.
        if self._fault_stream is None:
            self._fault_stream = torch.cuda.Stream(device=self.device)
        self._fault_stream.wait_event(after_20)
        with torch.cuda.stream(self._fault_stream):
            for x in (self.s.p, self.s.m, self.s.v, self.s.p16, self.s.W):
                if x is not None:
                    x.zero_()
            if self.s.staging is not None:
                self.s.staging_slot(21).fill_(0xA5)
        self.cur.wait_stream(self._fault_stream)      # recovery is ordered after the fault on the device only
        t0 = time.perf_counter()
        r0, r1, r2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        r0.record(self.cur)
        if two_phase:
            self.side.wait_stream(self.cur)
            back = self.s.restore_async(self.side)
            self.s.restore_wait_params(self.cur)      # forward/backward may start: the parameters are back
            r1.record(self.cur)
            self.gemm_window(G)
        else:
            back = self.s.restore()
            r1.record(self.cur)
        self.step = back
        self.do_step()                                # recompute of the in-flight step (a7)
        r2.record(self.cur)
        torch.cuda.synchronize()
        wall_ms = (time.perf_counter() - t0) * 1e3
        for t in range(22, 26):
            self.do_step()
            self.s.flush_async(self.side)
        self.s.wait(25)
        torch.cuda.synchronize()
        same = all(torch.equal(x, y) for x, y in ((self.s.p, ref.p), (self.s.m, ref.m), (self.s.v, ref.v),
                                                  (self.s.p16, ref.p16)))
        ref.close()
        del ref
        rms = r0.elapsed_time(r1)
        if two_phase:
            return {"restored_step": int(back), "params_ready_ms": rms, "recomputed_iteration_ms": r1.elapsed_time(r2),
                    "compute_window_ms": G * self.gemm_ms, "recovery_plus_recomputed_iteration_ms": r0.elapsed_time(r2),
                    "trajectory_bit_exact_vs_uninterrupted": bool(same), "gemms_per_iter": G, "mode": self.restore_mode_name,
                    "note": "phx_restore_async: the timed region holds the recomputed iteration's G GEMMs; m and v "
                            "come back behind them"}
        return {"restored_step": int(back), "restore_ms": rms, "recompute_ms": r1.elapsed_time(r2),
                "restore_plus_recompute_ms": r0.elapsed_time(r2), "restore_plus_recompute_wall_ms": wall_ms,
                "host_link_gbs": 12 * N / (rms * 1e-3) / 1e9, "trajectory_bit_exact_vs_uninterrupted": bool(same),
                "steps_before_fault": 20, "steps_after": 5, "gemms_per_iter": G, "mode": self.restore_mode_name,
                "fault": "second stream, no host sync: lands while flush(20) is in flight and step 21 is queued or running; the timed "
                         "region starts on the compute stream behind step 21"}

    # -- the stand-in compute window ----------------------------------------------------------------
    def gemm_setup(self):
        torch = self.torch
        if self._gemm is None:
            a = torch.randn(4096, 4096, device=self.device, dtype=torch.bfloat16)
            b = torch.randn(4096, 4096, device=self.device, dtype=torch.bfloat16)
            c = torch.empty(4096, 4096, device=self.device, dtype=torch.bfloat16)
            self._gemm = (a, b, c)
            for _ in range(20):
                torch.matmul(a, b, out=c)
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(self.cur)
            for _ in range(200):
                torch.matmul(a, b, out=c)
            g1.record(self.cur)
            torch.cuda.synchronize()
            self.gemm_ms = g0.elapsed_time(g1) / 200
        return self.gemm_ms

    def gemm_window(self, G):
        """The stand-in compute window: G bf16 4096^3 GEMMs (BASELINE.json:configs[1])."""
        a, b, c = self._gemm
        mm = self.torch.matmul
        for _ in range(G):
            mm(a, b, out=c)

    def gemms_for(self, flush_ms, factor=4.0, pow2=True):
        """R21: smallest power of two G with T_c >= factor x T_D2H (or the plain quotient for the tight window)."""
        gm = self.gemm_setup()
        if not pow2:
            return max(1, int(round(factor * flush_ms / gm)))
        G = 64
        while G * gm < factor * flush_ms:
            G *= 2
        return G

    def iters_for(self, G):
        if self.args.overlap_iters > 0:
            return self.args.overlap_iters
        t_iter = (G * self.gemm_ms * 1.1 + 1.0) * 1e-3
        return max(8, min(30, int(self.args.overlap_secs / t_iter)))

    def overlap(self, G, iters, arms=("off", "on"), warm=2, reps=1):
        """Iterations of G GEMMs + the hot path, EAGERLY launched, arms alternated `reps` times:
          off    — snapshot-disabled kernel, no flush (the paper's baseline run);
          staged — snapshot-on kernel (writes the staging slot), no flush;
          on     — snapshot-on kernel + flush on the side stream (PHOENIX enabled).
        Per-iteration times from CUDA events on the compute stream; PAPER.md:283 trimming."""
        torch = self.torch
        self.gemm_setup()
        it_ms = {k: [] for k in arms}
        hp_ms = {k: [] for k in arms}
        for rep in range(reps):
            # the arms alternate AND swap their order from one repetition to the next (off, on | on, off | ...), so
            # that a drift of the GEMM rate over the leg (the board warming up to its power limit) does not always
            # land on the same arm
            for arm in (arms if rep % 2 == 0 else tuple(reversed(arms))):
                evs, kevs = [], []
                for it in range(warm + iters):
                    e0 = torch.cuda.Event(enable_timing=True)
                    e0.record(self.cur)
                    self.gemm_window(G)
                    k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    k0.record(self.cur)
                    if arm == "off":
                        self.do_step_off()
                    else:
                        self.do_step()
                    k1.record(self.cur)
                    if arm == "on":
                        self.flush()
                        if self.k_peers and self.peers_in_overlap:
                            self.B.phx_snapshot_flush_peers_async(self.s.h, self.peer_stream)
                    evs.append(e0)
                    kevs.append((k0, k1))
                end = torch.cuda.Event(enable_timing=True)
                end.record(self.cur)
                torch.cuda.synchronize()
                if arm == "on":
                    self.s.wait(self.step)
                    if self.k_peers and self.peers_in_overlap:
                        self.B.phx_snapshot_wait_peers(self.s.h, self.step)
                evs.append(end)
                it_ms[arm] += [evs[i].elapsed_time(evs[i + 1]) for i in range(warm, warm + iters)]
                hp_ms[arm] += [x.elapsed_time(y) for x, y in kevs[warm:]]
        t = {k: trimmed_mean(v) for k, v in it_ms.items()}
        out = {"gemms_per_iter": G, "gemm_ms": self.gemm_ms, "compute_window_ms": G * self.gemm_ms,
               "launch": "eager", "iters_per_arm": iters * reps,
               "protocol": "PAPER.md:283: warm-up dropped, slowest 5% dropped, mean of the rest"}
        for k in arms:
            out[f"iter_ms_{k}"] = t[k]
            out[f"hot_path_ms_in_loop_{k}"] = trimmed_mean(hp_ms[k])
        if "on" in t and "off" in t:
            out["exposed_ms"] = t["on"] - t["off"]
            out["exposed_frac_of_compute_step"] = (t["on"] - t["off"]) / t["off"]
        if "staged" in t and "off" in t:
            out["exposed_ms_kernel_only"] = t["staged"] - t["off"]
        return out

    def overlap_graph_step(self, G, iters, warm=1, arms=("off", "on")):
        """The same experiment with the WHOLE iteration captured in a CUDA graph — the B200-native launch form
        (DESIGN.md §12): [flush of snapshot k-1 on the side stream ‖ G GEMMs] -> step k, L = lcm(staging depth, 2)
        iterations per graph (staging / host slot ping-pong), through the graph-capturable form of the step
        (phx_graph_*).  Arms: off = snapshot-disabled handle, no flush; on = snapshots + flush.  One eager event pair
        per replay: iteration time = replay time / L."""
        torch, B = self.torch, self.B
        self.gemm_setup()
        hp = self.wl.hyper
        cap = torch.cuda.Stream(device=self.device)
        L = {1: 2, 2: 2, 3: 6, 4: 4}[self.depth] if self.source_name == "staged" else 2
        nrep = max(3, (iters + L - 1) // L)
        with torch.cuda.stream(cap):
            self.gemm_window(2)                                          # cuBLAS handle / workspace of this stream exist before capture
        torch.cuda.synchronize()
        graphs = {}
        for arm in arms:                                                 # capture every arm once; the handles differ, the live memory is shared
            h = self.off_shard() if arm == "off" else self.s.h
            B.phx_graph_begin(h, hp.lr, hp.beta1, hp.beta2, hp.eps, hp.wd, cap)
            B.phx_graph_step_and_snapshot(h, self.grads[1], cap)         # a snapshot for the first captured flush
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=cap):
                for i in range(L):
                    if arm == "on":
                        self.side.wait_stream(cap)                       # fork: the flush runs beside the window
                        B.phx_graph_flush_async(h, self.side)
                    self.gemm_window(G)
                    B.phx_graph_step_and_snapshot(h, self.grads[i & 1], cap)   # a2 joins the flush back
                if arm == "on":
                    cap.wait_stream(self.side)
            graphs[arm] = (h, graph)
        # timed blocks in swapped order (off, on | on, off) like the eager arms, one warm-up replay per block
        order = list(arms) + list(reversed(arms)) if len(arms) > 1 else list(arms)
        per_block = max(2, (nrep + 1) // 2) if len(arms) > 1 else nrep
        ms = {arm: [] for arm in arms}
        for arm in order:
            graph = graphs[arm][1]
            times = []
            with torch.cuda.stream(cap):                                 # replay() launches on the current stream
                for r in range(warm + per_block):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(cap)
                    graph.replay()
                    e1.record(cap)
                    times.append((e0, e1))
            torch.cuda.synchronize()
            ms[arm] += [a.elapsed_time(b) / L for a, b in times[warm:]]
        res = {arm: trimmed_mean(v) for arm, v in ms.items()}
        for arm in arms:
            h, graph = graphs[arm]
            last = B.phx_graph_end(h)
            if arm == "on":
                self.step = last
                self.s.flush_async(self.side)                            # the newest snapshot is still staged
                self.s.wait(self.step)
            else:
                self.off_step = last
            del graph
        nrep = per_block * (2 if len(arms) > 1 else 1)
        out = {"gemms_per_iter": G, "compute_window_ms": G * self.gemm_ms, "launch": f"cuda graph ({L} iterations per graph)",
               "iters_per_arm": L * nrep}
        for arm in arms:
            out[f"iter_ms_{arm}"] = res[arm]
        if "on" in res and "off" in res:
            out["exposed_ms"] = res["on"] - res["off"]
            out["exposed_frac_of_compute_step"] = (res["on"] - res["off"]) / res["off"]
        return out

    def close(self):
        self.close_peers()
        if self.s_off is not None:
            self.B.phx_shard_destroy(self.s_off)
            self.s_off = None
        self.s.close()


def measure_host_link(torch, device, nbytes=1 << 30, reps=10):
    """Measured pinned-copy peak of the host link, each direction (north_star)."""
    h = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d = torch.empty(nbytes, dtype=torch.uint8, device=device)
    out = {}
    for name, (dst, src) in (("d2h_gbs", (h, d)), ("h2d_gbs", (d, h))):
        best = 0.0
        for _ in range(reps + 1):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            dst.copy_(src, non_blocking=True)
            e1.record()
            torch.cuda.synchronize()
            best = max(best, nbytes / (e0.elapsed_time(e1) * 1e-3) / 1e9)
        out[name] = best
    del h, d
    return out


def measure_hbm_mix_ceiling(torch, device, plane_elems, reps=150):
    """No-arithmetic streaming passes with the fused kernel's access pattern (libphx_probe.so, bench-only): the HBM
    ceiling for a read:write mix.  Returns GB/s per mix; planes of `plane_elems` fp32 each (larger than L2)."""
    from paper_2607_01646_b200 import probe as PB
    mixes = {"read_only_4r": (4, 0), "write_only_4w": (0, 4), "copy_1r1w": (1, 1), "step_mix_3r6w": (3, 6),
             "off_mix_3r3w": (3, 3)}
    plane_bytes = int(plane_elems) * 4
    buf = torch.empty(9 * plane_bytes, dtype=torch.uint8, device=device)
    buf.zero_()
    st = torch.cuda.current_stream(device)
    out = {}
    for name, (r, w) in mixes.items():
        for _ in range(3):
            assert PB.phx_hbm_probe_async(buf, plane_bytes, r, w, st) == 0
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for _ in range(reps):
            PB.phx_hbm_probe_async(buf, plane_bytes, r, w, st)
        e1.record(st)
        torch.cuda.synchronize()
        out[name] = (r + w) * plane_bytes / (e0.elapsed_time(e1) / reps * 1e-3) / 1e9
    del buf
    return out


def gpu_setup(args):
    import torch
    rank, world, local_rank = rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl phx needs a B200: there is no CPU fallback")
    if args.debug_shared_gpu:
        local_rank = 0
    elif world > 1 and torch.cuda.device_count() < world:
        raise SystemExit(f"bench.py: {world} ranks but {torch.cuda.device_count()} CUDA device(s)")
    torch.cuda.set_device(local_rank)
    dist_init(world, not args.debug_shared_gpu)
    return torch, rank, world, local_rank


# ----------------------------------------------------------------------------------------------
# one config: every number of SURVEY.md §8(d) for it
# ----------------------------------------------------------------------------------------------


def measure_config(args, key, link, clk, rank, world, local_rank, K, Wm, peak, headline, n_head):
    """Returns (record, extras): `record` goes into the line's `configs` array; `extras` carries what only the
    headline config reports at top level (launch count, per-step times, the Rig itself for the N > 1 legs).
    K is exact on the headline config; the other configs run as many steps as move the same number of elements
    (so every step leg lasts about as long and gets its share of clock samples)."""
    import torch
    rig = Rig(args, key, rank, world, local_rank)
    device, N, wl, B = rig.device, rig.N, rig.wl, rig.B
    if not headline and n_head:
        K = max(K, int(math.ceil(K * n_head / N)))
    tag = key
    BPE = rig.bytes_per_elem
    step_bpe = step_bytes_per_elem(wl, rig.source_name)
    rec = {"config": key, "workload": wl.title, "elements": int(N), "state_bytes": int(12 * N),
           "clip": "local a1 pass over the bf16 gradients" if rig.clip else "none"}

    # ---- the step: K back-to-back a1..a3 passes, inputs resident in HBM --------------------------------
    for _ in range(Wm):
        rig.do_step()
    torch.cuda.synchronize()
    barrier(world)
    with clk.leg(f"{tag}.step"):
        total_ms, per, launches = rig.time_steps(K, 0)
    barrier(world)
    step_ms = max_over_ranks(total_ms, world, device) / K
    with clk.leg(f"{tag}.kernel"):
        kern_ms = rig.time_fused_kernel_alone(K) if rig.clip else step_ms
        off_ms = rig.time_steps_off(K)
    step_gbs = step_bpe * N / (step_ms * 1e-3) / 1e9
    kern_gbs = BPE * N / (kern_ms * 1e-3) / 1e9
    rec.update(step_ms=step_ms, step_bytes_per_element=step_bpe, step_gbs=step_gbs,
               step_frac_of_measured_peak=step_gbs / peak,
               kernel_ms=kern_ms, kernel_bytes_per_element=BPE, kernel_gbs=kern_gbs,
               kernel_frac_of_measured_peak=kern_gbs / peak, kernel_frac_of_nominal_8TBps=kern_gbs / NOMINAL_HBM_GBS,
               elements_per_s=N / (step_ms * 1e-3), snapshot_off_step_ms=off_ms,
               host_enqueue_us_per_step=rig.host_enqueue_us,   # Python binding + C call + launches, first 48 steps
               snapshot_off_gbs=(step_bpe - 12) * N / (off_ms * 1e-3) / 1e9, steps_timed=K)
    if rig.clip and not rig.fp32 and rank == 0:
        with clk.leg(f"{tag}.producer_clip"):
            fin_ms, pstep_ms, pl = rig.time_producer_clip(max(50, K // 2))
        rec["clip_source_producer"] = {
            "clip_source": "producer", "step_ms": pstep_ms, "step_bytes_per_element": BPE,
            "step_gbs": BPE * N / (pstep_ms * 1e-3) / 1e9, "kernels_per_step": pl,
            "finalize_ms": fin_ms, "finalize_bytes_per_element": 6,
            "finalize_gbs": 6 * N / (fin_ms * 1e-3) / 1e9,
            "note": "SURVEY 8(f4b): phx_grads_finalize_async (fp32 main grads -> bf16 + fp64 sum of squares, ONE pass, "
                    "in the gradient producer) + phx_set_clip_partials(count=1): the step runs no a1 pass"}
    extras = {"launches": int(launches), "per_step": per, "rig": rig}

    # ---- e2e: host buffers through the same C-ABI calls --------------------------------------------------
    d2h_bytes = int(rig.s.info.host_snapshot_bytes)
    h2d_bytes = int(rig.grad_bytes * N)
    est = (d2h_bytes / (link["d2h_gbs"] * 1e9) if link else 0.05) * 1e3
    Ke = args.e2e_steps or max(10, int(math.ceil(1500.0 / est)))
    with clk.leg(f"{tag}.e2e"):
        e2e_ms = max_over_ranks(rig.e2e(Ke, world), world, device)
    rec["e2e"] = {"ms_per_step": e2e_ms, "steps": Ke, "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": d2h_bytes,
                  "link_gbs": (h2d_bytes + d2h_bytes) / (e2e_ms * 1e-3) / 1e9,
                  "metric_gbs": step_bpe * N / (e2e_ms * 1e-3) / 1e9}
    if rank != 0:
        return rec, extras

    # ---- flush alone (a4+a5) against the measured pinned-copy peak -------------------------------------
    with clk.leg(f"{tag}.flush"):
        nfl = max(3, int(math.ceil(800.0 / est)))
        fl = sorted(rig.time_flush() for _ in range(nfl))
    flush_ms = fl[0]
    ach = d2h_bytes / (flush_ms * 1e-3) / 1e9
    rec["flush"] = {"ms": flush_ms, "ms_median": fl[len(fl) // 2], "repeats": nfl, "gbs": ach,
                    "frac_of_d2h_peak": ach / link["d2h_gbs"], "chunk_mib": rig.chunk_mib, "bytes": d2h_bytes}

    # ---- exposed checkpoint ms/iteration (PAPER.md:283 protocol) ----------------------------------------
    if not args.no_overlap:
        ov = {}
        for wname, factor, pow2 in (("headline_window", 4.0, True), ("tight_window", 1.25, False)):
            G = args.gemms if (args.gemms > 0 and pow2) else rig.gemms_for(flush_ms, factor, pow2)
            iters = rig.iters_for(G)
            with clk.leg(f"{tag}.overlap.{wname}.eager"):
                o = rig.overlap(G, max(4, (iters + 1) // 2), reps=2)
            w = {"rule": ("G = smallest power of two with T_c >= 4 x T_D2H" if pow2 else "G = round(1.25 x T_D2H / T_gemm)")
                 if args.gemms <= 0 or not pow2 else "G given", "gemms_per_iter": G,
                 "compute_window_ms": G * rig.gemm_ms, "flush_ms": flush_ms, "iter_ms_off": o["iter_ms_off"],
                 "exposed_ms_eager": o["exposed_ms"], "exposed_pct_eager": 100.0 * o["exposed_frac_of_compute_step"],
                 "iter_ms_on_eager": o["iter_ms_on"], "iters_per_arm": o["iters_per_arm"]}
            if not args.no_graph_step and not rig.full:
                with clk.leg(f"{tag}.overlap.{wname}.graph_step"):
                    og = rig.overlap_graph_step(G, iters)
                w.update(iter_ms_off_graph_step=og["iter_ms_off"], iter_ms_on_graph_step=og["iter_ms_on"],
                         exposed_ms_graph_step=og["exposed_ms"],
                         exposed_pct_graph_step=100.0 * og["exposed_frac_of_compute_step"])
            # SURVEY 8(d) decomposition: the kernel's own share (12 B/element of staging stores, from the isolated
            # step timings above) vs everything else (sync-point stall + slowdown of the window under copy traffic)
            kd = step_ms - off_ms
            w["exposed_decomposition_ms"] = {"kernel_delta_isolated": kd, "rest_eager": o["exposed_ms"] - kd}
            if "exposed_ms_graph_step" in w:
                w["exposed_decomposition_ms"]["rest_graph_step"] = w["exposed_ms_graph_step"] - kd
            ov[wname] = w
        rec["overlap"] = ov
        rec["exposed_ckpt_ms_per_iter"] = ov["headline_window"]["exposed_ms_eager"]
        rec["exposed_pct"] = ov["headline_window"]["exposed_pct_eager"]

    # ---- restore + recompute (a6, a7); the c4 hot-swap scenario ----------------------------------------
    with clk.leg(f"{tag}.restore"):
        nrs = max(3, int(math.ceil(800.0 / est)))
        rs = sorted((rig.restore_timing() for _ in range(nrs)), key=lambda x: x[1])   # same committed slot every time
        back, rms, cms = rs[0]
        rec["restore"] = {"restore_ms": rms, "restore_ms_median": rs[len(rs) // 2][1], "repeats": nrs, "recompute_ms": cms,
                          "restore_plus_recompute_ms": rms + cms,
                          "mode": rig.restore_mode_name, "restored_step": int(back),
                          "host_link_gbs": (d2h_bytes - 256) / (rms * 1e-3) / 1e9,
                          "frac_of_h2d_peak": (d2h_bytes - 256) / (rms * 1e-3) / 1e9 / link["h2d_gbs"]}
        if not args.no_overlap:
            rec["restore"]["two_phase"] = rig.restore_two_phase(rig.gemms_for(flush_ms, 1.25, False))
        if key in ("c4a", "c4b"):
            rec["hotswap"] = rig.hotswap(rig.gemms_for(flush_ms, 1.25, False))
            if not args.no_overlap:
                rec["hotswap"]["two_phase"] = rig.hotswap(rig.gemms_for(flush_ms, 1.25, False), two_phase=True)
    return rec, extras


def measure_direct_source(args, key, link, clk, replica, K):
    """The same config with PHX_SNAPSHOT_DIRECT: no staging ring and no staging stores — under the paper's own sync
    point the flush DMAs the live planes themselves, the kernel moves 28 B/element.  Kernel, flush and
    the exposed checkpoint time at the tight window in both launch forms."""
    import torch
    rig = Rig(args, key, source="direct", replica=replica, host_grads=False)
    N = rig.N
    for _ in range(3):
        rig.do_step()
    with clk.leg(f"{key}.direct.step"):
        tot, _, _ = rig.time_steps(K, 0)
        kern_ms = rig.time_fused_kernel_alone(K) if rig.clip else tot / K
    with clk.leg(f"{key}.direct.flush"):
        fl = sorted(rig.time_flush() for _ in range(9))
    flush_ms = fl[0]
    out = {"snapshot_source": "direct", "step_ms": tot / K, "kernel_ms": kern_ms, "kernel_bytes_per_element": BYTES_PER_ELEM_OFF,
           "kernel_gbs": BYTES_PER_ELEM_OFF * N / (kern_ms * 1e-3) / 1e9, "flush_ms": flush_ms,
           "flush_gbs": (256 + 12 * N) / (flush_ms * 1e-3) / 1e9,
           "flush_frac_of_d2h_peak": (256 + 12 * N) / (flush_ms * 1e-3) / 1e9 / link["d2h_gbs"], "overlap": {}}
    # the tight window only in the default line (the staged source reports both; `--config c3 --source direct` gives
    # the direct source's full record)
    for wname, factor, pow2 in (("tight_window", 1.25, False),):
        G = rig.gemms_for(flush_ms, factor, pow2)
        iters = rig.iters_for(G)
        with clk.leg(f"{key}.direct.overlap.{wname}"):
            o = rig.overlap(G, iters)
            w = {"gemms_per_iter": G, "iter_ms_off": o["iter_ms_off"], "exposed_ms_eager": o["exposed_ms"],
                 "exposed_pct_eager": 100.0 * o["exposed_frac_of_compute_step"]}
            if not args.no_graph_step:
                og = rig.overlap_graph_step(G, iters)
                w.update(iter_ms_off_graph_step=og["iter_ms_off"], exposed_ms_graph_step=og["exposed_ms"],
                         exposed_pct_graph_step=100.0 * og["exposed_frac_of_compute_step"])
        out["overlap"][wname] = w
    rig.close()
    del rig
    torch.cuda.empty_cache()
    return out


def measure_c5_grid(args, link, clk, replica, flush_ref):
    """BASELINE.json:configs[4]: D2H chunk size x staging depth at the TIGHT window (T_c = 1.25 x T_D2H, where
    depth and chunking can matter): exposed checkpoint ms/iteration and host-link GB/s per cell; reduced grid in the
    default line (the full 7 x 4 x 2 grid is `--mode sweep`)."""
    import torch
    cells = []
    base = base_g = G = None
    for sync, depth, chunk in [("strict", 2, 4), ("strict", 2, 16), ("strict", 2, 64), ("strict", 2, 256),
                               ("strict", 1, 8), ("relaxed", 4, 8), ("relaxed", 4, 64), ("relaxed", 3, 256)]:
        rig = Rig(args, "c5", depth=depth, chunk_mib=chunk, sync=sync, replica=replica, host_grads=False)
        rig.gemm_setup()
        if G is None:       # ONE window for the baseline and every cell (the per-rig GEMM timing moves by a few per cent)
            G = max(1, int(round(1.25 * flush_ref / rig.gemm_ms)))
        iters = max(8, min(16, rig.iters_for(G)))
        if base is None:
            base = rig.overlap(G, iters, arms=("off",))["iter_ms_off"]
            if not args.no_graph_step:
                base_g = rig.overlap_graph_step(G, 8, arms=("off",))["iter_ms_off"]
        fl = rig.time_flush()
        o = rig.overlap(G, iters, arms=("on",))
        cell = {"sync_mode": sync, "depth": depth, "chunk_mib": chunk, "flush_ms": fl,
                "host_link_gbs": (256 + 12 * rig.N) / (fl * 1e-3) / 1e9, "gemms_per_iter": G,
                "iter_ms_on": o["iter_ms_on"], "iter_ms_off": base, "exposed_ms": o["iter_ms_on"] - base,
                "exposed_pct": 100.0 * (o["iter_ms_on"] - base) / base}
        if base_g is not None:
            og = rig.overlap_graph_step(G, 8, arms=("on",))
            cell.update(iter_ms_on_graph_step=og["iter_ms_on"], iter_ms_off_graph_step=base_g,
                        exposed_ms_graph_step=og["iter_ms_on"] - base_g,
                        exposed_pct_graph_step=100.0 * (og["iter_ms_on"] - base_g) / base_g)
        cells.append(cell)
        last_cell = (sync, depth, chunk) == ("relaxed", 3, 256)
        if last_cell:       # the snapshot-off baseline once more AFTER the cells: the mean of the two brackets the drift
            base2 = rig.overlap(G, iters, arms=("off",))["iter_ms_off"]
            base2_g = None if base_g is None else rig.overlap_graph_step(G, 8, arms=("off",))["iter_ms_off"]
        rig.close()
        del rig
        torch.cuda.empty_cache()
    b, bg = 0.5 * (base + base2), None if base_g is None else 0.5 * (base_g + base2_g)
    for c in cells:         # re-reference every cell to the bracketing baseline
        c.update(iter_ms_off=b, exposed_ms=c["iter_ms_on"] - b, exposed_pct=100.0 * (c["iter_ms_on"] - b) / b,
                 iter_ms_off_before_after=[base, base2])
        if bg is not None:
            c.update(iter_ms_off_graph_step=bg, exposed_ms_graph_step=c["iter_ms_on_graph_step"] - bg,
                     exposed_pct_graph_step=100.0 * (c["iter_ms_on_graph_step"] - bg) / bg,
                     iter_ms_off_graph_step_before_after=[base_g, base2_g])
    best = min(cells, key=lambda c: c["exposed_ms"])
    worst = max(cells, key=lambda c: c["exposed_ms"])
    return {"window": "tight: T_c = 1.25 x T_D2H", "d2h_peak_gbs": link["d2h_gbs"], "best": best, "worst": worst,
            "cells": cells, "note": "reduced grid; the full chunk {4..256} x depth {1..4} x sync grid is --mode sweep"}


def multi_gpu_legs(args, rig, rank, world, clk):
    """The N > 1 rows on the headline config: the ring send over real CUDA-IPC peers
    (k = 1 and 2), restore from the holder, the parameter publication fused vs copy engine, the DP-global clip."""
    import torch
    from paper_2607_01646_b200 import ring as PR
    B, device, N, wl = rig.B, rig.device, rig.N, rig.wl
    out = {}
    # ---- f1: ring replication ---------------------------------------------------------------------------
    ks = [args.peers] if args.peers > 0 else ([1, 2] if world > 1 and args.peers < 0 else [])
    ks = [k for k in ks if world == 1 or k <= world - 1]
    peer_rows = []
    for k in ks:
        row = {"k": k}
        try:
            row["link"] = rig.setup_peers(k, rank, world)
            with clk.leg(f"peers.k{k}"):
                pf_ms = max_over_ranks(min(rig.time_peer_flush() for _ in range(3)), world, device)
            pbytes = k * int(rig.s.info.snapshot_bytes)
            row.update(flush_ms=pf_ms, bytes_per_step=pbytes, gbs_per_gpu=pbytes / (pf_ms * 1e-3) / 1e9,
                       streams="one copy stream per peer" if k > 1 else "caller's stream",
                       note="replication of one packed snapshot to all k peers, copy engine, alone; max over ranks, "
                            "all ranks sending at once")
            # the flush to the peers INSIDE the overlap arm (with the host flush): does NVLink traffic expose anything?
            if not args.no_overlap and world > 1:
                rig.peers_in_overlap = True
                fl = rig.time_flush()
                G = rig.gemms_for(fl, 4.0, True)
                with clk.leg(f"peers.k{k}.overlap"):
                    o = rig.overlap(G, rig.iters_for(G))
                row["overlap_with_host_and_peer_flush"] = {
                    "gemms_per_iter": G, "iter_ms_off": o["iter_ms_off"], "iter_ms_on": o["iter_ms_on"],
                    "exposed_ms": max_over_ranks(o["exposed_ms"], world, device)}
                rig.peers_in_overlap = False
            # recovery stage 3: restore from the ring successor's received buffer
            src = rig.ring.opened[0] if world > 1 else rig.recv.ptrs[0]
            rig.s.drop_live()
            torch.cuda.synchronize()
            p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            p0.record(rig.cur)
            back = B.phx_restore_from(rig.s.h, src, rig.cur)
            p1.record(rig.cur)
            torch.cuda.synchronize()
            rig.step = back
            pms = max_over_ranks(p0.elapsed_time(p1), world, device)
            row.update(restore_from_holder_ms=pms, restore_from_holder_gbs=12 * N / (pms * 1e-3) / 1e9,
                       restored_step=int(back))
        except Exception as e:  # noqa: BLE001  (PeerRing makes every rank fail together)
            row["error"] = str(e)[:300]
        barrier(world)
        rig.close_peers()
        peer_rows.append(row)
    if peer_rows:
        out["peer_replication"] = peer_rows

    # ---- f3: parameter publication ------------------------------------------------------------------------
    pmodes = {"auto": (["fused", "copy"] if world > 1 else []), "none": [], "both": ["fused", "copy"],
              "fused": ["fused"], "copy": ["copy"]}[args.publish]
    pubs = []
    for name in pmodes:
        pmode = B.PHX_PUBLISH_FUSED if name == "fused" else B.PHX_PUBLISH_COPY_ENGINE
        pub_stream = torch.cuda.Stream(device=device)
        row = {"mode": name}
        try:
            lbufs = None
            if world > 1:
                pg, nb = PR.ParamGroup(rig.s, pmode, ring_size=world, ring_rank=rank), world
                row["link"] = "P2P into every rank's parameter buffer (CUDA IPC), own buffer included"
            else:
                nb = min(wl.dp_size - 1, B.PHX_MAX_PARAM_PEERS)
                lbufs = [torch.zeros(wl.dp_size * N, dtype=torch.float32 if rig.fp32 else torch.bfloat16, device=device)
                         for _ in range(nb)]
                B.phx_shard_bind_param_peers(rig.s.h, lbufs, pmode)
                pg = None
                row["link"] = "loopback stand-in: dp_size-1 parameter buffers on the SAME GPU (HBM writes, not NVLink)"
            for _ in range(3):
                rig.do_step()
            torch.cuda.synchronize()
            barrier(world)
            q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with clk.leg(f"publish.{name}"):
                q0.record(rig.cur)
                for _ in range(20):
                    rig.do_step()
                    if pmode == B.PHX_PUBLISH_COPY_ENGINE:
                        B.phx_publish_params_async(rig.s.h, pub_stream)
                        rig.cur.wait_stream(pub_stream)      # the next forward pass needs the published parameters
                q1.record(rig.cur)
                torch.cuda.synchronize()
            barrier(world)
            pms = max_over_ranks(q0.elapsed_time(q1) / 20, world, device)
            row.update(buffers_written=nb, step_plus_publish_ms=pms,
                       bytes_published_per_step=int(nb * N * (4 if rig.fp32 else 2)))
            B.phx_shard_bind_param_peers(rig.s.h, [])
            if pg is not None:
                pg.close()
            del lbufs
        except Exception as e:  # noqa: BLE001
            row["error"] = str(e)[:300]
        barrier(world)
        pubs.append(row)
    if pubs:
        out["publication"] = pubs

    # ---- (e): the DP-global clip on a config that has one -----------------------------------------------------
    scope = args.clip_scope
    if rig.clip and (scope == "global" or (scope == "auto" and world > 1)):
        from paper_2607_01646_b200.clip import GlobalClip
        gc = GlobalClip(rig.s)
        rig.gclip = gc
        for _ in range(3):
            rig.do_step()
        torch.cuda.synchronize()
        barrier(world)
        with clk.leg("global_clip"):
            tot, _, l = rig.time_steps(50, 0)
        barrier(world)
        rig.gclip = None
        out["global_clip"] = {"step_ms": max_over_ranks(tot, world, device) / 50, "kernels_per_step": l / 50,
                              "exchange": "all-gather of one fp64 sum per rank (8 x %d bytes), then the fixed-tree sum "
                                          "inside the step" % world,
                              "backend": "nccl" if not args.debug_shared_gpu and world > 1 else
                                         ("gloo via host staging (debug)" if world > 1 else "single rank")}
    return out


def run_headline(args):
    torch, rank, world, local_rank = gpu_setup(args)
    device = torch.device(f"cuda:{local_rank}")
    K, Wm = args.steps, max(args.warmup, 3)
    keys = [k for k in (args.configs.split(",") if args.configs else (ALL_CONFIGS if world == 1 else [args.headline])) if k]
    if args.headline not in keys:
        keys.append(args.headline)
    try:
        uuid = "GPU-" + str(torch.cuda.get_device_properties(local_rank).uuid)
    except Exception:
        uuid = ""
    clk = ClockLog(local_rank, uuid=uuid) if rank == 0 else contextlib.nullcontext()
    if rank != 0:
        clk = type("NoClk", (), {"leg": staticmethod(lambda name: contextlib.nullcontext())})()
    link = measure_host_link(torch, device) if rank == 0 else {}
    if world > 1:   # every rank needs an estimate for its e2e step count; rank 0's measurement is the one reported
        link0 = [link]
        import torch.distributed as dist
        dist.broadcast_object_list(link0, src=0)
        link_all = link0[0]
    else:
        link_all = link
    peak, peak_src = measured_peaks()

    records, head, head_extras = [], None, None
    n_head = shard_elements(args, args.headline)
    for key in keys:
        is_head = key == args.headline
        rec, extras = measure_config(args, key, link_all, clk, rank, world, local_rank, K, Wm, peak, is_head, n_head)
        rig = extras.pop("rig")
        if is_head:
            head, head_extras = rec, extras
            # ---- roofline of the dominant kernel, on the headline config ------------------------------------
            BPE, N = rig.bytes_per_elem, rig.N
            tkey = key + ("" if rig.source_name == "staged" else "-direct") + ("-fp32" if rig.fp32 else "") + \
                ("-groups" if args.decay_groups else "")
            roofline = {"bound": "hbm", "achieved": rec["kernel_gbs"], "peak": peak, "unit": "GB/s",
                        "frac": rec["kernel_gbs"] / peak, "traffic": committed_traffic(tkey), "peak_source": peak_src,
                        "frac_of_nominal_8TBps": rec["kernel_gbs"] / NOMINAL_HBM_GBS, "kernel": rig.kernel_name(),
                        "kernel_ms": rec["kernel_ms"], "step_ms": rec["step_ms"],
                        "algorithmic_bytes_per_launch": BPE * N, "bytes_per_element": BPE,
                        "note": "kernel_ms: the fused kernel alone (a second handle with the clip off on the same memory); "
                                "step_ms: the whole device-side hot path incl. the a1 pass where the config has one"}
            if rank == 0 and not args.no_mix_ceiling:
                with clk.leg("mix_ceiling"):
                    ceil = measure_hbm_mix_ceiling(torch, device, N)
                roofline["mix_ceiling_gbs"] = ceil
                roofline["frac_of_mix_ceiling"] = rec["kernel_gbs"] / ceil["off_mix_3r3w" if rig.source_name == "direct"
                                                                          else "step_mix_3r6w"]
            head_extras["roofline"] = roofline
            head_extras["rig_desc"] = dict(depth=rig.depth, chunk_mib=rig.chunk_mib, sync=rig.sync_name,
                                           source=rig.source_name, fp32=rig.fp32, full=rig.full, N=int(rig.N),
                                           title=f"{rig.wl.key}: {rig.wl.title}", clip=rig.clip)
            head_extras["multi"] = multi_gpu_legs(args, rig, rank, world, clk)
            if (rank == 0 and world == 1 and rig.source_name == "staged" and not args.no_overlap and not args.no_direct
                    and not rig.full and "flush" in rec):
                rec["direct_source"] = measure_direct_source(args, key, link, clk, rig.s.replica, max(50, K // 2))
        if key == "c5" and rank == 0 and world == 1 and not args.no_grid and not args.no_overlap and "flush" in rec:
            replica, flush_ref = rig.s.replica, rec["flush"]["ms"]
            barrier(world)
            rig.close()
            del rig
            torch.cuda.empty_cache()
            with clk.leg("c5.grid"):
                rec["chunk_depth_grid"] = measure_c5_grid(args, link, clk, replica, flush_ref)
            del replica
        else:
            barrier(world)      # peers' received buffers stay mapped until every rank is done with them
            rig.close()
            del rig
        records.append(rec)
        torch.cuda.empty_cache()

    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            wl = workload_of(args, args.headline)
            with clk.leg("cpu_baseline"):
                cpu = cpu_baseline(wl, args.cpu_sample or ORACLE_SAMPLE, 5, 1)
        clocks_all, clocks_legs = clk.stop()
        d = head_extras["rig_desc"]
        units = sum_over_ranks(float(d["N"]), 1, device) * world     # weak scaling: every rank owns a shard of the same size
        step_bpe = head["step_bytes_per_element"]
        value = step_bpe * units / (head["step_ms"] * 1e-3) / 1e9
        he = head["e2e"]
        worst_exposed = None
        if all("exposed_pct" in r for r in records):
            w = max(records, key=lambda r: r["exposed_pct"])
            worst_exposed = {"config": w["config"], "exposed_pct": w["exposed_pct"], "exposed_ms": w["exposed_ckpt_ms_per_iter"]}
        slowest = min(records, key=lambda r: r["step_gbs"])
        hl_clock = dict(clocks_legs.get(f"{args.headline}.step", clocks_all), sampler=clk.source)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": head["step_ms"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": d["title"] + " — the largest single-GPU configuration of BASELINE.json:configs; "
                                   "every other bandwidth-sized config is in `configs`",
                       "configs_measured": keys, "elements_per_shard": d["N"], "state_bytes": 12 * d["N"],
                       "staging_depth": d["depth"], "chunk_mib": d["chunk_mib"], "sync_mode": d["sync"],
                       "snapshot_source": d["source"], "bytes_per_element": step_bpe,
                       "bytes_per_element_note": "42 = a1 pass (2 read) + a3 (14 read + 26 written); 40 without the clip pass",
                       "precision": ("fp32 state + fp32 grads, no bf16 copy (PAPER.md:270)" if d["fp32"] else
                                     "fp32 state + bf16 grads + bf16 copy (north_star)"),
                       "decay_groups": bool(args.decay_groups),
                       "l2": "inputs larger than L2 (working set %.2f GB per step >> 126 MB)" % (step_bpe * d["N"] / 1e9),
                       "timed_region": "K x phx_step_and_snapshot (a1 clip pass, a2 sync-point wait, a3 fused AdamW + bf16 "
                                       "copy + packed snapshot); a4/a5 host flush is in e2e and overlap",
                       "host_payload": "full rank state (SURVEY 8(f4))" if d["full"] else "optimizer shard: envelope + p,m,v",
                       "parallelism": f"dp{world} independent shards, no data-path collective in the timed region",
                       "shared_gpu_debug": bool(args.debug_shared_gpu)},
            "elements_per_s": units / (head["step_ms"] * 1e-3),
            "value_min_over_configs": {"config": slowest["config"], "step_gbs": slowest["step_gbs"]},
            "exposed_ckpt_ms_per_iter": head.get("exposed_ckpt_ms_per_iter"),
            "exposed_pct_worst_config": worst_exposed,
            "roofline": head_extras["roofline"],
            "host_link": ({"bound": "host_link", "achieved": head["flush"]["gbs"], "peak": link["d2h_gbs"], "unit": "GB/s",
                           "frac": head["flush"]["frac_of_d2h_peak"], "flush_ms": head["flush"]["ms"],
                           "chunk_mib": d["chunk_mib"], "h2d_peak_gbs": link["h2d_gbs"]} if "flush" in head else None),
            "e2e": {"value": he["metric_gbs"] * world, "unit": UNIT, "h2d_bytes_per_step": he["h2d_bytes_per_step"],
                    "d2h_bytes_per_step": he["d2h_bytes_per_step"], "ms_per_step": he["ms_per_step"], "steps": he["steps"],
                    "link_gbs": he["link_gbs"],
                    "note": "H2D grads from pinned host + fused step + chunked D2H of the packed snapshot + commit, per step; "
                            "host-link bound by construction (14 N bytes must cross PCIe): ms_per_step and link_gbs are "
                            "the physical numbers, `value` restates them in the metric's unit"},
            "configs": records,
            "cpu_baseline": cpu, "gpu_launches": head_extras["launches"],
            "clocks": hl_clock, "clocks_all_legs": clocks_all, "clocks_legs": clocks_legs,
            "step_ms_min_max": [min(head_extras["per_step"]), max(head_extras["per_step"])],
        }
        line.update(head_extras["multi"])
        if world > 1:
            import torch.distributed as dist
            line["process_group"] = {"backend": dist.get_backend(), "nranks": dist.get_world_size(),
                                     "nccl_version": ".".join(map(str, torch.cuda.nccl.version())) if dist.get_backend() == "nccl" else None}
        path = write_full_record(line)
        print(compact_line(line, path), flush=True)      # the ONLY stdout line; nothing is printed after it
    barrier(world)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


# ----------------------------------------------------------------------------------------------
# the deeper measurement rows of SURVEY.md §8(d): one JSON line per measurement
# ----------------------------------------------------------------------------------------------


def emit(**kw):
    print(json.dumps(kw), flush=True)


def rig_bytes(N):
    return 256 + 12 * N


def run_overlap_curve(args):
    """Exposed checkpoint ms/iteration against the length of the compute window (R21), eager and graph-captured."""
    torch, rank, world, local_rank = gpu_setup(args)
    rig = Rig(args, args.headline, host_grads=False)
    flush_ms = rig.time_flush()
    gm = rig.gemm_setup()
    Gs = [args.gemms] if args.gemms > 0 else [64, 256, 1024, 4096, 16384]
    head = rig.gemms_for(flush_ms)
    for G in sorted(set(Gs + [head])):
        iters = rig.iters_for(G)
        o = rig.overlap(G, iters, arms=("off", "staged", "on"), reps=2)
        if not args.no_graph_step:
            og = rig.overlap_graph_step(G, iters)
            o["graph_step"] = {k: og[k] for k in ("iter_ms_off", "iter_ms_on", "exposed_ms", "exposed_frac_of_compute_step")}
        emit(mode="overlap-curve", config=args.headline, elements=int(rig.N), flush_ms=flush_ms, headline=(G == head),
             knee_gemms=flush_ms / gm, sync_mode=rig.sync_name, depth=rig.depth, chunk_mib=rig.chunk_mib, **o)
    rig.close()
    return 0


def run_timeline(args):
    """Copy/compute overlap as a timeline from CUDA events (nsys is not on the image): per iteration, when the
    GEMM window, the hot path (a1-a3) and the side-stream flush (a4+a5) of that iteration's snapshot start and end,
    all in ms since the first iteration's start.  One JSON line per iteration plus a summary."""
    torch, rank, world, local_rank = gpu_setup(args)
    rig = Rig(args, args.headline, host_grads=False)
    flush_ms = rig.time_flush()
    rig.gemm_setup()
    a, b, c = rig._gemm
    G = args.gemms if args.gemms > 0 else rig.gemms_for(flush_ms)
    iters, marks = 6, 8
    E = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731
    rows = []
    for _ in range(2):                       # warm-up iterations (not recorded)
        rig.gemm_window(G)
        rig.do_step()
        rig.flush()
    torch.cuda.synchronize()
    base = E()
    base.record(rig.cur)
    for it in range(iters):
        ev = {"gemm": [E()], "k0": E(), "k1": E(), "f0": E(), "f1": E()}
        ev["gemm"][0].record(rig.cur)
        for part in range(marks):
            rig.gemm_window(G // marks)
            e = E()
            e.record(rig.cur)
            ev["gemm"].append(e)
        ev["k0"].record(rig.cur)
        rig.do_step()                         # a2: waits (stream-side) for the commit of the previous flush
        ev["k1"].record(rig.cur)
        ev["f0"].record(rig.side)             # side stream: flush of THIS step's snapshot, runs under the next window
        rig.flush()
        ev["f1"].record(rig.side)
        rows.append(ev)
    torch.cuda.synchronize()
    rig.s.wait(rig.step)
    t = lambda e: base.elapsed_time(e)  # noqa: E731
    for it, ev in enumerate(rows):
        # the flush is enqueued behind an event of the step kernel: its real start is max(f0, k1)
        emit(mode="timeline", config=args.headline, iteration=it, gemms=G,
             gemm_window_ms=[t(ev["gemm"][0]), t(ev["gemm"][-1])],
             gemm_marks_ms=[t(e) for e in ev["gemm"]],
             hot_path_ms=[t(ev["k0"]), t(ev["k1"])],
             flush_ms=[max(t(ev["f0"]), t(ev["k1"])), t(ev["f1"])])
    under, waits = [], []
    for it in range(iters - 1):
        f0, f1 = max(t(rows[it]["f0"]), t(rows[it]["k1"])), t(rows[it]["f1"])
        g0, g1 = t(rows[it + 1]["gemm"][0]), t(rows[it + 1]["gemm"][-1])
        under.append(max(0.0, min(f1, g1) - max(f0, g0)) / (f1 - f0))
        waits.append(max(0.0, f1 - t(rows[it + 1]["k0"])))
    emit(mode="timeline-summary", config=args.headline, gemms=G, flush_alone_ms=flush_ms,
         flush_fraction_under_next_gemm_window=under, commit_after_next_step_enqueued_ms=waits,
         note="commit_after_next_step_enqueued_ms > 0 would be a stall at the single sync point (PAPER.md:226)")

    # ---- recovery timeline: fault, two-phase restore (phx_restore_async) beside the recomputed iteration ---------
    Gr = rig.gemms_for(flush_ms, 1.25, False)
    for form in ("one_phase", "two_phase"):
        rig.do_step()
        rig.flush()
        rig.s.wait(rig.step)
        torch.cuda.synchronize()
        rig.s.drop_live()
        torch.cuda.synchronize()
        r0, rp, rs, k0, k1 = E(), E(), E(), E(), E()
        gm = []
        r0.record(rig.cur)
        if form == "two_phase":
            rig.side.wait_stream(rig.cur)
            rig.step = rig.s.restore_async(rig.side)      # side stream: p -> bf16 copy -> m -> v
            rs.record(rig.side)
            rig.s.restore_wait_params(rig.cur)            # compute stream: waits for "parameters ready" only
        else:
            rig.step = rig.s.restore()
            rs.record(rig.cur)
        rp.record(rig.cur)
        for part in range(marks):
            rig.gemm_window(Gr // marks)
            e = E()
            e.record(rig.cur)
            gm.append(e)
        k0.record(rig.cur)
        rig.do_step()                                     # waits (stream-side) for the moments
        k1.record(rig.cur)
        torch.cuda.synchronize()
        tr = lambda e: r0.elapsed_time(e)  # noqa: E731
        emit(mode="timeline-recovery", config=args.headline, form=form, gemms=Gr // marks * marks,
             params_ready_ms=tr(rp), state_ready_ms=tr(rs), gemm_window_ms=[tr(rp), tr(gm[-1])],
             gemm_marks_ms=[tr(e) for e in gm], step_ms=[tr(k0), tr(k1)],
             note="ms since the fault was detected; two_phase: the moments (state_ready) arrive on the side stream "
                  "while the recomputed iteration's GEMMs run on the compute stream")
    rig.close()
    return 0


def run_sweep(args):
    """BASELINE.json:configs[4]: D2H chunk size 4..256 MiB x staging depth 1..4 (x sync mode), reporting exposed
    checkpoint ms/iteration and host-link GB/s.  Run at a TIGHT compute window (T_c = 1.25 x T_D2H, where depth and
    chunking can matter) and, on a reduced grid, at the headline window (T_c >= 4 x T_D2H)."""
    torch, rank, world, local_rank = gpu_setup(args)
    key = args.headline if args.config else "c5"
    device = torch.device(f"cuda:{local_rank}")
    link = measure_host_link(torch, device)
    probe = Rig(args, key, host_grads=False)
    replica = probe.s.replica                        # pin once, reuse for every grid point
    flush_ref = probe.time_flush()
    gm = probe.gemm_setup()
    G_tight = max(1, int(round(1.25 * flush_ref / gm)))
    G_head = probe.gemms_for(flush_ref)
    it_t, it_h = probe.iters_for(G_tight), max(5, probe.iters_for(G_head) // 2)
    base = probe.overlap(G_tight, it_t, arms=("off",))
    base_head = probe.overlap(G_head, it_h, arms=("off",))
    base_g = None if args.no_graph_step else probe.overlap_graph_step(G_tight, it_t, arms=("off",))["iter_ms_off"]
    probe.close()
    del probe
    torch.cuda.empty_cache()
    chunks = [int(x) for x in args.chunks.split(",")]
    for sync in args.syncs.split(","):
        for depth in [int(x) for x in args.depths.split(",")]:
            for chunk in chunks:
                rig = Rig(args, key, depth=depth, chunk_mib=chunk, sync=sync, replica=replica, host_grads=False)
                flush_ms = rig.time_flush()
                o = rig.overlap(G_tight, it_t, arms=("on",))
                gx = {}
                if base_g is not None:
                    og = rig.overlap_graph_step(G_tight, it_t, arms=("on",))
                    gx = dict(iter_ms_on_graph_step=og["iter_ms_on"], iter_ms_off_graph_step=base_g,
                              exposed_ms_graph_step=og["iter_ms_on"] - base_g,
                              exposed_frac_graph_step=(og["iter_ms_on"] - base_g) / base_g)
                emit(mode="sweep", window="tight(1.25xT_D2H)", config=key, elements=int(rig.N), sync_mode=sync,
                     depth=depth, chunk_mib=chunk, flush_ms=flush_ms, **gx,
                     host_link_gbs=rig_bytes(rig.N) / (flush_ms * 1e-3) / 1e9, d2h_peak_gbs=link["d2h_gbs"],
                     gemms_per_iter=G_tight, iter_ms_on=o["iter_ms_on"], iter_ms_off=base["iter_ms_off"],
                     exposed_ms=o["iter_ms_on"] - base["iter_ms_off"],
                     exposed_frac=(o["iter_ms_on"] - base["iter_ms_off"]) / base["iter_ms_off"],
                     hot_path_ms_in_loop_on=o["hot_path_ms_in_loop_on"])
                if depth in (1, 2) and chunk in (chunks[0], 64, 256):
                    o = rig.overlap(G_head, it_h, arms=("on",))
                    emit(mode="sweep", window="headline(>=4xT_D2H)", config=key, elements=int(rig.N), sync_mode=sync,
                         depth=depth, chunk_mib=chunk, flush_ms=flush_ms, gemms_per_iter=G_head,
                         iter_ms_on=o["iter_ms_on"], iter_ms_off=base_head["iter_ms_off"],
                         exposed_ms=o["iter_ms_on"] - base_head["iter_ms_off"],
                         exposed_frac=(o["iter_ms_on"] - base_head["iter_ms_off"]) / base_head["iter_ms_off"],
                         hot_path_ms_in_loop_on=o["hot_path_ms_in_loop_on"])
                rig.close()
                del rig
                torch.cuda.empty_cache()
    return 0


def run_probe(args):
    """Structure evidence for the fused kernel: the no-arithmetic streaming pass of the bench-only probe
    library for several read:write mixes, in the ONE-SHOT structure the step uses (one 8-element group per thread,
    short-lived CTAs) and in the PERSISTENT structure (148 x c CTAs with a grid stride).  One JSON line per cell."""
    torch, rank, world, local_rank = gpu_setup(args)
    from paper_2607_01646_b200 import probe as PB
    device = torch.device(f"cuda:{local_rank}")
    N = shard_elements(args, args.headline)
    plane_bytes = 4 * N
    buf = torch.empty(9 * plane_bytes, dtype=torch.uint8, device=device)
    buf.zero_()
    st = torch.cuda.current_stream(device)
    sms = torch.cuda.get_device_properties(device).multi_processor_count
    for name, (r, w) in {"step_mix_3r6w": (3, 6), "off_mix_3r3w": (3, 3), "copy_1r1w": (1, 1), "finalize_mix_2r1w": (2, 1),
                         "write_only_4w": (0, 4)}.items():
        for label, grid in [("one-shot", 0)] + [(f"persistent {c} CTAs/SM", sms * c) for c in (2, 4, 8)]:
            def go():
                if grid:
                    return PB.phx_hbm_probe_persistent_async(buf, plane_bytes, r, w, grid, st)
                return PB.phx_hbm_probe_async(buf, plane_bytes, r, w, st)
            for _ in range(3):
                assert go() == 0
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            for _ in range(20):
                go()
            e1.record(st)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / 20
            emit(mode="probe", mix=name, planes_read=r, planes_written=w, structure=label, plane_elements=int(N), ms=ms,
                 gbs=(r + w) * plane_bytes / (ms * 1e-3) / 1e9)
    return 0


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return self_spawn(args)
    if args.impl == "reference":
        return run_reference(args)
    return {"headline": run_headline, "overlap-curve": run_overlap_curve, "sweep": run_sweep,
            "timeline": run_timeline, "probe": run_probe}[args.mode](args)


if __name__ == "__main__":
    sys.exit(main())
