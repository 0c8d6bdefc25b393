#!/usr/bin/env python
"""bench.py — measures the phx hot path on B200 and prints ONE JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c2] [--impl phx|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

What is timed (config c2 = BASELINE.json:configs[1], the 1.3B-style shard, by default):
  value     fused AdamW+snapshot HBM GB/s: K back-to-back passes of a1..a3 (phx_step_and_snapshot:
            [clip,] sync-point wait, ONE fused kernel writing live state + bf16 copy + packed snapshot
            into the staging ring) with gradients already resident in HBM; 40 algorithmic bytes per
            element / device time (CUDA events on the launching stream).  Working set >> L2.
  e2e       the same metric through the same C-ABI calls with HOST buffers: every step copies the
            step's bf16 gradients from pinned host memory (H2D) and brings the step's result — the
            packed snapshot — back to the pinned host replica (a4 chunked D2H + a5 commit).
  overlap   the paper's experiment: iterations of G bf16 4096^3 GEMMs (stand-in for
            forward/backward) + the hot path, with the flush on a side stream, against the same loop
            with snapshots disabled; exposed checkpoint ms/iteration = difference of trimmed means.
  roofline  HBM roofline of the dominant (fused) kernel; host_link: the flush against the measured
            pinned-copy peak.
  cpu_baseline  the oracle as it stands on the box's host cores (rank 0, N=1), bounded sample.
`--impl reference` times the oracle instead (the reference arm of this tier).
"""
from __future__ import annotations

import argparse
import json
import os
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
BYTES_PER_ELEM = 40          # 14 read + 26 written
BYTES_PER_ELEM_OFF = 28
NOMINAL_HBM_GBS = 8000.0     # north_star "~8 TB/s"
FALLBACK_HBM_GBS = 6650.0    # /opt/skills/guides/B200_PROFILING.md, only if MEASURED_PEAKS.json is absent


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="phx", choices=["phx", "reference"])
    ap.add_argument("--config", default="c2", help="workload key (c1, c2, c3, c4a, c4b, c5)")
    ap.add_argument("--variant", type=int, default=0, help="fused-kernel variant (tuning)")
    ap.add_argument("--depth", type=int, default=2)
    ap.add_argument("--chunk-mib", type=int, default=64)
    ap.add_argument("--sync", default="strict", choices=["strict", "relaxed"])
    ap.add_argument("--gemms", type=int, default=0, help="GEMMs per overlapped iteration (0 = auto: T_c >= 4 T_D2H)")
    ap.add_argument("--overlap-iters", type=int, default=20)
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--no-overlap", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample", type=int, default=0, help="elements of the shard the oracle is timed on (0 = auto)")
    return ap.parse_args()


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


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(",") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for k, nme in enumerate(names):
                    if r[3 + k].strip().lower().startswith("active"):
                        reasons.add(nme)
            except Exception:
                continue
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


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


def max_over_ranks(x: float, world, device) -> float:
    """The slowest rank defines the step time (max over ranks)."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, world, device) -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


# ----------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the oracle on the host cores
# ----------------------------------------------------------------------------------------------


def time_oracle(wl, sample, steps, warmup, nthreads):
    """Oracle AdamW step (phx_oracle.c, as it stands) on the first `sample` elements of the shard."""
    import numpy as np
    import torch
    from oracle import oracle as O
    from paper_2607_01646_b200 import workloads as W
    d = O.define_shard(wl.layout(), wl.dp_size, wl.dp_rank, (wl.tp_size, wl.tp_rank), (wl.pp_size, wl.pp_rank))
    n = min(sample, d["n_padded"])
    segs = []
    for tid, _, off, ln in d["segments"]:
        if off < n:
            segs.append((tid, off, min(ln, n - off)))
    p = W.init_params(n, n, wl.seed).numpy()
    m = np.zeros(n, np.float32)
    v = np.zeros(n, np.float32)
    p16 = np.zeros(n, np.uint16)
    g = W.gen_grads(wl, segs, n, 1, wl.seed).view(torch.int16).numpy().view(np.uint16)
    h = wl.hyper
    times = []
    for t in range(1, warmup + steps + 1):
        coef = 1.0
        t0 = time.perf_counter()
        if h.max_grad_norm > 0:
            coef = float(O.clip_coef(O.sumsq(g), h.max_grad_norm))
        O.adamw_step(p, m, v, g, p16, h.lr, h.beta1, h.beta2, h.eps, h.wd, t, coef, nthreads)
        dt = time.perf_counter() - t0
        if t > warmup:
            times.append(dt)
    return n, times


def run_reference(args):
    rank, world, _ = rank_env()
    if rank != 0:
        return 0
    from paper_2607_01646_b200 import workloads as W
    wl = W.CONFIGS[args.config]
    cores = len(os.sched_getaffinity(0))
    sample = args.cpu_sample or (1 << 24)
    n, times = time_oracle(wl, sample, args.steps, args.warmup, cores)
    ms = 1e3 * sum(times) / len(times)
    value = BYTES_PER_ELEM * n / (ms * 1e-3) / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{wl.key}: {wl.title}", "sample_elements": n,
                   "note": "oracle/phx_oracle.c AdamW step (+clip) on the first sample_elements of the shard, OpenMP over all host cores"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"first {n} of {wl.n_expected} elements, {args.steps} steps",
                         "elements_per_s": n / (ms * 1e-3)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------------------------
# phx arm
# ----------------------------------------------------------------------------------------------


def measure_host_link(torch, device, nbytes=1 << 30, reps=5):
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


def run_phx(args):
    import torch
    rank, world, local_rank = rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl phx needs a B200: there is no CPU fallback")
    device = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(device)
    dist_init(world, True)

    from paper_2607_01646_b200 import binding as B
    from paper_2607_01646_b200 import workloads as W
    from paper_2607_01646_b200.shard import Shard
    import dataclasses

    base = W.CONFIGS[args.config]
    # weak scaling: every rank owns one DP shard of the same model (its own dp_rank), no data-path collective
    wl = dataclasses.replace(base, dp_rank=rank % base.dp_size)
    sync = B.PHX_SYNC_STRICT if args.sync == "strict" else B.PHX_SYNC_RELAXED
    chunk = args.chunk_mib << 20
    K, Wm = args.steps, max(args.warmup, 3)

    s = Shard(wl, device=device, staging_depth=args.depth, sync_mode=sync, chunk_bytes=chunk)
    B.phx_set_kernel_variant(s.h, args.variant)
    N = s.n_padded
    s.p.copy_(W.init_params(s.n, N, wl.seed, device=device))
    s.set_state(0)
    grads = [W.gen_grads(wl, s.segments, N, t, wl.seed, device=device) for t in (1, 2)]
    hgrads = [g.cpu().pin_memory() for g in grads]       # e2e: the step's inputs live in pinned host memory
    torch.cuda.synchronize()
    cur = torch.cuda.current_stream(device)
    side = torch.cuda.Stream(device=device)
    step = 0

    link = measure_host_link(torch, device) if rank == 0 else {}

    # ---- value: K back-to-back a1..a3 passes, inputs resident in HBM ---------------------------------
    for _ in range(Wm):
        step += 1
        s.step_and_snapshot(grads[step & 1], step)
    torch.cuda.synchronize()
    barrier(world)
    clocks = ClockSampler(local_rank) if rank == 0 else None
    l0 = B.phx_kernel_launches(s.h)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    ev[0].record(cur)
    for k in range(K):
        step += 1
        s.step_and_snapshot(grads[step & 1], step)
        ev[k + 1].record(cur)
    torch.cuda.synchronize()
    barrier(world)
    launches = B.phx_kernel_launches(s.h) - l0
    total_ms = ev[0].elapsed_time(ev[K])
    clk = clocks.stop() if clocks else None
    per = [ev[k].elapsed_time(ev[k + 1]) for k in range(K)]
    total_ms = max_over_ranks(total_ms, world, device)
    ms_per_step = total_ms / K
    units = sum_over_ranks(float(N), world, device)            # elements all ranks processed per step
    value = BYTES_PER_ELEM * units / (ms_per_step * 1e-3) / 1e9

    # dominant kernel alone (differs from the step only when the clip kernels run): a handle with
    # clipping off bound to the same memory
    kern_ms = ms_per_step
    if wl.hyper.max_grad_norm > 0:
        cfg0 = dataclasses.replace(wl, hyper=dataclasses.replace(wl.hyper, max_grad_norm=0.0))
        h0 = B.phx_shard_create(cfg0.layout(), cfg0.dp_size, cfg0.dp_rank, tp=(cfg0.tp_size, cfg0.tp_rank),
                                pp=(cfg0.pp_size, cfg0.pp_rank), staging_depth=args.depth, sync_mode=sync,
                                chunk_bytes=chunk)
        B.phx_shard_bind(h0, s.p, s.m, s.v, s.p16, s.staging, s.replica)
        B.phx_shard_set_state(h0, 0, cur)
        hp = wl.hyper
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for k in range(3):
            B.phx_step_and_snapshot(h0, grads[k & 1], hp.lr, hp.beta1, hp.beta2, hp.eps, hp.wd, k + 1, cur)
        e0.record(cur)
        for k in range(3, 3 + K):
            B.phx_step_and_snapshot(h0, grads[k & 1], hp.lr, hp.beta1, hp.beta2, hp.eps, hp.wd, k + 1, cur)
        e1.record(cur)
        torch.cuda.synchronize()
        kern_ms = e0.elapsed_time(e1) / K
        B.phx_shard_destroy(h0)
    peak, peak_src = measured_peaks()
    achieved = BYTES_PER_ELEM * N / (kern_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": committed_traffic(args.config), "peak_source": peak_src,
                "frac_of_nominal_8TBps": achieved / NOMINAL_HBM_GBS, "kernel": "phx::k_step8<1,1,true>",
                "kernel_ms": kern_ms, "algorithmic_bytes_per_launch": BYTES_PER_ELEM * N}

    # ---- e2e: host buffers in, host replica out, through the same C-ABI calls ------------------------
    Ke = args.e2e_steps
    def e2e_loop(k_steps):
        nonlocal step
        for _ in range(k_steps):
            step += 1
            g = grads[step & 1]
            g.copy_(hgrads[step & 1], non_blocking=True)          # H2D of this step's inputs
            s.step_and_snapshot(g, step)
            s.flush_async(side)                                   # D2H of this step's result (a4 + a5)
        s.wait(step)
    e2e_loop(2)
    torch.cuda.synchronize()
    barrier(world)
    t0 = time.perf_counter()
    e2e_loop(Ke)
    torch.cuda.synchronize()
    barrier(world)
    e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3 / Ke, world, device)
    e2e_val = BYTES_PER_ELEM * units / (e2e_ms * 1e-3) / 1e9
    d2h_bytes = int(s.info.snapshot_bytes)
    e2e = {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(2 * N), "d2h_bytes_per_step": d2h_bytes,
           "ms_per_step": e2e_ms, "steps": Ke,
           "note": "H2D grads from pinned host + fused step + chunked D2H of the packed snapshot + commit, per step"}

    # flush alone (a4+a5) against the measured pinned-copy peak
    host_link = None
    if rank == 0:
        step += 1
        s.step_and_snapshot(grads[step & 1], step)
        torch.cuda.synchronize()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record(side)
        s.flush_async(side)
        f1.record(side)
        s.wait(step)
        torch.cuda.synchronize()
        flush_ms = f0.elapsed_time(f1)
        ach = d2h_bytes / (flush_ms * 1e-3) / 1e9
        host_link = {"bound": "host_link", "achieved": ach, "peak": link["d2h_gbs"], "unit": "GB/s",
                     "frac": ach / link["d2h_gbs"], "flush_ms": flush_ms, "chunk_mib": args.chunk_mib,
                     "h2d_peak_gbs": link["h2d_gbs"]}

    # ---- overlap: exposed checkpoint ms/iteration (PAPER.md:283 protocol) -----------------------------
    overlap = None
    if not args.no_overlap and rank == 0:
        overlap = measure_overlap(torch, B, W, Shard, s, wl, grads, args, device, side, step,
                                  host_link["flush_ms"])
        step = overlap.pop("_step")

    # ---- restore + recompute (a6, a7) -------------------------------------------------------------------
    restore = None
    if rank == 0:
        torch.cuda.synchronize()          # every flush issued so far has been waited for above
        s.drop_live()
        torch.cuda.synchronize()
        r0, r1, r2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        r0.record(cur)
        back = s.restore()
        r1.record(cur)
        s.step_and_snapshot(grads[(back + 1) & 1], back + 1)
        r2.record(cur)
        torch.cuda.synchronize()
        rms = r0.elapsed_time(r1)
        restore = {"restore_ms": rms, "recompute_ms": r1.elapsed_time(r2), "mode": "bulk_kernel",
                   "host_link_gbs": 12 * N / (rms * 1e-3) / 1e9,
                   "frac_of_h2d_peak": 12 * N / (rms * 1e-3) / 1e9 / link["h2d_gbs"]}

    # ---- cpu baseline: the oracle on the host cores (rank 0, N == 1 only) ------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = len(os.sched_getaffinity(0))
        sample = args.cpu_sample or min(N, 1 << 28)
        n_s, times = time_oracle(wl, sample, 3, 1, cores)
        t = sum(times) / len(times)
        n_1, times1 = time_oracle(wl, min(sample, 1 << 25), 2, 1, 1)
        t1 = sum(times1) / len(times1)
        cpu = {"value": BYTES_PER_ELEM * n_s / t / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {n_s} of {N} elements of the shard, 3 steps after 1 warm-up",
               "elements_per_s": n_s / t, "single_thread_elements_per_s": n_1 / t1}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{wl.key}: {wl.title}", "elements_per_shard": int(N),
                       "state_bytes": int(12 * N), "staging_depth": args.depth, "chunk_mib": args.chunk_mib,
                       "sync_mode": args.sync, "kernel_variant": args.variant,
                       "l2": "inputs larger than L2 (working set %.2f GB per step >> 126 MB)" % (BYTES_PER_ELEM * N / 1e9),
                       "timed_region": "K x phx_step_and_snapshot (a1 clip if configured, a2 sync-point wait, a3 fused "
                                       "AdamW+bf16 copy+packed snapshot); a4/a5 host flush is in e2e and overlap",
                       "parallelism": f"dp{world} independent shards, no data-path collective"},
            "elements_per_s": units / (ms_per_step * 1e-3),
            "exposed_ckpt_ms_per_iter": overlap["exposed_ms"] if overlap else None,
            "roofline": roofline, "host_link": host_link, "e2e": e2e, "overlap": overlap, "restore": restore,
            "cpu_baseline": cpu, "gpu_launches": int(launches), "clocks": clk,
            "step_ms_min_max": [min(per), max(per)],
        }
        print(json.dumps(line), flush=True)
    s.close()
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


def measure_overlap(torch, B, W, Shard, s_on, wl, grads, args, device, side, step, flush_ms):
    """Iterations of G GEMMs + hot path (snapshot on, flush on the side stream) versus the same
    loop with the snapshot-off kernel and no flush; per-iteration times from CUDA events on the
    compute stream; trimmed means per PAPER.md:283."""
    cur = torch.cuda.current_stream(device)
    a = torch.randn(4096, 4096, device=device, dtype=torch.bfloat16)
    b = torch.randn(4096, 4096, device=device, dtype=torch.bfloat16)
    c = torch.empty(4096, 4096, device=device, dtype=torch.bfloat16)
    for _ in range(20):
        torch.matmul(a, b, out=c)
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record(cur)
    for _ in range(200):
        torch.matmul(a, b, out=c)
    g1.record(cur)
    torch.cuda.synchronize()
    gemm_ms = g0.elapsed_time(g1) / 200
    G = args.gemms
    if G <= 0:
        G = 64
        while G * gemm_ms < 4.0 * flush_ms:      # headline rule: smallest power of two with T_c >= 4 T_D2H
            G *= 2
    iters, warm = args.overlap_iters, 3

    s_off = Shard(wl, device=device, snapshot=False)
    s_off.p.copy_(s_on.p)
    s_off.set_state(0)

    def loop(shard, flush, first_step):
        st = first_step
        evs = []
        kevs = []
        for it in range(warm + iters):
            e0 = torch.cuda.Event(enable_timing=True)
            e0.record(cur)
            for _ in range(G):
                torch.matmul(a, b, out=c)
            k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            k0.record(cur)
            st += 1
            shard.step_and_snapshot(grads[st & 1], st)
            k1.record(cur)
            if flush:
                shard.flush_async(side)
            evs.append(e0)
            kevs.append((k0, k1))
        end = torch.cuda.Event(enable_timing=True)
        end.record(cur)
        torch.cuda.synchronize()
        evs.append(end)
        it_ms = [evs[i].elapsed_time(evs[i + 1]) for i in range(warm, warm + iters)]
        k_ms = [x.elapsed_time(y) for x, y in kevs[warm:]]
        return st, it_ms, k_ms

    # interleave on/off/on/off halves to average out slow clock drift
    step, on1, kon1 = loop(s_on, True, step)
    _, off1, koff1 = loop(s_off, False, 0)
    s_on.wait(step)
    on, off, kon, koff = on1, off1, kon1, koff1
    t_on, t_off = trimmed_mean(on), trimmed_mean(off)
    out = {
        "gemms_per_iter": G, "gemm_ms": gemm_ms, "compute_window_ms": G * gemm_ms, "iters": iters,
        "iter_ms_snapshot_on": t_on, "iter_ms_snapshot_off": t_off, "exposed_ms": t_on - t_off,
        "exposed_frac_of_compute_step": (t_on - t_off) / t_off,
        "hot_path_ms_in_loop_on": trimmed_mean(kon), "hot_path_ms_in_loop_off": trimmed_mean(koff),
        "flush_ms": flush_ms, "protocol": "PAPER.md:283: warm-up dropped, slowest 5% dropped, mean of the rest",
        "_step": step,
    }
    s_off.close()
    return out


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_phx(args)


if __name__ == "__main__":
    sys.exit(main())
