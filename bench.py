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
    ap.add_argument("--chunk-mib", type=int, default=8)
    ap.add_argument("--sync", default="strict", choices=["strict", "relaxed"])
    ap.add_argument("--gemms", type=int, default=0, help="GEMMs per overlapped iteration (0 = auto: T_c >= 4 T_D2H)")
    ap.add_argument("--overlap-iters", type=int, default=20)
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--no-overlap", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-mix-ceiling", action="store_true", help="skip the no-arithmetic HBM mix-ceiling probe")
    ap.add_argument("--cpu-sample", type=int, default=0, help="elements of the shard the oracle is timed on (0 = auto)")
    ap.add_argument("--mode", default="headline",
                    choices=["headline", "configs", "overlap-curve", "sweep", "hotswap", "timeline"],
                    help="headline: the ONE contract line (default).  The others print one JSON line per "
                         "measurement: configs = every config's kernel/flush/restore; overlap-curve = exposed ms vs G; "
                         "sweep = chunk x depth x sync-mode grid (BASELINE.json:configs[4]); hotswap = configs[3]")
    ap.add_argument("--overlap-reps", type=int, default=2, help="ABAB alternations of the overlap arms")
    ap.add_argument("--source", default="staged", choices=["staged", "direct"],
                    help="snapshot source: staged = fused kernel also writes the staging slot (40 B/elem, north_star); "
                         "direct = flush DMAs the live planes under the strict sync point (28 B/elem)")
    ap.add_argument("--restore-mode", default="copy", choices=["bulk", "copy"])
    ap.add_argument("--peers", type=int, default=-1,
                    help="k ring peers the snapshot is also replicated to over NVLink (SURVEY 8(f1)); -1 = auto: 1 when "
                         "--gpus > 1 (real P2P ring over CUDA IPC), 0 at one GPU; k > 0 at one GPU measures a loopback "
                         "stand-in (received buffer on the same device)")
    ap.add_argument("--publish", default="none", choices=["none", "fused", "copy"],
                    help="SURVEY 8(f3): also publish the model-param copy into the other DP ranks' parameter buffers — "
                         "fused = P2P stores from the step kernel, copy = copy engine after it.  N > 1: real buffers over "
                         "CUDA IPC; N = 1: loopback stand-in with dp_size-1 buffers on the same GPU")
    ap.add_argument("--precision", default="bf16", choices=["bf16", "fp32"],
                    help="bf16 = fp32 state + bf16 grads + bf16 copy (north_star, default); fp32 = the paper's own "
                         "all-FP32 setting (PAPER.md:270; SURVEY 8(f2)): fp32 grads, no bf16 copy, 16 B read + 24 B written")
    ap.add_argument("--decay-groups", action="store_true",
                    help="flag biases and norm weights no-decay (per-tensor AdamW parameter groups, SURVEY 8(f2))")
    ap.add_argument("--window", default="eager", choices=["eager", "graph"],
                    help="how the stand-in GEMM window of the overlap runs is launched: eager torch.matmul calls "
                         "(default) or replays of a CUDA graph of 64 GEMMs")
    ap.add_argument("--no-graph-arm", action="store_true", help="skip the CUDA-graph repeat of the overlap run")
    ap.add_argument("--payload", default="optimizer", choices=["optimizer", "full"],
                    help="what the local host slots hold: optimizer = p,m,v + envelope (the H2H payload, default); "
                         "full = SURVEY 8(f4), the paper's D2H payload (PAPER.md:145): p,m,v + the rank's whole "
                         "model-parameter buffer W + envelope, for in-place recovery")
    ap.add_argument("--clip-scope", default="local", choices=["local", "global"],
                    help="configs with a clip (c3): local = the shard's own norm (a1 inside the step); global = "
                         "SURVEY 8(e): per-rank sum of squares, all-gather of one double per rank (NCCL when "
                         "--gpus > 1), coefficient from the D sums inside the step")
    ap.add_argument("--chunks", default="4,8,16,32,64,128,256", help="chunk sizes (MiB) of --mode sweep")
    ap.add_argument("--depths", default="1,2,3,4", help="staging depths of --mode sweep")
    ap.add_argument("--syncs", default="strict,relaxed", help="sync modes of --mode sweep")
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


def workload_of(args, key):
    """BASELINE.json config `key`, in the precision / decay-group variant the flags ask for."""
    import dataclasses
    from paper_2607_01646_b200 import workloads as W
    return dataclasses.replace(W.CONFIGS[key], precision=args.precision, decay_groups=bool(args.decay_groups))


def time_oracle(wl, sample, steps, warmup, nthreads):
    """Oracle AdamW step (phx_oracle.c, as it stands) on the first `sample` elements of the shard."""
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
    times = []
    for t in range(1, warmup + steps + 1):
        coef = 1.0
        t0 = time.perf_counter()
        if h.max_grad_norm > 0:
            coef = float(O.clip_coef(O.sumsq(g), h.max_grad_norm))
        if fp32 or mask is not None:
            O.adamw_step_ex(p, m, v, g, None if fp32 else p16, mask, h.lr, h.beta1, h.beta2, h.eps, h.wd, t, coef, nthreads)
        else:
            O.adamw_step(p, m, v, g, p16, h.lr, h.beta1, h.beta2, h.eps, h.wd, t, coef, nthreads)
        dt = time.perf_counter() - t0
        if t > warmup:
            times.append(dt)
    return n, times


def run_reference(args):
    rank, world, _ = rank_env()
    if rank != 0:
        return 0
    wl = workload_of(args, args.config)
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


class Rig:
    """One shard on one GPU plus everything the measurements need around it: gradients resident in HBM
    and in pinned host memory, a flush stream, the GEMM operands of the stand-in compute window."""

    def __init__(self, args, key, rank=0, world=1, local_rank=0, depth=None, chunk_mib=None, sync=None,
                 replica=None, host_grads=True, restore_mode=None, source=None):
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
        sync_mode = B.PHX_SYNC_STRICT if self.sync_name == "strict" else B.PHX_SYNC_RELAXED
        self.source_name = source or args.source
        self.source = B.PHX_SNAPSHOT_DIRECT if self.source_name == "direct" else B.PHX_SNAPSHOT_STAGED
        self.bytes_per_elem = BYTES_PER_ELEM_OFF if self.source_name == "direct" else BYTES_PER_ELEM
        if restore_mode is None:
            restore_mode = B.PHX_RESTORE_COPY_ENGINE if args.restore_mode == "copy" else B.PHX_RESTORE_BULK_KERNEL
        self.restore_mode_name = "copy_engine" if restore_mode == B.PHX_RESTORE_COPY_ENGINE else "bulk_kernel"
        self.full = getattr(args, "payload", "optimizer") == "full"
        self.s = Shard(self.wl, device=self.device, staging_depth=self.depth, sync_mode=sync_mode,
                       chunk_bytes=self.chunk_mib << 20, replica=replica, restore_mode=restore_mode,
                       snapshot_source=self.source,
                       payload=B.PHX_PAYLOAD_FULL_RANK_STATE if self.full else B.PHX_PAYLOAD_OPTIMIZER)
        B.phx_set_kernel_variant(self.s.h, args.variant)
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
        self.gemm_ms = None
        self.k_peers = 0
        self.peers_in_overlap = False
        self.gclip = None
        if getattr(args, "clip_scope", "local") == "global" and self.wl.hyper.max_grad_norm > 0:
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
            return "NVLink/NVSwitch P2P into the ring successors' HBM, received buffers mapped over CUDA IPC"
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

    def precision_code(self):
        return self.B.PHX_PRECISION_FP32 if self.fp32 else self.B.PHX_PRECISION_BF16_GRADS

    def kernel_name(self):
        mode = (1 if self.fp32 else 0) | (2 if any(self.wl.flags()) else 0)
        return "phx::k_step8<1,1,%s,%d>" % ("true" if self.source_name == "staged" else "false", mode)

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
        for k in range(K):
            self.do_step()
            ev[k + 1].record(self.cur)
        torch.cuda.synchronize()
        per = [ev[k].elapsed_time(ev[k + 1]) for k in range(K)]
        return ev[0].elapsed_time(ev[K]), per, B.phx_kernel_launches(self.s.h) - l0

    def time_fused_kernel_alone(self, K):
        """The dominant kernel without the clip kernels: a second handle with clipping off bound to the same memory."""
        torch, B, wl = self.torch, self.B, self.wl
        h0 = B.phx_shard_create(wl.layout(), wl.dp_size, wl.dp_rank, tp=(wl.tp_size, wl.tp_rank),
                                pp=(wl.pp_size, wl.pp_rank), staging_depth=self.depth, max_grad_norm=0.0,
                                snapshot_source=self.source, flags=wl.flags(), precision=self.precision_code())
        B.phx_shard_bind(h0, self.s.p, self.s.m, self.s.v, self.s.p16, self.s.staging, self.s.replica)
        B.phx_shard_set_state(h0, 0, self.cur)
        B.phx_set_kernel_variant(h0, self.args.variant)
        hp = wl.hyper
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for k in range(3 + K):
            if k == 3:
                e0.record(self.cur)
            B.phx_step_and_snapshot(h0, self.grads[k & 1], hp.lr, hp.beta1, hp.beta2, hp.eps, hp.wd, k + 1, self.cur)
        e1.record(self.cur)
        torch.cuda.synchronize()
        B.phx_shard_destroy(h0)
        return e0.elapsed_time(e1) / K

    def off_shard(self):
        """Snapshot-disabled handle (the paper's 'mechanism disabled' baseline) bound to the same live arrays."""
        if self.s_off is None:
            B, wl = self.B, self.wl
            h = B.phx_shard_create(wl.layout(), wl.dp_size, wl.dp_rank, tp=(wl.tp_size, wl.tp_rank),
                                   pp=(wl.pp_size, wl.pp_rank), snapshot_disabled=True,
                                   max_grad_norm=wl.hyper.max_grad_norm, flags=wl.flags(),
                                   precision=self.precision_code())
            B.phx_shard_bind(h, self.s.p, self.s.m, self.s.v, self.s.p16, None, None)
            B.phx_shard_set_state(h, 0, self.cur)
            B.phx_set_kernel_variant(h, self.args.variant)
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

    def gemm_window(self, G, mode=None):
        """The stand-in compute window: G GEMMs, launched eagerly (default) or — `--window graph` — as replays of
        one CUDA graph of 64 GEMMs (plus an eager remainder), the launch form a B200 training step would use."""
        torch = self.torch
        a, b, c = self._gemm
        if (mode or getattr(self.args, "window", "eager")) != "graph":
            for _ in range(G):
                torch.matmul(a, b, out=c)
            return
        if getattr(self, "_graph", None) is None:
            s = torch.cuda.Stream(device=self.device)
            s.wait_stream(self.cur)
            with torch.cuda.stream(s):
                for _ in range(3):
                    torch.matmul(a, b, out=c)
            self.cur.wait_stream(s)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                for _ in range(64):
                    torch.matmul(a, b, out=c)
            self._graph = g
        for _ in range(G // 64):
            self._graph.replay()
        for _ in range(G % 64):
            torch.matmul(a, b, out=c)

    def headline_gemms(self, flush_ms, factor=4.0):
        """R21: smallest power of two G with T_c >= factor x T_D2H."""
        gm = self.gemm_setup()
        G = 64
        while G * gm < factor * flush_ms:
            G *= 2
        return G

    def overlap(self, G, iters, reps, arms=("off", "staged", "on"), warm=2, window=None):
        """Iterations of G GEMMs + the hot path, three arms alternated `reps` times (ABCABC) to average
        out clock drift:
          off    — snapshot-disabled kernel, no flush (the paper's baseline run);
          staged — snapshot-on kernel (writes the staging slot), no flush;
          on     — snapshot-on kernel + flush on the side stream (PHOENIX enabled).
        Per-iteration times from CUDA events on the compute stream; PAPER.md:283 trimming."""
        torch = self.torch
        self.gemm_setup()
        a, b, c = self._gemm
        it_ms = {k: [] for k in arms}
        hp_ms = {k: [] for k in arms}
        for _ in range(reps):
            for arm in arms:
                evs, kevs = [], []
                for it in range(warm + iters):
                    e0 = torch.cuda.Event(enable_timing=True)
                    e0.record(self.cur)
                    self.gemm_window(G, window)
                    k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    k0.record(self.cur)
                    if arm == "off":
                        self.do_step_off()
                    else:
                        self.do_step()
                    k1.record(self.cur)
                    if arm == "on":
                        self.flush()
                        if getattr(self, "k_peers", 0) and self.peers_in_overlap:
                            self.B.phx_snapshot_flush_peers_async(self.s.h, self.peer_stream)
                    evs.append(e0)
                    kevs.append((k0, k1))
                end = torch.cuda.Event(enable_timing=True)
                end.record(self.cur)
                torch.cuda.synchronize()
                if arm == "on":
                    self.s.wait(self.step)
                    if getattr(self, "k_peers", 0) and self.peers_in_overlap:
                        self.B.phx_snapshot_wait_peers(self.s.h, self.step)
                evs.append(end)
                it_ms[arm] += [evs[i].elapsed_time(evs[i + 1]) for i in range(warm, warm + iters)]
                hp_ms[arm] += [x.elapsed_time(y) for x, y in kevs[warm:]]
        t = {k: trimmed_mean(v) for k, v in it_ms.items()}
        out = {"gemms_per_iter": G, "gemm_ms": self.gemm_ms, "compute_window_ms": G * self.gemm_ms,
               "window_launch": window or getattr(self.args, "window", "eager"),
               "iters_per_arm": iters * reps, "reps": reps,
               "protocol": "PAPER.md:283: warm-up dropped, slowest 5% dropped, mean of the rest; arms alternated"}
        for k in arms:
            out[f"iter_ms_{k}"] = t[k]
            out[f"hot_path_ms_in_loop_{k}"] = trimmed_mean(hp_ms[k])
        if "on" in t and "off" in t:
            out["exposed_ms"] = t["on"] - t["off"]
            out["exposed_frac_of_compute_step"] = (t["on"] - t["off"]) / t["off"]
        if "staged" in t and "off" in t:
            out["exposed_ms_kernel_only"] = t["staged"] - t["off"]
        return out

    def close(self):
        self.close_peers()
        if self.s_off is not None:
            self.B.phx_shard_destroy(self.s_off)
            self.s_off = None
        self.s.close()


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


def measure_hbm_mix_ceiling(torch, B, device, plane_elems, reps=20):
    """No-arithmetic streaming passes with the fused kernel's access pattern (phx_hbm_probe_async): the HBM
    ceiling for a read:write mix.  Returns GB/s per mix; planes of `plane_elems` fp32 each (larger than L2)."""
    mixes = {"read_only_4r": (4, 0), "write_only_4w": (0, 4), "copy_1r1w": (1, 1), "step_mix_3r6w": (3, 6),
             "off_mix_3r3w": (3, 3)}
    plane_bytes = int(plane_elems) * 4
    buf = torch.empty(9 * plane_bytes, dtype=torch.uint8, device=device)
    buf.zero_()
    st = torch.cuda.current_stream(device)
    out = {}
    for name, (r, w) in mixes.items():
        for _ in range(3):
            B.phx_hbm_probe_async(buf, plane_bytes, r, w, st)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for _ in range(reps):
            B.phx_hbm_probe_async(buf, plane_bytes, r, w, st)
        e1.record(st)
        torch.cuda.synchronize()
        out[name] = (r + w) * plane_bytes / (e0.elapsed_time(e1) / reps * 1e-3) / 1e9
    del buf
    return out


def gpu_setup():
    import torch
    rank, world, local_rank = rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl phx needs a B200: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist_init(world, True)
    return torch, rank, world, local_rank


def run_headline(args):
    torch, rank, world, local_rank = gpu_setup()
    rig = Rig(args, args.config, rank, world, local_rank)
    device, N, wl, B = rig.device, rig.N, rig.wl, rig.B
    K, Wm = args.steps, max(args.warmup, 3)
    link = measure_host_link(torch, device) if rank == 0 else {}

    # ---- value: K back-to-back a1..a3 passes, inputs resident in HBM ---------------------------------
    for _ in range(Wm):
        rig.do_step()
    torch.cuda.synchronize()
    barrier(world)
    clocks = ClockSampler(local_rank) if rank == 0 else None
    total_ms, per, launches = rig.time_steps(K, 0)
    barrier(world)
    clk = clocks.stop() if clocks else None
    total_ms = max_over_ranks(total_ms, world, device)
    ms_per_step = total_ms / K
    units = sum_over_ranks(float(N), world, device)            # elements all ranks processed per step
    BPE = rig.bytes_per_elem                                   # 40 staged (north_star), 28 direct
    value = BPE * units / (ms_per_step * 1e-3) / 1e9

    kern_ms = rig.time_fused_kernel_alone(K) if wl.hyper.max_grad_norm > 0 else ms_per_step
    off_ms = rig.time_steps_off(min(K, 50))
    peak, peak_src = measured_peaks()
    achieved = BPE * N / (kern_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": committed_traffic(args.config + ("" if rig.source_name == "staged" else "-direct")
                                             + ("-fp32" if rig.fp32 else "") + ("-groups" if args.decay_groups else "")),
                "peak_source": peak_src, "frac_of_nominal_8TBps": achieved / NOMINAL_HBM_GBS,
                "kernel": rig.kernel_name(),
                "kernel_ms": kern_ms, "algorithmic_bytes_per_launch": BPE * N, "bytes_per_element": BPE,
                "snapshot_off_step_ms": off_ms,
                "snapshot_off_gbs": BYTES_PER_ELEM_OFF * N / (off_ms * 1e-3) / 1e9}
    if rank == 0 and not args.no_mix_ceiling:
        # context, not the denominator: what a kernel with NO arithmetic reaches with this read:write mix
        ceil = measure_hbm_mix_ceiling(torch, rig.B, device, N)
        roofline["mix_ceiling_gbs"] = ceil
        roofline["frac_of_mix_ceiling"] = achieved / ceil["off_mix_3r3w" if rig.source_name == "direct" else "step_mix_3r6w"]

    # ---- e2e -----------------------------------------------------------------------------------------
    e2e_ms = max_over_ranks(rig.e2e(args.e2e_steps, world), world, device)
    d2h_bytes = int(rig.s.info.host_snapshot_bytes)          # = snapshot_bytes unless --payload full
    e2e = {"value": BPE * units / (e2e_ms * 1e-3) / 1e9, "unit": UNIT,
           "h2d_bytes_per_step": int(rig.grad_bytes * N), "d2h_bytes_per_step": d2h_bytes, "ms_per_step": e2e_ms,
           "steps": args.e2e_steps,
           "note": "H2D grads from pinned host + fused step + chunked D2H of the packed snapshot + commit, per step"}

    # ---- §8(f1): ring peers (real NVLink ring at N > 1; opt-in loopback stand-in at N = 1) -------------
    k_peers = args.peers if args.peers >= 0 else (1 if world > 1 else 0)
    k_peers = min(k_peers, max(world - 1, 0)) if world > 1 else k_peers
    peer = None
    if k_peers > 0:
        try:
            peer = {"k": k_peers, "link": rig.setup_peers(k_peers, rank, world)}
            rig.peers_in_overlap = world > 1      # the loopback copy is not NVLink traffic: keep it out of the overlap arm
        except Exception as e:  # noqa: BLE001  (PeerRing makes every rank fail together)
            peer = {"k": k_peers, "error": str(e)[:300]}
            rig.k_peers = 0
    if peer and "error" not in peer:
        pf_ms = max_over_ranks(rig.time_peer_flush(), world, device)
        pbytes = k_peers * int(rig.s.info.snapshot_bytes)
        peer.update(flush_ms=pf_ms, bytes_per_step=pbytes, gbs_per_gpu=pbytes / (pf_ms * 1e-3) / 1e9,
                    note="replication of one packed snapshot to all k peers, copy engine, alone; max over ranks, "
                         "all ranks sending at once")

    # ---- §8(f3): parameter publication (opt-in) --------------------------------------------------------
    publication = None
    if args.publish != "none":
        from paper_2607_01646_b200 import ring as PR
        pmode = B.PHX_PUBLISH_FUSED if args.publish == "fused" else B.PHX_PUBLISH_COPY_ENGINE
        pub_stream = torch.cuda.Stream(device=device)
        try:
            if world > 1:
                pg, npeers = PR.ParamGroup(rig.s, pmode, ring_size=world, ring_rank=rank), world
                plink = "NVLink/NVSwitch P2P into every rank's parameter buffer (CUDA IPC), own buffer included"
            else:
                npeers = min(wl.dp_size - 1, B.PHX_MAX_PARAM_PEERS)
                lbufs = [torch.zeros(wl.dp_size * N, dtype=torch.float32 if rig.fp32 else torch.bfloat16, device=device)
                         for _ in range(npeers)]
                B.phx_shard_bind_param_peers(rig.s.h, lbufs, pmode)
                pg = None
                plink = "loopback stand-in: dp_size-1 parameter buffers on the SAME GPU (HBM writes, not NVLink)"
            for _ in range(3):
                rig.do_step()
            torch.cuda.synchronize()
            barrier(world)
            q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
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
            publication = {"mode": args.publish, "buffers_written": npeers, "link": plink, "step_plus_publish_ms": pms,
                           "bytes_published_per_step": int(npeers * N * (4 if rig.fp32 else 2))}
            B.phx_shard_bind_param_peers(rig.s.h, [])
            if pg is not None:
                pg.close()
        except Exception as e:  # noqa: BLE001
            publication = {"mode": args.publish, "error": str(e)[:300]}

    host_link = overlap = restore = cpu = None
    if rank == 0:
        # flush alone (a4+a5) against the measured pinned-copy peak
        flush_ms = rig.time_flush()
        ach = d2h_bytes / (flush_ms * 1e-3) / 1e9
        host_link = {"bound": "host_link", "achieved": ach, "peak": link["d2h_gbs"], "unit": "GB/s",
                     "frac": ach / link["d2h_gbs"], "flush_ms": flush_ms, "chunk_mib": rig.chunk_mib,
                     "h2d_peak_gbs": link["h2d_gbs"]}
        # overlap: exposed checkpoint ms/iteration (PAPER.md:283 protocol)
        if not args.no_overlap:
            G = args.gemms if args.gemms > 0 else rig.headline_gemms(flush_ms)
            overlap = rig.overlap(G, args.overlap_iters, args.overlap_reps)
            if args.window == "eager" and not args.no_graph_arm:
                # the same experiment with the GEMM window replayed from a CUDA graph: separates the part of the
                # exposed time that is kernel-LAUNCH interference (PCIe busy with the D2H) from real contention
                og = rig.overlap(G, args.overlap_iters, args.overlap_reps, arms=("off", "on"), window="graph")
                overlap["graph_window"] = {k: og[k] for k in ("iter_ms_off", "iter_ms_on", "exposed_ms",
                                                              "exposed_frac_of_compute_step", "window_launch")}
            overlap["flush_ms"] = flush_ms
            overlap["rule"] = "G = smallest power of two with T_c >= 4 x T_D2H" if args.gemms <= 0 else "G given"
        # restore + recompute (a6, a7)
        back, rms, cms = rig.restore_timing()
        restore = {"restore_ms": rms, "recompute_ms": cms, "mode": rig.restore_mode_name, "restored_step": back,
                   "host_link_gbs": (d2h_bytes - 256) / (rms * 1e-3) / 1e9,
                   "frac_of_h2d_peak": (d2h_bytes - 256) / (rms * 1e-3) / 1e9 / link["h2d_gbs"]}
        # restore from the ring successor's received buffer (recovery stage 3 over NVLink)
        if peer and "error" not in peer:
            src = rig.ring.opened[0] if world > 1 else rig.recv.ptrs[0]
            rig.s.drop_live()
            torch.cuda.synchronize()
            p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            p0.record(rig.cur)
            back_p = B.phx_restore_from(rig.s.h, src, rig.cur)
            p1.record(rig.cur)
            torch.cuda.synchronize()
            rig.step = back_p
            pms = p0.elapsed_time(p1)
            peer.update(restore_from_peer_ms=pms, restore_from_peer_gbs=12 * N / (pms * 1e-3) / 1e9,
                        restored_step=back_p)
        # cpu baseline: the oracle on the host cores (rank 0, N == 1 only)
        if world == 1 and not args.no_cpu_baseline:
            cores = len(os.sched_getaffinity(0))
            sample = args.cpu_sample or min(N, 1 << 28)
            n_s, times = time_oracle(wl, sample, 3, 1, cores)
            t = sum(times) / len(times)
            n_1, times1 = time_oracle(wl, min(sample, 1 << 25), 2, 1, 1)
            t1 = sum(times1) / len(times1)
            cpu = {"value": BYTES_PER_ELEM * n_s / t / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": f"first {n_s} of {N} elements of the shard, 3 steps after 1 warm-up",
                   "elements_per_s": n_s / t, "single_thread_elements_per_s": n_1 / t1}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{wl.key}: {wl.title}", "elements_per_shard": int(N),
                       "state_bytes": int(12 * N), "staging_depth": rig.depth, "chunk_mib": rig.chunk_mib,
                       "sync_mode": rig.sync_name, "kernel_variant": args.variant, "snapshot_source": rig.source_name,
                       "bytes_per_element": BPE,
                       "precision": ("fp32 state + fp32 grads, no bf16 copy (PAPER.md:270): 16 B read + 24 B written"
                                     if rig.fp32 else "fp32 state + bf16 grads + bf16 copy (north_star): 14 B read + 26 B written"),
                       "decay_groups": bool(args.decay_groups),
                       "l2": "inputs larger than L2 (working set %.2f GB per step >> 126 MB)" % (BYTES_PER_ELEM * N / 1e9),
                       "timed_region": "K x phx_step_and_snapshot (a1 clip if configured, a2 sync-point wait, a3 fused "
                                       "AdamW+bf16 copy+packed snapshot); a4/a5 host flush is in e2e and overlap",
                       "host_payload": ("full rank state: envelope + p,m,v + model-parameter buffer W (SURVEY 8(f4))"
                                        if rig.full else "optimizer shard: envelope + p,m,v"),
                       "clip_scope": ("global: all-gather of one fp64 sum per rank (SURVEY 8(e))" if rig.gclip is not None
                                      else ("local" if wl.hyper.max_grad_norm > 0 else "none")),
                       "parallelism": (f"dp{world} shards, one 8-byte-per-rank all-gather per step (global clip)"
                                       if rig.gclip is not None else
                                       f"dp{world} independent shards, no data-path collective")},
            "elements_per_s": units / (ms_per_step * 1e-3),
            "exposed_ckpt_ms_per_iter": overlap["exposed_ms"] if overlap else None,
            "roofline": roofline, "host_link": host_link, "e2e": e2e, "overlap": overlap, "restore": restore,
            "peer_replication": peer, "publication": publication, "cpu_baseline": cpu, "gpu_launches": int(launches), "clocks": clk,
            "step_ms_min_max": [min(per), max(per)],
        }
        print(json.dumps(line), flush=True)
    barrier(world)      # peers' received buffers stay mapped until rank 0 has finished writing into them
    rig.close()
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


# ----------------------------------------------------------------------------------------------
# the other measurement rows of SURVEY.md §8(d): one JSON line per measurement
# ----------------------------------------------------------------------------------------------


def emit(**kw):
    print(json.dumps(kw), flush=True)


def run_configs(args):
    """Every config's kernel, snapshot-off kernel, clip pass, flush, both restore modes."""
    torch, rank, world, local_rank = gpu_setup()
    keys = [args.config] if args.config != "c2" else ["c1", "c2", "c3", "c4a", "c4b", "c5"]
    link = measure_host_link(torch, torch.device(f"cuda:{local_rank}"))
    peak, _ = measured_peaks()
    for key in keys:
        rig = Rig(args, key, host_grads=False)
        N = rig.N
        total_ms, per, _ = rig.time_steps(args.steps, max(args.warmup, 3))
        step_ms = total_ms / args.steps
        kern_ms = rig.time_fused_kernel_alone(args.steps) if rig.wl.hyper.max_grad_norm > 0 else step_ms
        off_ms = rig.time_steps_off(args.steps)
        flush_ms = rig.time_flush()
        _, r_bulk, rec = rig.restore_timing()
        B = rig.B
        replica, back_step = rig.s.replica, rig.step
        rig.close()
        # copy-engine restore on a fresh handle bound to the same replica (a replacement rank)
        r2 = rig.Shard(rig.wl, device=rig.device, restore_mode=B.PHX_RESTORE_COPY_ENGINE, replica=replica)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        r2.restore()
        e1.record()
        torch.cuda.synchronize()
        r_ce = e0.elapsed_time(e1)
        r2.close()
        gbs = BYTES_PER_ELEM * N / (kern_ms * 1e-3) / 1e9
        emit(mode="configs", config=key, elements=int(N), step_ms=step_ms, fused_kernel_ms=kern_ms,
             fused_gbs=gbs, frac_of_measured_peak=gbs / peak, frac_of_nominal=gbs / NOMINAL_HBM_GBS,
             elements_per_s=N / (step_ms * 1e-3), snapshot_off_step_ms=off_ms,
             snapshot_extra_ms=step_ms - off_ms, flush_ms=flush_ms,
             flush_gbs=rig_bytes(N) / (flush_ms * 1e-3) / 1e9, d2h_peak_gbs=link["d2h_gbs"],
             restore_bulk_ms=r_bulk, restore_bulk_gbs=12 * N / (r_bulk * 1e-3) / 1e9,
             restore_copy_engine_ms=r_ce, restore_copy_engine_gbs=12 * N / (r_ce * 1e-3) / 1e9,
             h2d_peak_gbs=link["h2d_gbs"], recompute_ms=rec,
             note="c1 fits in L2: reported, not an HBM figure" if key == "c1" else "")
        del rig, r2, replica
        torch.cuda.empty_cache()
    return 0


def rig_bytes(N):
    return 256 + 12 * N


def run_overlap_curve(args):
    """Exposed checkpoint ms/iteration against the length of the compute window (R21)."""
    torch, rank, world, local_rank = gpu_setup()
    rig = Rig(args, args.config, host_grads=False)
    flush_ms = rig.time_flush()
    gm = rig.gemm_setup()
    Gs = [int(x) for x in str(args.gemms).split(",")] if args.gemms > 0 else [64, 256, 1024, 4096, 16384]
    head = rig.headline_gemms(flush_ms)
    for G in sorted(set(Gs + [head])):
        t_iter = G * gm * 1.2 + 1.0
        iters = max(5, min(20, int(3000.0 / t_iter)))
        o = rig.overlap(G, iters, args.overlap_reps)
        emit(mode="overlap-curve", config=args.config, elements=int(rig.N), flush_ms=flush_ms, headline=(G == head),
             knee_gemms=flush_ms / gm, sync_mode=rig.sync_name, depth=rig.depth, chunk_mib=rig.chunk_mib, **o)
    rig.close()
    return 0


def run_timeline(args):
    """Copy/compute overlap as a timeline from CUDA events (nsys is not on the image): per iteration, when the
    GEMM window, the hot path (a1-a3) and the side-stream flush (a4+a5) of that iteration's snapshot start and end,
    all in ms since the first iteration's start.  One JSON line per iteration plus a summary."""
    torch, rank, world, local_rank = gpu_setup()
    rig = Rig(args, args.config, host_grads=False)
    flush_ms = rig.time_flush()
    rig.gemm_setup()
    a, b, c = rig._gemm
    G = args.gemms if args.gemms > 0 else rig.headline_gemms(flush_ms)
    iters, marks = 6, 8
    E = lambda: torch.cuda.Event(enable_timing=True)
    rows = []
    for _ in range(2):                       # warm-up iterations (not recorded)
        for _ in range(G):
            torch.matmul(a, b, out=c)
        rig.do_step()
        rig.flush()
    torch.cuda.synchronize()
    base = E()
    base.record(rig.cur)
    for it in range(iters):
        ev = {"gemm": [E()], "k0": E(), "k1": E(), "f0": E(), "f1": E()}
        ev["gemm"][0].record(rig.cur)
        for part in range(marks):
            for _ in range(G // marks):
                torch.matmul(a, b, out=c)
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
    t = lambda e: base.elapsed_time(e)
    for it, ev in enumerate(rows):
        # the flush is enqueued behind an event of the step kernel: its real start is max(f0, k1)
        emit(mode="timeline", config=args.config, iteration=it, gemms=G,
             gemm_window_ms=[t(ev["gemm"][0]), t(ev["gemm"][-1])],
             gemm_marks_ms=[t(e) for e in ev["gemm"]],
             hot_path_ms=[t(ev["k0"]), t(ev["k1"])],
             flush_ms=[max(t(ev["f0"]), t(ev["k1"])), t(ev["f1"])])
    # summary: how much of each flush lies under the NEXT iteration's GEMM window, and the wait at the sync point
    under, waits = [], []
    for it in range(iters - 1):
        f0, f1 = max(t(rows[it]["f0"]), t(rows[it]["k1"])), t(rows[it]["f1"])
        g0, g1 = t(rows[it + 1]["gemm"][0]), t(rows[it + 1]["gemm"][-1])
        under.append(max(0.0, min(f1, g1) - max(f0, g0)) / (f1 - f0))
        waits.append(max(0.0, f1 - t(rows[it + 1]["k0"])))
    emit(mode="timeline-summary", config=args.config, gemms=G, flush_alone_ms=flush_ms,
         flush_fraction_under_next_gemm_window=under, commit_after_next_step_enqueued_ms=waits,
         note="commit_after_next_step_enqueued_ms > 0 would be a stall at the single sync point (PAPER.md:226)")
    rig.close()
    return 0


def run_sweep(args):
    """BASELINE.json:configs[4]: D2H chunk size 4..256 MiB x staging depth 1..4 (x sync mode), reporting exposed
    checkpoint ms/iteration and host-link GB/s.  Run at a TIGHT compute window (T_c = 1.25 x T_D2H, where depth and
    chunking can matter) and, on a reduced grid, at the headline window (T_c >= 4 x T_D2H)."""
    torch, rank, world, local_rank = gpu_setup()
    key = args.config if args.config != "c2" else "c5"
    device = torch.device(f"cuda:{local_rank}")
    link = measure_host_link(torch, device)
    probe = Rig(args, key, host_grads=False)
    replica = probe.s.replica                        # pin once, reuse for every grid point
    flush_ref = probe.time_flush()
    gm = probe.gemm_setup()
    G_tight = max(1, int(round(1.25 * flush_ref / gm)))
    G_head = probe.headline_gemms(flush_ref)
    base = probe.overlap(G_tight, args.overlap_iters, 1, arms=("off",))
    base_head = probe.overlap(G_head, max(5, args.overlap_iters // 2), 1, arms=("off",))
    probe.close()
    del probe
    torch.cuda.empty_cache()
    chunks = [int(x) for x in args.chunks.split(",")]
    for sync in args.syncs.split(","):
        for depth in [int(x) for x in args.depths.split(",")]:
            for chunk in chunks:
                rig = Rig(args, key, depth=depth, chunk_mib=chunk, sync=sync, replica=replica, host_grads=False)
                flush_ms = rig.time_flush()
                o = rig.overlap(G_tight, args.overlap_iters, 1, arms=("on",))
                row = dict(mode="sweep", window="tight(1.25xT_D2H)", config=key, elements=int(rig.N), sync_mode=sync,
                           depth=depth, chunk_mib=chunk, flush_ms=flush_ms,
                           host_link_gbs=rig_bytes(rig.N) / (flush_ms * 1e-3) / 1e9, d2h_peak_gbs=link["d2h_gbs"],
                           gemms_per_iter=G_tight, iter_ms_on=o["iter_ms_on"], iter_ms_off=base["iter_ms_off"],
                           exposed_ms=o["iter_ms_on"] - base["iter_ms_off"],
                           exposed_frac=(o["iter_ms_on"] - base["iter_ms_off"]) / base["iter_ms_off"],
                           hot_path_ms_in_loop_on=o["hot_path_ms_in_loop_on"])
                emit(**row)
                if depth in (1, 2) and chunk in (chunks[0], 64, 256):
                    o = rig.overlap(G_head, max(5, args.overlap_iters // 2), 1, arms=("on",))
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


def run_hotswap(args):
    """BASELINE.json:configs[3]: 20 steps with snapshots, drop the live shard while step 21 is in flight, restore
    from the pinned host replica, recompute step 21, run 22..25; time restore + recompute and check the trajectory
    bit-exactly against an uninterrupted run (GPU vs GPU; GPU vs oracle is in tests/)."""
    torch, rank, world, local_rank = gpu_setup()
    keys = [args.config] if args.config != "c2" else ["c4a", "c4b"]
    for key in keys:
        for rmode_name in ("bulk_kernel", "copy_engine"):
            from paper_2607_01646_b200 import binding as B
            rmode = B.PHX_RESTORE_BULK_KERNEL if rmode_name == "bulk_kernel" else B.PHX_RESTORE_COPY_ENGINE
            rig = Rig(args, key, host_grads=False, restore_mode=rmode)
            W, wl, N = rig.W, rig.wl, rig.N
            G = rig.headline_gemms(rig.time_flush(), factor=1.25)
            rig.s.p.copy_(W.init_params(rig.s.n, N, wl.seed, device=rig.device))
            rig.s.m.zero_(); rig.s.v.zero_()
            rig.s.set_state(0)
            rig.step = 0
            a, b, c = rig._gemm
            # uninterrupted reference trajectory first (snapshot-off handle on its own arrays)
            ref = rig.Shard(wl, device=rig.device, snapshot=False)
            ref.p.copy_(rig.s.p); ref.set_state(0)
            for t in range(1, 26):
                ref.step_and_snapshot(rig.grads[t & 1], t)
            torch.cuda.synchronize()
            for t in range(1, 21):                       # 20 steps, snapshot + flush every step, overlapped
                for _ in range(G):
                    torch.matmul(a, b, out=c)
                rig.do_step()
                rig.s.flush_async(rig.side)
            rig.do_step()                                # step 21 launched: in flight when the fault hits
            torch.cuda.synchronize()
            rig.s.drop_live()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            r0, r1, r2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            r0.record(rig.cur)
            back = rig.s.restore()
            r1.record(rig.cur)
            rig.step = back
            rig.do_step()                                # recompute of the in-flight step (a7)
            r2.record(rig.cur)
            torch.cuda.synchronize()
            wall_ms = (time.perf_counter() - t0) * 1e3
            for t in range(22, 26):
                rig.do_step()
                rig.s.flush_async(rig.side)
            rig.s.wait(25)
            torch.cuda.synchronize()
            same = all(torch.equal(x, y) for x, y in ((rig.s.p, ref.p), (rig.s.m, ref.m), (rig.s.v, ref.v),
                                                      (rig.s.p16, ref.p16)))
            rms = r0.elapsed_time(r1)
            emit(mode="hotswap", config=key, elements=int(N), restore_mode=rmode_name, restored_step=int(back),
                 restore_ms=rms, recompute_ms=r1.elapsed_time(r2), restore_plus_recompute_wall_ms=wall_ms,
                 host_link_gbs=12 * N / (rms * 1e-3) / 1e9, trajectory_bit_exact_vs_uninterrupted=bool(same),
                 steps_before_fault=20, steps_after=5, gemms_per_iter=G)
            ref.close()
            rig.close()
            del rig, ref
            torch.cuda.empty_cache()
            if not same:
                return 1
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return {"headline": run_headline, "configs": run_configs, "overlap-curve": run_overlap_curve,
            "sweep": run_sweep, "hotswap": run_hotswap, "timeline": run_timeline}[args.mode](args)


if __name__ == "__main__":
    sys.exit(main())
