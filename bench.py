#!/usr/bin/env python
"""bench.py -- request-steps scheduled per second on B200 and fraction of the HBM roofline.

Workload (BASELINE.json configs[4], the largest single-GPU configuration, "config5"): 65536 replicas x 8192
requests, 50/50 chat/reasoning mix, Poisson arrivals at 95 % load, KV capacity 16384 blocks, queue cap 2048,
BOOST gamma = 0.3, swap-vs-recompute preemption; seeded synthetic traces (workloads.config5).

A "step" is one ub_step(h, ITERS) call: every replica advances ITERS scheduler iterations, each iteration one
launch of the streaming step kernel ub::k_stream per half of the replicas (all of a0..a5: the replica's window goes
HBM -> SM -> HBM once); what it queues for the team kernels (nothing in this config) runs once per ub_step call.  Before the timed
region every replica is advanced SPINUP iterations (not timed, default 65536 = the middle of the ~1.4e5
iterations a config-5 replica runs) so that the queues are in their loaded regime.  The timed region is K steps on
the device (CUDA events, barrier + synchronize on both sides, max over ranks).  The windows read per launch
(~0.4 GB) are larger than L2 (126 MB), so no explicit flush is needed.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_18431_b200 import workloads as W  # noqa: E402

RESIDENT_IPL = 16
KERNELS_PER_ROUND = 2                # a round = two halves on two streams, one ub::k_stream launch each (team kernels run once per ub_step)
TRAFFIC_BYTES_PER_LAUNCH = 463.3e6   # dram read+write bytes of the two ub::k_stream launches of one round, profiles/r01g_stream.md
ALG_BYTES_PER_REQUEST_STEP = 40      # read a,P,D,d,cached,flags (28 B) + write d,cached,flags (12 B)
METRIC = "request-steps scheduled/sec"
UNIT = "request-steps/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--iters", type=int, default=128, help="scheduler iterations per step")
    ap.add_argument("--spinup", type=int, default=65536, help="untimed iterations before the warm-up")
    ap.add_argument("--replicas", type=int, default=65536, help="replicas per GPU (config5: 65536)")
    ap.add_argument("--requests", type=int, default=8192)
    ap.add_argument("--iters-per-launch", type=int, default=1)
    ap.add_argument("--cpu-sample", type=int, default=64, help="replicas the oracle baseline runs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_rate(wl, replica_ids, n_iters):
    """The oracle as it stands, single thread, on a bounded sample of the same workload."""
    from oracle import oracle as O
    sub = wl.select(replica_ids)
    o = O.OracleSim(sub.sim, sub.replicas, sub.traces())
    t0 = time.perf_counter()
    o.step(n_iters)
    dt = time.perf_counter() - t0
    rs = sum(s["request_steps"] for s in o.stats())
    o.close()
    return rs, dt


def run_reference(args):
    """--impl reference: the CPU oracle (kind 'oracle') on the box's host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    wl = W.config5(n_seeds=args.replicas, n_requests=args.requests)
    from oracle import oracle as O
    ids = list(range(0, args.replicas, max(1, args.replicas // 32)))[:32]
    sub = wl.select(ids)
    o = O.OracleSim(sub.sim, sub.replicas, sub.traces())
    o.step(args.spinup)                                   # same populated-queue regime as the CUDA arm
    rs0 = sum(s["request_steps"] for s in o.stats())
    for _ in range(args.warmup):
        o.step(args.iters)
    rs1 = sum(s["request_steps"] for s in o.stats())
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(args.iters)
    dt = time.perf_counter() - t0
    rs2 = sum(s["request_steps"] for s in o.stats())
    val = (rs2 - rs1) / dt
    sample = f"{len(ids)} of {args.replicas} replicas of config5, {args.steps} steps x {args.iters} iterations after {args.spinup} spin-up iterations"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": "config5: 65536 replicas x 8192 requests (oracle runs a bounded sample)",
                   "replicas_per_gpu": args.replicas, "requests": args.requests, "iters_per_step": args.iters},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))
    o.close()
    del rs0


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2606_18431_b200 import binding as B
    from paper_2606_18431_b200 import sharding as SH

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # ---- synthetic traces: replicas are independent units, sharded over ranks by seed (weak scaling)
    R, N = args.replicas, args.requests
    wl = SH.shard_workload(W.config5, rank, world, R, N)
    t_gen = time.perf_counter()
    a, p, d, n = wl.traces(workers=max(1, min(32, (os.cpu_count() or 1) // max(1, world))))
    t_gen = time.perf_counter() - t_gen
    pin = [torch.from_numpy(x).pin_memory() for x in (a, p, d)]       # e2e copies from pinned host memory
    a, p, d = [x.numpy() for x in pin]
    h2d_bytes = a.nbytes + p.nbytes + d.nbytes + n.nbytes

    stream = torch.cuda.current_stream().cuda_stream
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t_e2e0 = time.perf_counter()
    h = B.ub_create(B.make_config(wl.sim, args.iters_per_launch, local, stream))
    B.ub_load_trace(h, a, p, d, n)                                   # host -> device inside the e2e region
    B.ub_set_replicas(h, B.make_replicas(wl.replicas, R))
    sim = B.Sim.__new__(B.Sim); sim._h, sim.R, sim.N, sim.Q = h, R, N, int(wl.sim["queue_cap"])

    B.ub_step(h, args.spinup)                                        # populate the queues (untimed)
    for _ in range(args.warmup):
        B.ub_step(h, args.iters)
    def stats_table():
        st = sim.stats_raw()                                         # device percentile reduction + D2H
        words = B.C.sizeof(B.UbReplicaStats) // 8
        return np.frombuffer(st, dtype=np.int64).reshape(R, words).copy()
    COL = {name: i for i, name in enumerate(
        ["iterations", "request_steps", "n_completed", "evict_recompute", "evict_swap", "swapins", "tokens_lost",
         "tokens_emitted", "prefill_tokens", "decode_seqs", "t_end_us", "peak_active", "done", "swap_used"])}
    st1 = stats_table()
    rs1 = int(st1[:, COL["request_steps"]].sum()); it1 = int(st1[:, COL["iterations"]].max())
    live1 = int((st1[:, COL["done"]] == 0).sum())

    sampler = ClockSampler(local); sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    e0.record()
    for _ in range(args.steps):
        B.ub_step(h, args.iters)
    e1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()

    st2 = stats_table()
    t_e2e = time.perf_counter() - t_e2e0

    # resident-state mode, reported separately: 16 iterations per launch, a warp advances its
    # replica 16 iterations in a row and the window is re-read from L2; same schedule, fewer HBM bytes
    B.ub_set_iters_per_launch(h, RESIDENT_IPL)
    B.ub_step(h, args.iters)
    st3 = stats_table()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    for _ in range(args.steps):
        B.ub_step(h, args.iters)
    f1.record()
    torch.cuda.synchronize()
    ms_res = f0.elapsed_time(f1)
    st4 = stats_table()
    rs_res = int(st4[:, COL["request_steps"]].sum()) - int(st3[:, COL["request_steps"]].sum())
    B.ub_set_iters_per_launch(h, args.iters_per_launch)
    rs2 = int(st2[:, COL["request_steps"]].sum())
    d2h_bytes = R * (B.C.sizeof(B.UbReplicaStats))
    ttlt_p99_us = st2[:, 14 + 3 + 2][st2[:, COL["n_completed"]] > 0]          # ttlt_us[2]
    p99 = float(np.median(ttlt_p99_us)) * 1e-6 if ttlt_p99_us.size else 0.0
    rounds = args.steps * ((args.iters + max(1, args.iters_per_launch) - 1) // max(1, args.iters_per_launch))
    launches = rounds * KERNELS_PER_ROUND

    rs_timed, rs_all, ms, t_e2e = SH.aggregate(rs2 - rs1, rs2, ms, t_e2e, "cuda", world)

    if rank == 0:
        peak, peak_src = peaks()
        value = rs_timed / (ms * 1e-3)
        per_gpu_bytes = (rs2 - rs1) * ALG_BYTES_PER_REQUEST_STEP
        ach = per_gpu_bytes / (ms * 1e-3) / 1e9
        n_mean = (rs2 - rs1) / max(1, (args.steps * args.iters)) / max(1, live1)
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / max(1, args.steps), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
            "config": {"workload": "config5: 65536 replicas x 8192 requests, 50/50 chat/reasoning, 95% load, KV 16384 blocks, queue cap 2048",
                       "replicas_per_gpu": R, "requests": N, "iters_per_step": args.iters,
                       "iters_per_launch": max(1, args.iters_per_launch), "spinup_iters": args.spinup,
                       "mean_active_per_live_replica": n_mean, "live_replicas": live1,
                       "iterations_before_timed": int(it1), "l2": "inputs larger than L2 (no flush)",
                       "trace_generation_s": t_gen, "median_p99_ttlt_s": p99},
            "roofline": {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                         "traffic": TRAFFIC_BYTES_PER_LAUNCH, "peak_source": peak_src, "kernel": "ub::k_stream",
                         "alg_bytes_per_request_step": ALG_BYTES_PER_REQUEST_STEP,
                         "request_steps_per_launch": (rs2 - rs1) / max(1, rounds),
                         "avg_launch_ms": ms / max(1, rounds),
                         "note": "a round = every live replica advanced one iteration = two overlapping k_stream launches "
                                 "(one half of the replicas each, on two streams); the team kernels run once per ub_step; "
                                 "avg_launch_ms, request_steps_per_launch and traffic are per round; traffic = dram "
                                 "read+write bytes of the round's k_stream launches from profiles/ (ncu --set full)"},
            "e2e": {"value": rs_all / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": d2h_bytes,
                    "note": "one job: ub_create + ub_load_trace from pinned host + ub_set_replicas + spin-up + warm-up + timed steps + 2x ub_stats D2H; all request-steps / wall"},
            "resident": {"value": rs_res / (ms_res * 1e-3) * world, "unit": UNIT, "iters_per_launch": RESIDENT_IPL,
                         "note": "same K steps with 16 iterations per kernel launch (window re-read from L2, not HBM); "
                                 "per-rank value x ranks; not the roofline path"},
            "gpu_launches": launches, "clocks": clocks,
        }
        if not args.no_cpu_baseline:
            ids = list(range(0, R, max(1, R // args.cpu_sample)))[:args.cpu_sample]
            n_it = args.spinup + (args.warmup + args.steps) * args.iters
            rs_o, dt_o = oracle_rate(wl, ids, n_it)
            out["cpu_baseline"] = {"value": rs_o / dt_o, "unit": UNIT, "cores": 1, "kind": "oracle",
                                   "sample": f"{len(ids)} of {R} replicas of config5 for the same {n_it} iterations ({dt_o:.1f} s)"}
        print(json.dumps(out))
    sim.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
