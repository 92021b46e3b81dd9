#!/usr/bin/env python
"""bench.py -- request-steps scheduled per second on B200 and fraction of the HBM roofline.

Workload of the headline line (BASELINE.json configs[4], the largest single-GPU configuration, "config5"): 65536
replicas x 8192 requests, 50/50 chat/reasoning mix, Poisson arrivals at 95 % load, KV capacity 16384 blocks, queue cap
2048, BOOST gamma = 0.3, swap-vs-recompute preemption; seeded synthetic traces (workloads.config5).

A "step" is one ub_step(h, ITERS) call: every replica advances ITERS scheduler iterations, each iteration one launch of
the streaming step kernel ub::k_stream per half of the replicas (all of a0..a5: the replica's window goes HBM -> SM ->
HBM once); what it queues for the team kernels (nothing in this config) runs once per ub_step call.  Before the timed
region every replica is advanced SPINUP iterations (not timed, default 65536 = the middle of the ~1.4e5 iterations a
config-5 replica runs) so that the queues are in their loaded regime.  The timed region is K steps on the device (CUDA
events, barrier + synchronize on both sides, max over ranks).  The windows read per launch (~0.4 GB) are larger than L2
(126 MB), so no explicit flush is needed.

Beside the headline the line carries (extra keys): the same job from the first arrival to the last completion
(`whole_job`), the device-resident percentile reduction timed at full size (`stats`), the resident-state mode, and --
on one GPU -- the chat-heavy (config 2) and reasoning-heavy (config 3) workloads of BASELINE.json run as whole jobs
(`workloads`), the oracle on one host core and on all of them (`cpu_baseline`).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import socket
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
SMALL_JOB_IPL = 64                   # resident mode of the small whole jobs (configs 2, 3): 16 -> 64 is +10 %
ALG_BYTES_PER_REQUEST_STEP = 40      # read a,P,D,d,cached,flags (28 B) + write d,cached,flags (12 B)
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r02_stream_traffic.csv")   # written from the ncu --set full capture
METRIC = "request-steps scheduled/sec"
UNIT = "request-steps/s"
COLS = ["iterations", "request_steps", "n_completed", "evict_recompute", "evict_swap", "swapins", "tokens_lost",
        "tokens_emitted", "prefill_tokens", "decode_seqs", "t_end_us", "peak_active", "done", "swap_used"]
COL = {name: i for i, name in enumerate(COLS)}
TTLT_P99_COL = len(COLS) + 3 + 2       # ttft_us[3], then ttlt_us[2]


def parse(argv=None):
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
    ap.add_argument("--cpu-sample", type=int, default=64, help="replicas the one-core oracle baseline runs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="headline only: no whole job, no config 2 / 3 (profiling runs)")
    ap.add_argument("--probe", default=None, choices=["gamma_ada"],
                    help="run only this extra key of the bench line and print it (profiling runs: profiles/r02_gamma_ada.md)")
    return ap.parse_args(argv)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def profiled_traffic():
    """DRAM read + write bytes of the k_stream launches of one round, from the committed ncu capture of this kernel
    (profiles/r02_stream_traffic.csv: one row per launch of the round); None if the file is absent."""
    try:
        with open(TRAFFIC_CSV) as f:
            rows = [r for r in csv.DictReader(l for l in f if not l.startswith("#"))]
        return float(sum(float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]) for r in rows)), \
            os.path.relpath(TRAFFIC_CSV, ROOT)
    except Exception:
        return None, None


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


# ---------------------------------------------------------------------------------------------- the oracle legs

def _oracle_job(job):
    """(request-steps, seconds) of the oracle as it stands, single thread, on the given replicas of config 5."""
    n_seeds, n_requests, ids, n_iters = job
    from oracle import oracle as O
    sub = W.config5(n_seeds=n_seeds, n_requests=n_requests).select(ids)
    o = O.OracleSim(sub.sim, sub.replicas, sub.traces())
    t0 = time.perf_counter()
    o.step(n_iters)
    dt = time.perf_counter() - t0
    rs = sum(s["request_steps"] for s in o.stats())
    o.close()
    return rs, dt


def cpu_baselines(R, N, n_iters, sample):
    """The oracle on one host core, and on all of them (one process per core, each its own replicas)."""
    import multiprocessing as mp
    ids = list(range(0, R, max(1, R // sample)))[:sample]
    rs1, dt1 = _oracle_job((R, N, ids, n_iters))
    out = {"value": rs1 / dt1, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"{len(ids)} of {R} replicas of config5 for the same {n_iters} iterations ({dt1:.1f} s)"}
    nproc = os.cpu_count() or 1
    per = max(2, sample // 4)
    pool_ids = [r % R for r in range(1, 1 + nproc * per * 7, 7)]
    jobs = [(R, N, pool_ids[i * per:(i + 1) * per], n_iters) for i in range(nproc)]
    t0 = time.perf_counter()
    with mp.get_context("spawn").Pool(nproc) as pool:
        res = pool.map(_oracle_job, jobs)
    wall = time.perf_counter() - t0
    busy = max(dt for _, dt in res)
    out["all_cores"] = {"value": sum(rs for rs, _ in res) / busy, "unit": UNIT, "cores": nproc, "nproc": nproc,
                        "kind": "oracle, one process per core",
                        "sample": f"{per} replicas per process x {nproc} processes for the same {n_iters} iterations "
                                  f"(slowest process {busy:.1f} s, wall with start-up {wall:.1f} s)"}
    return out


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
    for _ in range(args.warmup):
        o.step(args.iters)
    rs1 = sum(s["request_steps"] for s in o.stats())
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(args.iters)
    dt = time.perf_counter() - t0
    rs2 = sum(s["request_steps"] for s in o.stats())
    val = (rs2 - rs1) / dt
    sample = (f"{len(ids)} of {args.replicas} replicas of config5, {args.steps} steps x {args.iters} iterations after "
              f"{args.spinup} spin-up iterations")
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


# ---------------------------------------------------------------------------------------------- the CUDA arm

def torchrun_command(args, argv, port):
    """The launch line of the contract: one rank per GPU of one node, rendezvous on 127.0.0.1."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def reexec_under_torchrun(args):
    """`python bench.py --gpus N` outside torchrun: launch N ranks of this script (one per GPU) and become them."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.execv(sys.executable, torchrun_command(args, sys.argv[1:], port))


def rank_layout(args, env):
    """(rank, world, local rank) of this process; `--gpus N` must agree with the launcher's WORLD_SIZE."""
    rank = int(env.get("RANK", "0")); world = int(env.get("WORLD_SIZE", "1")); local = int(env.get("LOCAL_RANK", "0"))
    if args.gpus != world:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE is {world}")
    return rank, world, local


def stats_table(B, sim, R):
    st = sim.stats_raw()                                             # device percentile reduction + D2H
    words = B.C.sizeof(B.UbReplicaStats) // 8
    return np.frombuffer(st, dtype=np.int64).reshape(R, words).copy()


def whole_job(B, wl, traces, stream, peak, label):
    """One workload from the first arrival to the last completion through ub_run; request-steps / device time of the
    step launches (CUDA events inside ub_run), the 40-byte roofline fraction and the mean window size."""
    R = int(wl.sim["n_replicas"])
    sim = B.Sim(wl.sim, wl.replicas, traces, stream=stream)
    t0 = time.perf_counter()
    issued = sim.run()
    wall = time.perf_counter() - t0
    ms, launches = sim.last_step_timing()
    t1 = time.perf_counter()
    st = stats_table(B, sim, R)
    t_stats = time.perf_counter() - t1
    rs = int(st[:, COL["request_steps"]].sum()); its = int(st[:, COL["iterations"]].sum())
    sim.close()
    # the same job with 64 iterations per launch (resident-state mode: same schedules, the mode for small configurations)
    sim = B.Sim(wl.sim, wl.replicas, traces, stream=stream, iters_per_launch=SMALL_JOB_IPL)
    sim.run()
    ms16, _ = sim.last_step_timing()
    rs16 = int(stats_table(B, sim, R)[:, COL["request_steps"]].sum())
    sim.close()
    assert rs16 == rs, "the schedule must not depend on iters_per_launch"
    return {"workload": label, "value_resident": rs16 / (ms16 * 1e-3), "resident_iters_per_launch": SMALL_JOB_IPL, "replicas": R, "value": rs / (ms * 1e-3), "unit": UNIT,
            "roofline_frac": rs * ALG_BYTES_PER_REQUEST_STEP / (ms * 1e-3) / 1e9 / peak,
            "request_steps": rs, "device_ms": ms, "wall_s": wall, "iterations_issued": int(issued),
            "iterations_executed_max": int(st[:, COL["iterations"]].max()), "rounds_launched": int(launches),
            "mean_window": rs / max(1, its), "ub_stats_s": t_stats,
            "completed": int(st[:, COL["n_completed"]].sum())}


def gamma_ada_probe(B, w4, tr4, stream, iters=4096):
    """Config 4 (distribution shift + memory pressure, 16384 replicas) for `iters` iterations from its loaded phase, once
    as the static gamma sweep and once with gamma-Ada on every replica: what a round costs when UPDATEGAMMA (k_gamma_ada,
    one warp per replica) and the hand-over of re-keyed replicas to the team kernels (k_step) run every round."""
    out = {}
    R = int(w4.sim["n_replicas"])
    for label, ada in (("static", None), ("gamma_ada", dict(window=256, min_samples=32, beta_shift=3, levels=32,
                                                            gamma_min=0.01, gamma_max=100.0, eps_us=1000))):
        sim = B.Sim(w4.sim, w4.replicas, tr4, stream=stream)
        if ada:
            sim.set_gamma_ada(ada, np.ones(R, np.uint8))
        sim.step(150000)                                             # into the overloaded second half of the trace
        rs0 = sum(int(st.request_steps) for st in sim.stats_raw())
        sim.step(iters)
        ms, rounds = sim.last_step_timing()
        st = sim.stats_raw()
        rs1 = sum(int(x.request_steps) for x in st)
        out[label] = {"us_per_round": 1e3 * ms / max(1, rounds), "value": (rs1 - rs0) / (ms * 1e-3), "unit": UNIT,
                      "mean_window": (rs1 - rs0) / max(1, iters) / R, "rounds": int(rounds)}
        if ada:
            out[label]["gamma_updates"] = int(sum(sim.gamma_state(r)[2] for r in range(0, R, 64)) * 64)
        sim.close()
    out["note"] = ("config4, 16384 replicas x 2000 requests, 4096 iterations after 150000; with adaptation on every round is "
                   "k_gamma_ada + ub::k_stream<true,...> + the team kernels for replicas whose level changed")
    return out


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    if args.probe == "gamma_ada":
        w4 = W.config4()
        tr4 = w4.traces(workers=max(1, min(32, os.cpu_count() or 1)))
        import torch
        from paper_2606_18431_b200 import binding as B
        if not torch.cuda.is_available():
            raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback")
        print(json.dumps({"gamma_ada": gamma_ada_probe(B, w4, tr4, torch.cuda.current_stream().cuda_stream)}))
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        reexec_under_torchrun(args)
    rank, world, local = rank_layout(args, os.environ)

    # ---- synthetic traces first (the generator forks worker processes: before CUDA / NCCL are initialised).
    # Replicas are independent units, sharded over ranks by seed (weak scaling).
    from paper_2606_18431_b200 import sharding as SH
    R, N = args.replicas, args.requests
    wl = SH.shard_workload(W.config5, rank, world, R, N)
    t_gen = time.perf_counter()
    nw = max(1, min(32, (os.cpu_count() or 1) // max(1, world)))
    a, p, d, n = wl.traces(workers=nw)
    t_gen = time.perf_counter() - t_gen
    # (on one GPU also the chat-heavy and reasoning-heavy workloads north_star names, run as whole jobs at the end)
    side = []
    if world == 1 and not args.no_extras:
        for mk, label in ((W.config2, "config2: chat-heavy, 1024 seeds x {FCFS, SRPT, BOOST}"),
                          (W.config3, "config3: reasoning-heavy, 4096 replicas, MMPP-2 arrivals, swap-vs-recompute")):
            w2 = mk()
            side.append((w2, w2.traces(workers=nw), label))
        w4 = W.config4()
        tr4 = w4.traces(workers=nw)

    import torch
    import torch.distributed as dist
    from paper_2606_18431_b200 import binding as B
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
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
    reps = B.make_replicas(wl.replicas, R)
    B.ub_set_replicas(h, reps)
    sim = B.Sim.__new__(B.Sim); sim._h, sim.R, sim.N, sim.Q = h, R, N, int(wl.sim["queue_cap"])

    B.ub_step(h, args.spinup)                                        # populate the queues (untimed)
    for _ in range(args.warmup):
        B.ub_step(h, args.iters)
    st1 = stats_table(B, sim, R)
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

    st2 = stats_table(B, sim, R)
    t_e2e = time.perf_counter() - t_e2e0
    rs2 = int(st2[:, COL["request_steps"]].sum())

    # resident-state mode, reported separately: 16 iterations per launch, a warp advances its
    # replica 16 iterations in a row and the window is re-read from L2; same schedule, fewer HBM bytes
    B.ub_set_iters_per_launch(h, RESIDENT_IPL)
    B.ub_step(h, args.iters)
    st3 = stats_table(B, sim, R)
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    for _ in range(args.steps):
        B.ub_step(h, args.iters)
    f1.record()
    torch.cuda.synchronize()
    ms_res = f0.elapsed_time(f1)
    st4 = stats_table(B, sim, R)
    rs_res = int(st4[:, COL["request_steps"]].sum()) - int(st3[:, COL["request_steps"]].sum())
    B.ub_set_iters_per_launch(h, args.iters_per_launch)

    d2h_bytes = R * (B.C.sizeof(B.UbReplicaStats))
    ttlt_p99_us = st2[:, TTLT_P99_COL][st2[:, COL["n_completed"]] > 0]
    p99 = float(np.median(ttlt_p99_us)) * 1e-6 if ttlt_p99_us.size else 0.0
    ipl = max(1, args.iters_per_launch)
    rounds = args.steps * ((args.iters + ipl - 1) // ipl)
    nsplit = 2 if R >= 8192 else 1
    # kernels of this library launched inside the timed region: per round one k_stream per half; per ub_step call the
    # hand-over flush (one k_step<8,8,1> per half in an all-streaming job; plus one 16-byte memset per half)
    launches = rounds * nsplit + args.steps * nsplit
    steps_in_job = args.spinup / max(1, args.iters) + args.warmup + args.steps

    # ---- the same job from the first arrival to the last completion (ub_set_replicas rewinds it), and the percentile
    # reduction at full size behind it
    extras = {}
    if not args.no_extras:
        B.ub_set_replicas(h, reps)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        issued = B.ub_run(h)
        wall = time.perf_counter() - t0
        ms_job, rounds_job = B.ub_last_step_timing(h)
        t0 = time.perf_counter()
        stj = stats_table(B, sim, R)
        t_stats = time.perf_counter() - t0
        rs_job = int(stj[:, COL["request_steps"]].sum())
        extras["whole_job"] = {
            "value": rs_job / (ms_job * 1e-3) * world, "unit": UNIT, "request_steps_per_gpu": rs_job,
            "device_s": ms_job * 1e-3, "wall_s": wall, "iterations_issued": int(issued),
            "iterations_executed_max": int(stj[:, COL["iterations"]].max()), "rounds_launched": int(rounds_job),
            "mean_window": rs_job / max(1, int(stj[:, COL["iterations"]].sum())),
            "completed_per_gpu": int(stj[:, COL["n_completed"]].sum()),
            "note": "config5 from the first arrival to the last completion through ub_run, one iteration per launch: "
                    "ramp-up with small windows, the loaded middle, the tail with few live replicas; per-rank value x ranks"}
        extras["stats"] = {"ub_stats_s": t_stats, "requests_reduced": int(stj[:, COL["n_completed"]].sum()),
                           "note": "ub_stats at full size: k_stats (6 exact nearest-rank selections per replica over its "
                                   "completed requests + TBT histogram percentiles) + D2H of R structs + host conversion"}

    rs_timed, rs_all, ms, t_e2e = SH.aggregate(rs2 - rs1, rs2, ms, t_e2e, "cuda", world)
    job_stats = SH.gather_replica_stats(st2[:, [COL["request_steps"], COL["n_completed"], TTLT_P99_COL]], "cuda", world)
    sim.close()

    if rank == 0:
        peak, peak_src = peaks()
        value = rs_timed / (ms * 1e-3)
        per_gpu_bytes = (rs2 - rs1) * ALG_BYTES_PER_REQUEST_STEP
        ach = per_gpu_bytes / (ms * 1e-3) / 1e9
        n_mean = (rs2 - rs1) / max(1, (args.steps * args.iters)) / max(1, live1)
        traffic, traffic_src = profiled_traffic()
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / max(1, args.steps), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
            "config": {"workload": "config5: 65536 replicas x 8192 requests, 50/50 chat/reasoning, 95% load, KV 16384 blocks, queue cap 2048",
                       "replicas_per_gpu": R, "requests": N, "iters_per_step": args.iters,
                       "iters_per_launch": ipl, "spinup_iters": args.spinup,
                       "mean_active_per_live_replica": n_mean, "live_replicas": live1,
                       "iterations_before_timed": int(it1), "l2": "inputs larger than L2 (no flush)",
                       "trace_generation_s": t_gen, "median_p99_ttlt_s": p99,
                       "job_replicas_gathered": int(job_stats.shape[0])},
            "roofline": {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                         "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                         "kernel": "ub::k_stream<false,false,false,false,true> (one iteration per launch, all replicas, the instance for all-BOOST-with-MemGuard jobs)",
                         "alg_bytes_per_request_step": ALG_BYTES_PER_REQUEST_STEP,
                         "request_steps_per_launch": (rs2 - rs1) / max(1, rounds),
                         "avg_launch_ms": ms / max(1, rounds),
                         "note": "a round = every live replica advanced one iteration = two overlapping k_stream launches "
                                 "(one half of the replicas each, on two streams); the team kernels run once per ub_step; "
                                 "avg_launch_ms, request_steps_per_launch and traffic are per round; traffic = dram "
                                 "read+write bytes of the round's k_stream launches in the committed ncu --set full capture"},
            "e2e": {"value": rs_all / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d_bytes / steps_in_job,
                    "d2h_bytes_per_step": 2 * d2h_bytes / steps_in_job, "h2d_bytes_per_job": h2d_bytes,
                    "d2h_bytes_per_job": 2 * d2h_bytes, "steps_in_job": steps_in_job,
                    "note": "one job through the C-ABI from pinned host buffers: ub_create + ub_load_trace (H2D) + ub_set_replicas "
                            "+ spin-up + warm-up + timed steps (steps_in_job steps of iters_per_step iterations) + 2x ub_stats "
                            "(D2H); all request-steps / wall; bytes per step = bytes of the job / steps_in_job"},
            "resident": {"value": rs_res / (ms_res * 1e-3) * world, "unit": UNIT, "iters_per_launch": RESIDENT_IPL,
                         "note": "same K steps with 16 iterations per kernel launch (window re-read from L2, not HBM); "
                                 "per-rank value x ranks; not the roofline path"},
            "gpu_launches": launches, "clocks": clocks,
        }
        out.update(extras)
        if world == 1 and not args.no_extras:
            # the chat-heavy and reasoning-heavy workloads north_star names, as whole jobs
            out["workloads"] = [whole_job(B, w2, tr2, stream, peak, label) for w2, tr2, label in side]
            out["gamma_ada"] = gamma_ada_probe(B, w4, tr4, stream)
        if not args.no_cpu_baseline and world == 1:
            n_it = args.spinup + (args.warmup + args.steps) * args.iters
            out["cpu_baseline"] = cpu_baselines(R, N, n_it, args.cpu_sample)
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
