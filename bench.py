#!/usr/bin/env python
"""bench.py -- headline measurement of the NCCLX on-device data path on B200.

    python bench.py --gpus N --steps K --warmup W            (N>1: launched by torchrun, one rank per GPU)
    python bench.py --impl reference --steps K --warmup W    (the CPU oracle on the host cores)

A STEP is one pass of the whole hot path (a1-a6, r1, r2) over one batch of
synthetic input at BASELINE.json's full sizes:
    config 3  MoE dispatch AllToAllv, R=64, 16384 tokens x 5120 bf16 per rank, Zipf(1.1) top-1   (a1-a5)
    config 3  the inverse (combine) AllToAllv                                                    (a6)
    config 2  AllReduce sum, R=8, 4,194,304 bf16 per rank                                        (r1)
    config 4  ReduceScatter sum, R=16, 268,435,456 bf16 per rank                                 (r2)
metric = achieved HBM GB/s = algorithmic bytes (read + written) of the step / device time.
Inputs (48.6 GiB touched per step) are far larger than the 126 MB L2, so every step is cold.
Multi-GPU: the path does not shard across GPUs (north_star: one GPU) -> "replicas only": every
rank runs the same step on its own data, no data-path collective; value = sum over ranks / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2510_20171_b200 import workloads as W  # noqa: E402

METRIC = "achieved HBM GB/s, AllToAllv-dev + sum-reduce hot path (cfg3 dispatch+combine, cfg2, cfg4)"
NOMINAL_HBM_GBS = 8000.0
FALLBACK_HBM_GBS = 6650.0
GiB = 1 << 30


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ------------------------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------ workloads
class A2A:
    """Device-resident AllToAllv problem: send/recv/back buffers, count matrices, pointer tables."""

    def __init__(self, cfg: W.A2AConfig, torch, nx, with_back=True):
        self.cfg, self.R = cfg, cfg.R
        C = cfg.counts
        self.C_host = C
        es = W.ELEM_SIZE[cfg.dtype]
        self.send_elems = [int(C[s].sum()) for s in range(cfg.R)]
        self.recv_elems = [int(C[:, d].sum()) for d in range(cfg.R)]
        self.bytes_one_way = sum(self.send_elems) * es
        self.send = [W.torch_values(max(n, 8), cfg.dtype, cfg.seed * 1000 + s) for s, n in enumerate(self.send_elems)]
        td = W.torch_dtype(cfg.dtype)
        self.recv = [torch.empty(max(n, 8), dtype=td, device="cuda") for n in self.recv_elems]
        self.back = [torch.empty(max(n, 8), dtype=td, device="cuda") for n in self.send_elems] if with_back else None
        self.C = torch.from_numpy(C).cuda()
        self.RC = torch.empty_like(self.C)
        self.C2 = torch.empty_like(self.C)
        self.st, self.rt = nx.device_ptr_table(self.send), nx.device_ptr_table(self.recv)
        self.bt = nx.device_ptr_table(self.back) if with_back else None
        self.nx = nx

    def dispatch(self):
        self.nx.ncclx_alltoallv_dev(self.st, self.C, self.rt, self.RC, self.R, self.cfg.dtype)

    def combine(self):
        self.nx.ncclx_alltoallv_dev(self.rt, self.RC, self.bt, self.C2, self.R, self.cfg.dtype)


class Reduce:
    def __init__(self, cfg: W.ReduceConfig, torch, nx, sets: int = 1):
        self.cfg, self.R, self.nx = cfg, cfg.R, nx
        td = W.torch_dtype(cfg.dtype)
        es = W.ELEM_SIZE[cfg.dtype]
        self.sets = []
        for i in range(sets):
            x = [W.torch_values(cfg.count, cfg.dtype, cfg.seed * 1000 + 17 * i + k, cfg.std) for k in range(cfg.R)]
            n_out = cfg.count if cfg.kind == "allreduce" else cfg.count // cfg.R
            y = [torch.empty(n_out, dtype=td, device="cuda") for _ in range(cfg.R)]
            self.sets.append((x, y, nx.device_ptr_table(x), nx.device_ptr_table(y)))
        self.n_out = n_out
        self.bytes = cfg.R * cfg.count * es + cfg.R * n_out * es     # read + written

    def run(self, i: int = 0):
        x, y, xt, yt = self.sets[i % len(self.sets)]
        if self.cfg.kind == "allreduce":
            self.nx.ncclx_allreduce_sum(xt, yt, self.cfg.count, self.R, self.cfg.dtype)
        else:
            self.nx.ncclx_reducescatter_sum(xt, yt, self.n_out, self.R, self.cfg.dtype)


def event_times_ms(torch, fn, iters, warm=3):
    for _ in range(warm):
        fn()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(iters)]
    torch.cuda.synchronize()
    for a, b in ev:
        a.record(); fn(); b.record()
    torch.cuda.synchronize()
    return np.array([a.elapsed_time(b) for a, b in ev])


def frac(gbs, peak):
    return {"GBps": round(gbs, 1), "frac_of_measured": round(gbs / peak, 4), "frac_of_nominal_8TBps": round(gbs / NOMINAL_HBM_GBS, 4)}


# ------------------------------------------------------------------------------------ CPU oracle leg
def oracle_sample_step(state, nthreads):
    import oracle
    a, ar, rs = state["a2a"], state["ar"], state["rs"]
    oracle.alltoallv(a["send"], a["C"], a["recv"], "bf16", nthreads)
    RC = np.ascontiguousarray(a["C"].T)
    oracle.alltoallv(a["recv"], RC, a["back"], "bf16", nthreads)
    oracle.allreduce_sum(ar["x"], "bf16", nthreads, out=ar["y"])
    oracle.reducescatter_sum(rs["x"], "bf16", nthreads, out=rs["y"])


def oracle_sample_state(div=4):
    """Bounded sample of the step's workload: config 3 with every (src,dst) row count // div, config 2
    in full, config 4 with count // div elements per rank.  Values: N(0,1)/N(0,1e-3) bf16 bit patterns
    from numpy (timing does not depend on values)."""
    rng = np.random.default_rng(0)
    block = {}

    def vals(n, std=1.0):
        # one 16 Mi-element N(0,std) bf16 block, tiled: the oracle's timing does not depend on the values
        if std not in block:
            f = rng.standard_normal(1 << 24, dtype=np.float32) * np.float32(std)
            block[std] = (f.view(np.uint32) >> 16).astype(np.uint16)
        return np.resize(block[std], n)

    c3 = W.scaled_a2a(W.a2a_config(3), div)
    C = c3.counts
    R = c3.R
    a = {"C": C, "send": [vals(int(C[s].sum())) for s in range(R)],
         "recv": [np.empty(int(C[:, d].sum()), np.uint16) for d in range(R)],
         "back": [np.empty(int(C[s].sum()), np.uint16) for s in range(R)]}
    c2 = W.reduce_config(2)
    ar = {"x": [vals(c2.count) for _ in range(c2.R)], "y": [np.empty(c2.count, np.uint16) for _ in range(c2.R)]}
    c4 = W.reduce_config(4)
    n4 = c4.count // div
    rs = {"x": [vals(n4, 1e-3) for _ in range(c4.R)], "y": [np.empty(n4 // c4.R, np.uint16) for _ in range(c4.R)]}
    nbytes = 2 * 2 * sum(x.nbytes for x in a["send"]) + 2 * c2.R * c2.count * 2 + (c4.R * n4 * 2 + n4 * 2)
    sample = (f"config 3 dispatch+combine with row counts // {div} ({sum(x.nbytes for x in a['send']) / GiB:.2f} GiB each way), "
              f"config 2 in full, config 4 with {n4} elements per rank (1/{div})")
    return {"a2a": a, "ar": ar, "rs": rs}, nbytes, sample


def run_oracle_leg(steps, warmup, div=4, single_thread=True):
    """The oracle as it stands on the box's host cores: (a) single-threaded, (b) on all cores
    (OpenMP over destination ranks / element ranges), on the same bounded sample."""
    cores = os.cpu_count() or 1
    state, nbytes, sample = oracle_sample_state(div)
    for _ in range(max(0, warmup)):
        oracle_sample_step(state, cores)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_sample_step(state, cores)
    dt = (time.perf_counter() - t0) / steps
    out = {"value": round(nbytes / dt / 1e9, 3), "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": sample,
           "s_per_sample_step": round(dt, 3), "all_cores": round(nbytes / dt / 1e9, 3), "single_thread": None}
    if single_thread:
        t0 = time.perf_counter()
        oracle_sample_step(state, 1)
        d1 = time.perf_counter() - t0
        out["single_thread"] = round(nbytes / d1 / 1e9, 3)
        out["s_per_sample_step_single_thread"] = round(d1, 3)
    return out, dt


# ------------------------------------------------------------------------------------ multi-rank host logic
def init_dist(world: int, local_rank: int, backend: str = "nccl"):
    """One process per GPU; rendezvous on 127.0.0.1 (env MASTER_* / RANK / WORLD_SIZE from torchrun)."""
    if world <= 1:
        return None
    import torch
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29517")
    if backend == "nccl":
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    else:
        dist.init_process_group(backend)
    return dist


def max_over_ranks(x: float, dist, device="cpu") -> float:
    """Device time of the job = the slowest rank's."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, step_bytes: int, ms_step: float) -> float:
    """Replicas only: every rank moves step_bytes per step; GB/s of the whole job."""
    return world * step_bytes / (ms_step * 1e-3) / 1e9


# ------------------------------------------------------------------------------------ main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the per-config table (cfg1/cfg5 latency, cfg2 warm/cold)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--latency-replays", type=int, default=10000)
    ap.add_argument("--probe", type=int, default=0, choices=[0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 11, 12, 13, 14],
                    help="run ONLY BASELINE.json config N (1-5) eagerly for --steps iterations, or one of the widenings "
                         "(6 = NEXT-4 latency, 7 = NEXT-1 dynamic, 8 = NEXT-3 top-k, 9 = HBM streaming ceilings, "
                         "11 = misaligned segments, 12 = NEXT-2 ReduceCopy variants + per-CTA ceiling, "
                         "13 = top-k at PAPER.md Table 3's decode shapes, 14 = R > 256 small messages): the commands "
                         "ncu captures are taken from")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    config = {"workload": "cfg3 MoE dispatch+combine AllToAllv (R=64, 16384 tok x 5120 bf16, Zipf 1.1) + cfg2 AllReduce "
                          "(R=8, 4Mi bf16) + cfg4 ReduceScatter (R=16, 256Mi bf16/rank); BASELINE.json configs[2],[1],[3]",
              "bytes_per_step_GiB": 48.625, "l2": "inputs larger than L2 (48.6 GiB touched per step vs 126 MB)",
              "launch": "one CUDA-graph replay per step (the four calls captured once; counts re-read on the device at every replay)",
              "parallelism": f"replicas x{world} (path does not shard across GPUs)"}

    if args.impl == "reference":
        if rank != 0:
            return 0
        cb, dt = run_oracle_leg(args.steps, args.warmup)
        line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": "GB/s", "n_gpus": args.gpus,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(dt * 1e3, 2), "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": dict(config, launch="CPU oracle, no GPU", sample_run_per_step=cb["sample"]),
                "cpu_baseline": cb,
                "e2e": {"value": cb["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    import torch
    import paper_2510_20171_b200 as nx

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = init_dist(world, local_rank, "nccl")
    nx.ncclx_init(128, local_rank)
    peak, peak_src = measured_peak()

    if args.probe:
        return probe(args, torch, nx, peak)

    a3 = A2A(W.a2a_config(3), torch, nx)
    r2 = Reduce(W.reduce_config(2), torch, nx)
    r4 = Reduce(W.reduce_config(4), torch, nx)
    step_bytes = 2 * 2 * a3.bytes_one_way + r2.bytes + r4.bytes
    assert config["bytes_per_step_GiB"] == round(step_bytes / GiB, 3)

    def step():
        a3.dispatch(); a3.combine(); r2.run(); r4.run()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    barrier()
    # sanity outside the timed region: the combine must have restored every send buffer (round trip = identity)
    assert all(torch.equal(b[:n], s[:n]) for b, s, n in zip(a3.back, a3.send, a3.send_elems)), "round trip broken"
    assert torch.equal(a3.C2, a3.C) and torch.equal(a3.RC, a3.C.t().contiguous())

    # The whole step is captured ONCE into a CUDA graph and every timed step is one replay (BASELINE.json configs[2]:
    # "counts device-resident, call captured in a CUDA graph"): the kernels re-read the device-resident
    # counts at every replay.  Profiling is off here: nothing but the graph launches sits in the timed region.
    nx.ncclx_set_param(nx.PARAM_PROFILE, 0)
    l0 = nx.ncclx_launch_count()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        step()
    launches_per_step = nx.ncclx_launch_count() - l0          # captured launches are counted once, at capture
    for b in a3.back:                                          # the replay itself has to restore these
        b.zero_()
    graph.replay()
    barrier()
    assert all(torch.equal(b[:n], s[:n]) for b, s, n in zip(a3.back, a3.send, a3.send_elems)), "round trip broken (graph replay)"
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        graph.replay()
    e1.record()
    barrier()
    launches = launches_per_step * args.steps
    clocks = sampler.stop()
    ms_total = e0.elapsed_time(e1)

    # Second pass, reported separately: the same K steps launched eagerly with the library's per-launch CUDA events on
    # (the events cannot sit inside a captured graph), for the per-kernel split and the dominant kernel's average
    # launch duration.
    nx.ncclx_profile_reset()
    nx.ncclx_set_param(nx.PARAM_PROFILE, 1)
    barrier()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    for _ in range(args.steps):
        step()
    p1.record()
    barrier()
    ms_profiled_total = p0.elapsed_time(p1)
    nx.ncclx_set_param(nx.PARAM_PROFILE, 0)
    copy_ms, copy_n = nx.ncclx_profile_read(nx.KERNEL_COPY)
    red_ms, red_n = nx.ncclx_profile_read(nx.KERNEL_REDUCE)
    cnt_ms, cnt_n = nx.ncclx_profile_read(nx.KERNEL_COUNTS)
    nx.ncclx_profile_reset()

    ms_total = max_over_ranks(ms_total, dist, "cuda")
    ms_step = ms_total / args.steps
    value = whole_job_value(world, step_bytes, ms_step)

    copy_avg_ms = copy_ms / max(copy_n, 1)
    copy_gbs = 2 * a3.bytes_one_way / (copy_avg_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "segment_copy_kernel", "achieved": round(copy_gbs, 1), "peak": peak,
                "unit": "GB/s", "frac": round(copy_gbs / peak, 4), "peak_source": peak_src,
                "frac_of_nominal_8TBps": round(copy_gbs / NOMINAL_HBM_GBS, 4),
                "algorithmic_bytes_per_launch": 2 * a3.bytes_one_way, "avg_launch_ms": round(copy_avg_ms, 4),
                "launches_timed": copy_n, "share_of_step": round(copy_ms / ms_profiled_total, 4),
                "timed_in": "second pass: the same steps launched eagerly with per-launch CUDA events (headline pass = graph replays, no events)",
                "per_kernel_pass_ms_per_step": round(ms_profiled_total / args.steps, 4),
                "traffic": None,
                "other_kernels": {"reduce_kernel": {"avg_ms": round(red_ms / max(red_n, 1), 4), "launches": red_n,
                                                    "share_of_step": round(red_ms / ms_profiled_total, 4)},
                                  "counts_kernel": {"avg_ms": round(cnt_ms / max(cnt_n, 1), 5), "launches": cnt_n,
                                                    "share_of_step": round(cnt_ms / ms_profiled_total, 5)}}}
    # dram bytes per launch from the committed ncu capture: profiles/traffic.csv is written from the capture's raw page
    # by `python -m paper_2510_20171_b200.ncu_traffic` (profiles/r3_summary.md section 2; ncu cannot run in this process)
    tr = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tr):
        try:
            import csv
            for row in csv.DictReader(open(tr)):
                if row["kernel"] == "segment_copy_kernel" and row["workload"] == "cfg3_dispatch":
                    roofline["traffic"] = int(row["bytes_per_launch"])
                    roofline["traffic_source"] = row["source"]
        except Exception:
            pass

    line = {"metric": METRIC, "value": round(value, 1), "unit": "GB/s", "n_gpus": world, "steps": args.steps,
            "warmup": warmup, "ms_per_step": round(ms_step, 4), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic", "config": config, "clocks": clocks,
            "gpu_launches": int(launches), "roofline": roofline,
            "frac_of_measured_peak": round(value / world / peak, 4),
            "frac_of_nominal_8TBps": round(value / world / NOMINAL_HBM_GBS, 4)}

    # ---- per-config table (rank 0, N=1 only): the five BASELINE.json configs one by one --------------------
    if rank == 0 and world == 1 and not args.no_extras:
        per = {}
        t = event_times_ms(torch, a3.dispatch, 10)
        per["cfg3_dispatch"] = {"ms_median": round(float(np.median(t)), 4), "ms_min": round(float(t.min()), 4),
                                **frac(2 * a3.bytes_one_way / (np.median(t) * 1e-3) / 1e9, peak)}
        t = event_times_ms(torch, a3.combine, 10)
        per["cfg3_combine"] = {"ms_median": round(float(np.median(t)), 4), "ms_min": round(float(t.min()), 4),
                               **frac(2 * a3.bytes_one_way / (np.median(t) * 1e-3) / 1e9, peak)}
        t = event_times_ms(torch, r4.run, 10)
        per["cfg4_reducescatter"] = {"ms_median": round(float(np.median(t)), 4), "ms_min": round(float(t.min()), 4),
                                     **frac(r4.bytes / (np.median(t) * 1e-3) / 1e9, peak)}
        # config 2 is a ~20 us kernel: an eager launch bracketed by events mostly measures launch latency, so
        # (like configs 1 and 5) it is timed as CUDA-graph replays.  cold = 6 rotating 128 MiB buffer sets
        # (768 MiB > L2) captured back to back; warm = the same set 6 times (footprint ~ L2 size).
        for label, sets in (("cfg2_allreduce_cold", 6), ("cfg2_allreduce_warm_L2", 1)):
            r2c = Reduce(W.reduce_config(2), torch, nx, sets=sets)
            for i in range(6):
                r2c.run(i)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                for i in range(6):
                    r2c.run(i)
            t = event_times_ms(torch, g.replay, 200, warm=10) / 6.0
            per[label] = {"calls_per_replay": 6, "replays": 200, "us_per_call_p50": round(float(np.percentile(t, 50)) * 1e3, 2),
                          "us_per_call_p99": round(float(np.percentile(t, 99)) * 1e3, 2),
                          **frac(r2.bytes / (np.percentile(t, 50) * 1e-3) / 1e9, peak)}
            del r2c, g
        for idx, reps in ((1, 1000), (5, args.latency_replays)):
            a = A2A(W.a2a_config(idx), torch, nx, with_back=False)
            a.dispatch(); torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                a.dispatch()
            t = event_times_ms(torch, g.replay, reps, warm=20)
            p50 = float(np.percentile(t, 50))
            # cross-check: the same number of replays back to back under ONE event pair, total / replays
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(reps):
                g.replay()
            e1.record()
            torch.cuda.synchronize()
            per[f"cfg{idx}_graph_replay"] = {"replays": reps, "p50_us": round(p50 * 1e3, 2), "p99_us": round(float(np.percentile(t, 99)) * 1e3, 2),
                                             "mean_us": round(float(t.mean()) * 1e3, 2),
                                             "total_over_replays_us": round(e0.elapsed_time(e1) / reps * 1e3, 2),
                                             "bytes_each_way": a.bytes_one_way,
                                             **frac(2 * a.bytes_one_way / (p50 * 1e-3) / 1e9, peak)}
            del a, g
        lr = min(args.latency_replays, 2000)
        per["next1_alltoallv_dynamic_R64_tok256"] = dynamic_extra(torch, nx, peak, lr)
        per["next2_reducecopy_cta_sweep"] = reducecopy_extra(torch, nx, peak)
        per["next3_topk_R64_T4096_k4"] = topk_extra(torch, nx, peak)
        per["next3_topk_table3_shapes"] = topk_table3_extra(torch, nx, peak, min(lr, 500))
        per["next4_latency"] = latency_extra(torch, nx, peak, lr)
        per["large_R_small_messages"] = large_r_extra(torch, nx, peak, min(lr, 500))
        per["misaligned_segments"] = misaligned_extra(torch, nx, peak)
        per["cfg4_shape_other_dtypes"] = reduce_dtype_extra(torch, nx, peak)
        per["hbm_ceiling_probe"] = ceiling_extra(torch, nx, peak)
        roofline["practical_ceiling_GBps"] = {k: per["hbm_ceiling_probe"][k]["GBps"] for k in ("read_only", "write_only", "copy")}
        line["per_config"] = per
        # the five BASELINE.json configs in compact form, also inside `roofline` (a key the driver's record keeps whole):
        # us p50/p99 for the latency configs, GB/s + both roofline fractions for the bandwidth configs
        c1, c5 = per["cfg1_graph_replay"], per["cfg5_graph_replay"]
        c2 = per["cfg2_allreduce_cold"]
        summary = {
            "cfg1_us_p50": c1["p50_us"], "cfg1_us_p99": c1["p99_us"],
            "cfg2_us_per_call_p50": c2["us_per_call_p50"], "cfg2_us_per_call_p99": c2["us_per_call_p99"],
            "cfg2_GBps": c2["GBps"], "cfg2_frac_nominal": c2["frac_of_nominal_8TBps"],
            "cfg3_dispatch_GBps": per["cfg3_dispatch"]["GBps"], "cfg3_dispatch_frac_nominal": per["cfg3_dispatch"]["frac_of_nominal_8TBps"],
            "cfg3_dispatch_frac_measured": per["cfg3_dispatch"]["frac_of_measured"],
            "cfg3_combine_GBps": per["cfg3_combine"]["GBps"],
            "cfg4_GBps": per["cfg4_reducescatter"]["GBps"], "cfg4_frac_nominal": per["cfg4_reducescatter"]["frac_of_nominal_8TBps"],
            "cfg4_frac_measured": per["cfg4_reducescatter"]["frac_of_measured"],
            "cfg5_us_p50": c5["p50_us"], "cfg5_us_p99": c5["p99_us"], "cfg5_us_total_over_replays": c5["total_over_replays_us"],
            "cfg5_GBps": c5["GBps"], "cfg5_frac_nominal": c5["frac_of_nominal_8TBps"],
            "next1_dynamic_us_p50": per["next1_alltoallv_dynamic_R64_tok256"]["p50_us"],
            "next1_dynamic_frac_nominal": per["next1_alltoallv_dynamic_R64_tok256"]["frac_of_nominal_8TBps"],
            "misaligned_odd_bf16_GBps": per["misaligned_segments"]["R16_bf16_odd_counts"]["GBps"],
            "misaligned_odd_u8_GBps": per["misaligned_segments"]["R16_u8_odd_counts"]["GBps"],
            "topk_dispatch_ms": per["next3_topk_R64_T4096_k4"]["dispatch"]["ms"],
            "topk_combine_ms": per["next3_topk_R64_T4096_k4"]["combine"]["ms"],
        }
        roofline["configs"] = summary

    # ---- e2e: same step through the host-buffer C ABI (H2D + kernels + D2H inside the timed region) --------
    if not args.no_e2e:
        line["e2e"] = run_e2e(torch, nx, a3, r2, r4, step_bytes, world, dist, min(args.steps, 3))

    # ---- CPU oracle baseline on the host cores (rank 0, N=1 only) --------------------------------------------
    if rank == 0 and world == 1 and not args.no_cpu:
        cb, _ = run_oracle_leg(2, 1)
        line["cpu_baseline"] = cb

    if rank == 0:
        if "configs" in roofline:
            line["configs_summary"] = roofline["configs"]       # last key: survives a truncated stdout tail
        print(json.dumps(line))
    nx.ncclx_finalize()
    if dist is not None:
        dist.destroy_process_group()
    return 0


def dynamic_extra(torch, nx, peak, reps):
    """the paper's full AllToAllvDynamic interface on an inference-shaped MoE dispatch
    (R=64, 256 tokens x 5120 bf16 per rank, 128 experts + one redundant hot expert), CUDA-graph replays; and two such
    calls (two layers) back to back: stream order vs double-buffered in two plan slots (L483)."""
    Ls, idx, bl, J = W.dynamic_moe_metadata()
    R, n = Ls.shape
    nx.ncclx_init_dynamic(n, R * R * J)
    tot = Ls.sum(axis=1)

    def problem(seed):
        send = [W.torch_values(int(t), "bf16", seed + s) for s, t in enumerate(tot)]
        recv = [torch.empty(int(tot[s]), dtype=torch.bfloat16, device="cuda") for d in range(R) for s in range(R)]
        return {"send": send, "recv": recv, "st": nx.device_ptr_table(send), "rt": nx.device_ptr_table(recv),
                "all": torch.empty((R, R, n), dtype=torch.int64, device="cuda")}
    A, B = problem(5000), problem(5100)
    Ld, Id, Bd = (torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in (Ls, idx, bl))
    side = torch.cuda.Stream()

    def call(p=A):
        nx.ncclx_alltoallv_dynamic_dev(p["st"], Ld, n, Id, idx.shape[1], Bd, J, p["rt"], p["all"], R, "bf16")

    def prep(slot, p):
        nx.ncclx_alltoallv_dynamic_prepare_dev(slot, p["st"], Ld, n, Id, idx.shape[1], Bd, J, p["rt"], p["all"], R, "bf16")

    def pair_plain():
        call(A); call(B)

    def pair_double_buffered():
        main = torch.cuda.current_stream()
        prep(0, A)
        side.wait_stream(main)
        with torch.cuda.stream(side):
            prep(1, B)
        nx.ncclx_alltoallv_execute_dev(0)
        main.wait_stream(side)
        nx.ncclx_alltoallv_execute_dev(1)
    one = graph_p50(torch, call, reps)
    moved = 0
    for s_ in range(R):
        pos = 0
        for d in range(R):
            moved += int(Ls[s_, idx[s_, pos:pos + bl[s_, d]]].sum()) * 2
            pos += int(bl[s_, d])
    res = {"replays": reps, **one, "bytes_each_way": moved, "segments": int(bl.sum()),
           **frac(2 * moved / (one["p50_us"] * 1e-6) / 1e9, peak)}
    for name, fn in (("pair_stream_order", pair_plain), ("pair_double_buffered", pair_double_buffered)):
        r = graph_p50(torch, fn, reps)
        res[name] = {**r, **frac(4 * moved / (r["p50_us"] * 1e-6) / 1e9, peak)}
    return res


def topk_extra(torch, nx, peak, R=64, T=4096, k=4, width=5120):
    """top-k dispatch with duplication on the way + combine fused with the fixed-order sum,
    at config-3 scale (k*T = 16384 virtual rows per rank): dispatch reads T rows and writes k*T, combine the reverse."""
    pos, C = W.topk_routing(R, T, k, 128, seed=7)
    X = [W.torch_values(T * width, "bf16", 7000 + s) for s in range(R)]
    recv = [torch.empty(max(int(C[:, d].sum()), 1) * width, dtype=torch.bfloat16, device="cuda") for d in range(R)]
    Z = [torch.empty(T * width, dtype=torch.bfloat16, device="cuda") for _ in range(R)]
    dpos, dC = torch.from_numpy(pos).cuda(), torch.from_numpy(C).cuda()
    dRC = torch.empty_like(dC)
    xt, rt, zt = nx.device_ptr_table(X), nx.device_ptr_table(recv), nx.device_ptr_table(Z)
    rows = R * T * width * 2
    t = event_times_ms(torch, lambda: nx.ncclx_moe_dispatch_topk_dev(xt, dpos, dC, rt, dRC, R, T, k, width, "bf16"), 10)
    td = float(np.median(t))
    t = event_times_ms(torch, lambda: nx.ncclx_moe_combine_topk_sum_dev(rt, dpos, dC, zt, R, T, k, width, "bf16"), 10)
    tc = float(np.median(t))
    nbytes = (1 + k) * rows
    ok = all(torch.equal(z.float(), k * x.float()) for z, x in zip(Z[:4], X[:4]))    # identity experts: Z = k * X exactly
    return {"dispatch": {"ms": round(td, 4), **frac(nbytes / (td * 1e-3) / 1e9, peak)},
            "combine": {"ms": round(tc, 4), **frac(nbytes / (tc * 1e-3) / 1e9, peak)},
            "algorithmic_bytes_each": nbytes, "combine_of_dispatch_equals_k_times_x": bool(ok),
            "note": "unfused path would move 2*k*rows per direction plus the shuffle / the separate k-way sum"}


def reducecopy_extra(torch, nx, peak, few=(1, 2, 4), many=(8, 16, 32, 64, 148)):
    """FTAR-style ReduceCopy step: bf16 message, 8 MiB chunks, out + fwd
    written (4 x message bytes of traffic), as a function of the number of CTAs, for both inner loops
    (pipelined register loads / TMA-fed shared-memory ring); and, at 1 / 2 / 4 CTAs, the per-SM ceiling beside it:
    the streaming copy probe on the same fixed grid (1:1 read:write like the 2-read / 2-write step)."""
    n = 64 << 20                                   # 128 MiB message: a 1-CTA pass stays well under a second
    a = W.torch_values(n, "bf16", 6001)
    b = W.torch_values(n, "bf16", 6002, 1e-3)
    out, fwd = torch.empty_like(a), torch.empty_like(a)
    res = {"message_MiB": n * 2 >> 20, "chunk_MiB": 8, "by_ctas": {}}
    src8, dst8 = a.view(torch.uint8), out.view(torch.uint8)
    for ctas in few + many:
        row = {}
        for tma, name in ((0, "pipelined"), (1, "tma_ring")):
            nx.ncclx_set_param(nx.PARAM_REDUCECOPY_TMA, tma)
            t = event_times_ms(torch, lambda: nx.ncclx_reducecopy_sum(a, b, out, fwd, n, "bf16", 8 << 20, ctas), 5, warm=2)
            m = float(np.median(t))
            row[name] = {"ms": round(m, 3), "traffic_GBps": round(4 * n * 2 / (m * 1e-3) / 1e9, 1),
                         "message_GBps": round(n * 2 / (m * 1e-3) / 1e9, 1)}
        nx.ncclx_set_param(nx.PARAM_REDUCECOPY_TMA, 0)
        if ctas in few:
            t = event_times_ms(torch, lambda: nx.ncclx_stream_probe_ctas(2, src8, dst8, n * 2, ctas), 5, warm=2)
            m = float(np.median(t))
            row["copy_probe_ceiling_GBps"] = round(2 * n * 2 / (m * 1e-3) / 1e9, 1)
            best = max(row["pipelined"]["traffic_GBps"], row["tma_ring"]["traffic_GBps"])
            row["best_frac_of_ceiling"] = round(best / row["copy_probe_ceiling_GBps"], 3)
        res["by_ctas"][str(ctas)] = row
    return res


def ceiling_extra(torch, nx, peak, nbytes=4 << 30):
    """read-only / write-only / copy streaming micro-probe (256-bit accesses, one pass over 4 GiB,
    far beyond L2): the practical HBM ceilings the kernels' roofline fractions are read against."""
    src = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    dst = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    src.fill_(7)
    res = {"bytes": nbytes}
    for mode, name, moved in ((0, "read_only", nbytes), (1, "write_only", nbytes), (2, "copy", 2 * nbytes),
                              (3, "write_only_tma", nbytes)):
        t = event_times_ms(torch, lambda: nx.ncclx_stream_probe(mode, src, dst, nbytes), 10)
        res[name] = {"ms_median": round(float(np.median(t)), 4), **frac(moved / (np.median(t) * 1e-3) / 1e9, peak)}
    return res


def reduce_dtype_extra(torch, nx, peak):
    """Config 4's shape (R = 16 ReduceScatter, N(0, 1e-3)) in the other reduction dtypes, 4 GiB of input."""
    res = {}
    for dtype, es in (("f32", 4), ("f16", 2)):
        cfg = W.ReduceConfig(f"cfg4_shape_{dtype}", "reducescatter", 16, (4 << 30) // (16 * es), dtype, 3, 1e-3)
        r = Reduce(cfg, torch, nx)
        t = event_times_ms(torch, r.run, 10)
        res[dtype] = {"ms_median": round(float(np.median(t)), 4), "bytes": r.bytes, **frac(r.bytes / (np.median(t) * 1e-3) / 1e9, peak)}
        del r
    return res


def misaligned_extra(torch, nx, peak):
    """Element-granular counts ('s_i number of tokens'): segments whose source and destination are
    misaligned differently modulo 16 -- odd bf16 counts, odd byte counts -- against the same bytes 16B-aligned.
    R = 16, ~360 MB each way; every byte goes through the TMA ring either way."""
    rng = np.random.default_rng(0)
    res = {}
    for key, rows, width, dtype in (("R16_bf16_odd_counts", rng.integers(300000, 400000, (16, 16)) * 2 + 1, 1, "bf16"),
                                    ("R16_bf16_aligned_counts", rng.integers(75000, 100000, (16, 16)) * 8, 1, "bf16"),
                                    ("R16_bf16_aligned_counts_4x_bytes", rng.integers(300000, 400000, (16, 16)) * 8, 1, "bf16"),
                                    ("R16_bf16_odd_counts_4x_bytes", rng.integers(1200000, 1600000, (16, 16)) * 2 + 1, 1, "bf16"),
                                    ("R16_u8_odd_counts", rng.integers(600000, 800000, (16, 16)) * 2 + 1, 1, "u8"),
                                    ("R64_bf16_odd_rows_of_5121", np.ones((64, 64), np.int64) * 41, 5121, "bf16")):
        a = A2A(W.A2AConfig(key, rows.shape[0], width, dtype, 1, rows.astype(np.int64)), torch, nx, with_back=False)
        t = event_times_ms(torch, a.dispatch, 10)
        m = float(np.median(t))
        res[key] = {"MB_each_way": round(a.bytes_one_way / 1e6, 1), "ms": round(m, 4), **frac(2 * a.bytes_one_way / (m * 1e-3) / 1e9, peak)}
        del a
    res["odd_bf16_over_aligned"] = round(res["R16_bf16_odd_counts"]["GBps"] / res["R16_bf16_aligned_counts"]["GBps"], 3)
    return res


def topk_table3_extra(torch, nx, peak, reps, shapes=None):
    """PAPER.md Table 3 (L493-516): decode-shaped MoE layer, k in {1, 4}, 128 / 256 tokens per rank, hidden 5120 bf16,
    R in {32, 64, 128}: dispatch -> combine replayed in ONE CUDA graph.  (a) top-k calls, one-call form (each runs its own
    metadata kernel); (b) plan-slot form (one metadata kernel per layer, the combine reuses the dispatch's offsets);
    (c) the plain AllToAllv pair on the same bytes with the k*T copies materialised by the caller."""
    width = 5120
    res = {}
    for R, T, k in (shapes or [(R, T, k) for R in (32, 64, 128) for T in (128, 256) for k in (1, 4)]):
        pos, C = W.topk_routing(R, T, k, 2 * R, seed=R + T + k)
        X = [W.torch_values(T * width, "bf16", 9000 + s) for s in range(R)]
        recv = [torch.empty(max(int(C[:, d].sum()), 1) * width, dtype=torch.bfloat16, device="cuda") for d in range(R)]
        Z = [torch.empty(T * width, dtype=torch.bfloat16, device="cuda") for _ in range(R)]
        dpos, dC = torch.from_numpy(pos).cuda(), torch.from_numpy(C).cuda()
        dRC = torch.empty_like(dC)
        xt, rt, zt = nx.device_ptr_table(X), nx.device_ptr_table(recv), nx.device_ptr_table(Z)

        def one_call():
            nx.ncclx_moe_dispatch_topk_dev(xt, dpos, dC, rt, dRC, R, T, k, width, "bf16")
            nx.ncclx_moe_combine_topk_sum_dev(rt, dpos, dC, zt, R, T, k, width, "bf16")

        def planned():
            nx.ncclx_moe_topk_prepare_dev(1, dC, dRC, R)
            nx.ncclx_moe_dispatch_topk_execute_dev(1, xt, dpos, rt, T, k, width, "bf16")
            nx.ncclx_moe_combine_topk_sum_execute_dev(1, rt, dpos, zt, T, k, width, "bf16")
        # plain AllToAllv on the materialised k*T rows (what a caller without the top-k calls would move)
        Cel = C * width
        mat = A2A(W.A2AConfig("mat", R, width, "bf16", 1, C), torch, nx, with_back=True)

        def plain_pair():
            mat.dispatch(); mat.combine()
        row = {"one_call": graph_p50(torch, one_call, reps), "plan_slot": graph_p50(torch, planned, reps),
               "plain_alltoallv_pair_materialised": graph_p50(torch, plain_pair, reps),
               "bytes_topk_pair": 2 * (1 + k) * R * T * width * 2, "bytes_plain_pair": 4 * int(Cel.sum()) * 2}
        ok = all(torch.equal(z.float(), k * x.float()) for z, x in zip(Z[:2], X[:2]))
        row["combine_of_dispatch_equals_k_times_x"] = bool(ok)
        res[f"R{R}_T{T}_k{k}"] = row
        del mat, X, recv, Z
    return res


def large_r_extra(torch, nx, peak, reps):
    """R > 256 (the coarse index of the descriptor table no longer fits the copy kernel's 16 KB of shared memory:
    claims locate their segment with the 128-ary search in L2): small-message shapes, one 14 KB row for ~30 % of the
    pairs, against R = 128 (the T_c*(N-1) term grows with the rank count)."""
    res = {}
    nx.ncclx_finalize()
    nx.ncclx_init(1024, torch.cuda.current_device())
    for R in (128, 256, 512, 1024):
        rng = np.random.default_rng(R)
        rows = (rng.random((R, R)) < 0.3).astype(np.int64)
        w = A2A(W.A2AConfig(f"R{R}", R, 7168, "bf16", 1, rows), torch, nx, with_back=False)
        r = graph_p50(torch, w.dispatch, reps)
        res[f"R{R}"] = {"pairs": int(rows.sum()), "bytes_each_way": w.bytes_one_way, **r,
                        **frac(2 * w.bytes_one_way / (r["p50_us"] * 1e-6) / 1e9, peak)}
        del w
    nx.ncclx_finalize()
    nx.ncclx_init(128, torch.cuda.current_device())
    return res


def graph_p50(torch, enqueue, reps, warm=20):
    """Capture `enqueue` once (after one eager run on a side stream), time `reps` replays with CUDA events."""
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        enqueue()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        enqueue()
    t = event_times_ms(torch, g.replay, reps, warm=warm)
    return {"p50_us": round(float(np.percentile(t, 50)) * 1e3, 2), "p99_us": round(float(np.percentile(t, 99)) * 1e3, 2)}


def latency_extra(torch, nx, peak, reps):
    """(a) config 1 as ONE fused kernel vs the two-kernel path;
    (b) dispatch + combine back to back (the MoE layer's two consecutive AllToAlls): plain stream order vs the
    split-phase form with two plan slots, where the combine's metadata phase runs beside the dispatch's payload."""
    res = {}
    x = torch.zeros(32, device="cuda")
    # context: what ANY one-kernel graph replay costs between two CUDA events on this box (a 32-element torch add)
    res["floor_one_tiny_kernel_graph"] = graph_p50(torch, lambda: x.add_(1), reps)
    a1 = A2A(W.a2a_config(1), torch, nx, with_back=True)

    def pair1():
        a1.dispatch(); a1.combine()
    res["cfg1_one_kernel"] = graph_p50(torch, a1.dispatch, reps)
    res["cfg1_pair_one_kernel_each"] = graph_p50(torch, pair1, reps)
    nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, 0)
    res["cfg1_two_kernels"] = graph_p50(torch, a1.dispatch, reps)
    res["cfg1_pair_two_kernels_each"] = graph_p50(torch, pair1, reps)
    nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, 32)
    del a1
    a5 = A2A(W.a2a_config(5), torch, nx, with_back=True)
    side = torch.cuda.Stream()

    def pair_plain():
        a5.dispatch(); a5.combine()

    def pair_double_buffered():
        main = torch.cuda.current_stream()
        nx.ncclx_alltoallv_prepare_dev(0, a5.st, a5.C, a5.rt, a5.RC, a5.R, a5.cfg.dtype)
        side.wait_stream(main)
        with torch.cuda.stream(side):
            nx.ncclx_alltoallv_prepare_dev(1, a5.rt, a5.RC, a5.bt, a5.C2, a5.R, a5.cfg.dtype)
        nx.ncclx_alltoallv_execute_dev(0)
        main.wait_stream(side)
        nx.ncclx_alltoallv_execute_dev(1)
    # the paper's inference regime (L90, L471: a few MB per operation, < 128 KB per peer): one row per pair
    for name, rows, width in (("R64_one_10KB_row_per_pair", np.ones((64, 64), np.int64), 5120),
                              ("R128_one_14KB_row_for_28pct_of_pairs", (a5.cfg.rows > 4).astype(np.int64), 7168)):
        w = A2A(W.A2AConfig(name, rows.shape[0], width, "bf16", 1, rows), torch, nx, with_back=False)
        r = {"bytes_each_way": w.bytes_one_way, "engines_chosen_on_device": graph_p50(torch, w.dispatch, reps)}
        nx.ncclx_set_param(nx.PARAM_COPY_BULK_ENGINES, 1)
        r["one_engine"] = graph_p50(torch, w.dispatch, reps)
        nx.ncclx_set_param(nx.PARAM_COPY_BULK_ENGINES, 0)
        res["small_" + name] = r
        del w
    res["cfg5_pair_stream_order"] = graph_p50(torch, pair_plain, reps)
    res["cfg5_pair_double_buffered"] = graph_p50(torch, pair_double_buffered, reps)
    ok = all(bool((a5.back[s][:n] == a5.send[s][:n]).all()) for s, n in enumerate(a5.send_elems) if n)
    res["cfg5_pair_roundtrip_identity"] = ok
    res["cfg5_pair_bytes"] = 4 * a5.bytes_one_way
    for k in ("cfg5_pair_stream_order", "cfg5_pair_double_buffered"):
        res[k].update(frac(4 * a5.bytes_one_way / (res[k]["p50_us"] * 1e-6) / 1e9, peak))
    return res


def probe(args, torch, nx, peak):
    """One config, eager launches, CUDA-event time per call (the command ncu captures are taken from)."""
    n = args.probe
    if n >= 6:
        res = (latency_extra(torch, nx, peak, args.steps) if n == 6 else
               dynamic_extra(torch, nx, peak, args.steps) if n == 7 else
               topk_extra(torch, nx, peak) if n == 8 else
               ceiling_extra(torch, nx, peak) if n == 9 else
               misaligned_extra(torch, nx, peak) if n == 11 else
               reducecopy_extra(torch, nx, peak) if n == 12 else
               topk_table3_extra(torch, nx, peak, args.steps) if n == 13 else
               large_r_extra(torch, nx, peak, args.steps))
        names = {6: "next4_latency", 7: "next1_dynamic", 8: "next3_topk", 9: "hbm_ceiling", 11: "misaligned",
                 12: "next2_reducecopy", 13: "next3_topk_table3", 14: "large_R"}
        print(json.dumps({"probe": names[n], **res}))
        nx.ncclx_finalize()
        return 0
    if n in (1, 3, 5):
        w = A2A(W.a2a_config(n), torch, nx, with_back=False)
        fn, nbytes = w.dispatch, 2 * w.bytes_one_way
    else:
        w = Reduce(W.reduce_config(n), torch, nx, sets=6 if n == 2 else 1)
        it = [0]

        def fn():
            w.run(it[0]); it[0] += 1
        nbytes = w.bytes
    t = event_times_ms(torch, fn, args.steps, warm=max(args.warmup, 3))
    print(json.dumps({"probe": f"cfg{n}", "calls": args.steps, "us_median": round(float(np.median(t)) * 1e3, 2),
                      "us_min": round(float(t.min()) * 1e3, 2), **frac(nbytes / (np.median(t) * 1e-3) / 1e9, peak)}))
    nx.ncclx_finalize()
    return 0


def run_e2e(torch, nx, a3, r2, r4, step_bytes, world, dist, steps):
    """Host-buffer step: pinned host inputs -> ncclx_*_host (H2D, kernels, D2H, sync) -> pinned host outputs."""
    import psutil
    R3 = a3.R
    need = 3 * a3.bytes_one_way + r4.cfg.R * r4.cfg.count * 2 + r4.n_out * r4.cfg.R * 2 + 2 * r2.cfg.R * r2.cfg.count * 2
    avail = psutil.virtual_memory().available
    try:
        lim = int(open("/sys/fs/cgroup/memory.max").read())
        cur = int(open("/sys/fs/cgroup/memory.current").read())
        avail = min(avail, lim - cur)
    except Exception:
        pass
    if need * world > 0.6 * avail:
        return {"value": None, "unit": "GB/s", "skipped": f"needs {need * world / GiB:.0f} GiB pinned host memory, {avail / GiB:.0f} GiB available"}

    def pin_like(ts, elems):
        return [torch.empty(max(n, 8), dtype=t.dtype).pin_memory() for t, n in zip(ts, elems)]

    h_send = pin_like(a3.send, a3.send_elems)
    for h, d in zip(h_send, a3.send):
        h.copy_(d)
    h_recv = pin_like(a3.recv, a3.recv_elems)
    h_back = pin_like(a3.back, a3.send_elems)
    C = np.ascontiguousarray(a3.C_host)
    RC = np.zeros_like(C)
    C2 = np.zeros_like(C)
    x2, y2 = r2.sets[0][0], r2.sets[0][1]
    x4, y4 = r4.sets[0][0], r4.sets[0][1]
    hx2 = [t.cpu().pin_memory() for t in x2]
    hy2 = [torch.empty_like(t, device="cpu").pin_memory() for t in y2]
    hx4 = [t.cpu().pin_memory() for t in x4]
    hy4 = [torch.empty_like(t, device="cpu").pin_memory() for t in y4]
    # free the device-resident copies: the host path stages through the library's own device buffers
    h2d = 2 * a3.bytes_one_way + r2.cfg.R * r2.cfg.count * 2 + r4.cfg.R * r4.cfg.count * 2 + 2 * C.nbytes
    d2h = 2 * a3.bytes_one_way + r2.cfg.R * r2.cfg.count * 2 + r4.cfg.R * r4.n_out * 2 + 2 * C.nbytes

    def estep():
        nx.ncclx_alltoallv_host(h_send, C, h_recv, RC, R3, "bf16")
        nx.ncclx_alltoallv_host(h_recv, RC, h_back, C2, R3, "bf16")
        nx.ncclx_allreduce_sum_host(hx2, hy2, r2.cfg.count, r2.cfg.R, "bf16")
        nx.ncclx_reducescatter_sum_host(hx4, hy4, r4.n_out, r4.cfg.R, "bf16")

    estep()
    torch.cuda.synchronize()
    ok = all(torch.equal(b[:n], s[:n]) for b, s, n in zip(h_back, h_send, a3.send_elems)) and (C2 == C).all()
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        estep()
    torch.cuda.synchronize()
    dt = max_over_ranks(time.perf_counter() - t0, dist, "cuda")
    # A/B: the same step with the kernels' direct access to pinned host memory switched off (device staging)
    staged_ms = None
    if world == 1:
        nx.ncclx_set_param(nx.PARAM_HOST_ZERO_COPY, 0)
        estep()
        t1 = time.perf_counter()
        estep()
        staged_ms = (time.perf_counter() - t1) * 1e3
        nx.ncclx_set_param(nx.PARAM_HOST_ZERO_COPY, 1)
    return {"value": round(whole_job_value(world, step_bytes, dt / steps * 1e3), 2), "unit": "GB/s", "steps": steps,
            "ms_per_step": round(dt / steps * 1e3, 2), "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
            "roundtrip_identity": bool(ok), "api": "ncclx_alltoallv_host x2 + ncclx_allreduce_sum_host + ncclx_reducescatter_sum_host",
            "transport": "pinned host buffers: AllToAllv and AllReduce kernels read/write host memory directly over PCIe "
                         "(both directions at once); ReduceScatter staged through device memory",
            "ms_per_step_all_staged": None if staged_ms is None else round(staged_ms, 2)}


if __name__ == "__main__":
    sys.exit(main())
