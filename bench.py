#!/usr/bin/env python
"""bench.py -- whole-solve throughput of the Cross-DEIM low-rank Poisson hot path on B200 (BASELINE.json metric:
effective DOF/s = n^2 / t_solve at 1 GPU; batched DST-I GB/s vs the HBM peak).

    python bench.py --gpus N --steps K --warmup W [--impl reference] [--workload C4]

A step = one pass of the whole hot path (forward DST-I of the RHS factors, all Cross-DEIM sweeps, inverse DST-I)
over one synthetic right-hand side.  Workload: config C4 of BASELINE.json (n = 2^20 - 1, rank-32 smooth random
factors), the size north_star quotes the end-to-end figure on.  N > 1: N independent replicas (one process per GPU,
different seeds, no data-path collective), launched by torchrun.
Prints ONE JSON line on rank 0.
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

from paper_2607_06021_b200 import replicas as R          # noqa: E402
from paper_2607_06021_b200 import workloads as W         # noqa: E402

METRIC = "Cross-DEIM Poisson solve: effective DOF/s (n^2/s)"
UNIT = "DOF/s"
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 148 SMs x 64 DFMA/clk x 2 flop x 1965 MHz
CPU_SAMPLE_N = (1 << 14) - 1                          # oracle sample: same recipe at n = 16383


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (profiling recipe's clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "25"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for nme, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nme)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_step(w):
    from oracle import lrp_oracle as O                  # the oracle arm: cpu_baseline / --impl reference only
    t0 = time.perf_counter()
    r = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, **w.opts())
    return time.perf_counter() - t0, r


def cpu_threads() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank, _, world = R.env_world()
    if rank != 0:
        return 0
    w = W.make(args.workload, 0, CPU_SAMPLE_N)
    for _ in range(args.warmup):
        oracle_step(w)
    ts = [oracle_step(w)[0] for _ in range(args.steps)]
    ms = 1e3 * float(np.mean(ts))
    val = float(w.n) ** 2 / (ms * 1e-3)
    sample = f"oracle (numpy fp64) full solve of the {args.workload} recipe at n={w.n} per step"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload} recipe, bounded CPU sample n={w.n}", "l2": "n/a (CPU)"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--timeline", default="", help="also write the per-launch timeline (CSV) of one real multi-stream solve here")
    ap.add_argument("--dst-p", type=int, default=20, help="log2(n+1) of the batched DST-I side measurement")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2607_06021_b200 import build, lrp
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    rank, local_rank, world = R.env_world()
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    dist = R.init("nccl", dev)
    if rank == 0:
        build.build()
    R.barrier(dist)
    ctx = lrp.Context(local_rank)
    steps, warmup = max(args.steps, 1), max(args.warmup, 3)

    w = W.make(args.workload, seed=rank)
    n, rF = w.n, w.rF
    UF = lrp.tall_from_numpy(w.UF, dev); VF = lrp.tall_from_numpy(w.VF, dev); SF = torch.from_numpy(w.SF).to(dev)
    kw = dict(tol=w.tol, max_rank=w.max_rank, oversample=w.oversample, max_sweeps=w.max_sweeps, safeguard=w.safeguard)
    in_bytes = (UF.numel() + VF.numel() + SF.numel()) * 8

    def step():
        return ctx.cross_deim_solve(UF, SF, VF, **kw)

    for _ in range(warmup):
        res = step()
    # ---- timed region: K solves, device-resident inputs, CUDA events on the launching stream
    stream = torch.cuda.current_stream(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    clocks = ClockSampler(local_rank)
    R.barrier(dist); torch.cuda.synchronize(dev)
    clocks.start()
    l0 = ctx.launch_count()
    e0.record(stream)
    for _ in range(steps):
        res = step()
    e1.record(stream)
    torch.cuda.synchronize(dev); R.barrier(dist)
    launches = ctx.launch_count() - l0
    local_ms = e0.elapsed_time(e1)
    agg = R.throughput(dist, local_ms, float(n) ** 2 * steps, dev)
    clk = clocks.stop()

    # ---- end to end through the public call with HOST buffers (pinned), H2D + solve + D2H every step
    hUF = torch.from_numpy(np.ascontiguousarray(w.UF.T)).pin_memory(); hVF = torch.from_numpy(np.ascontiguousarray(w.VF.T)).pin_memory()
    hSF = torch.from_numpy(w.SF).pin_memory()
    hUW = torch.empty((w.max_rank, n), dtype=torch.float64).pin_memory(); hVW = torch.empty_like(hUW).pin_memory()
    hSW = torch.empty(w.max_rank, dtype=torch.float64).pin_memory()
    dUF, dVF, dSF = torch.empty_like(UF), torch.empty_like(VF), torch.empty_like(SF)
    d2h = 0

    def e2e_step():
        nonlocal d2h
        dUF.copy_(hUF, non_blocking=True); dVF.copy_(hVF, non_blocking=True); dSF.copy_(hSF, non_blocking=True)
        r = ctx.cross_deim_solve(dUF, dSF, dVF, **kw)
        k = r["rank"]
        hUW[:k].copy_(r["UW"], non_blocking=True); hVW[:k].copy_(r["VW"], non_blocking=True); hSW[:k].copy_(r["SW"], non_blocking=True)
        torch.cuda.synchronize(dev)
        d2h = (2 * n * k + k) * 8
    e2e_step()
    R.barrier(dist); torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    for _ in range(steps):
        e2e_step()
    torch.cuda.synchronize(dev)
    e2e_ms = 1e3 * (time.perf_counter() - t0)
    R.barrier(dist)
    agg_e2e = R.throughput(dist, e2e_ms, float(n) ** 2 * steps, dev)

    if args.timeline and rank == 0:                 # start/end of every launch of one solve, streams NOT serialised
        ctx.profile_reset(); ctx.profile_enable(2)
        step()
        ctx.profile_timeline(args.timeline)
        ctx.profile_enable(False); ctx.profile_reset()

    # ---- per-kernel profile (separate pass: events around every launch), roofline of the dominant kernel
    ctx.profile_reset(); ctx.profile_enable(True)
    nprof = 2
    for _ in range(nprof):
        step()
    prof = ctx.profile()
    ctx.profile_enable(False); ctx.profile_reset()
    hbm_peak, peak_src = measured_peaks()
    tot_ms = sum(v["ms"] for v in prof.values()) or 1.0
    kernels = []
    for name, v in sorted(prof.items(), key=lambda kv: -kv[1]["ms"]):
        ms = v["ms"]
        gbs = v["bytes"] / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
        tfl = v["flops"] / (ms * 1e-3) / 1e12 if ms > 0 else 0.0
        kernels.append({"kernel": name, "launches_per_step": v["count"] / nprof, "ms_per_step": ms / nprof,
                        "share": ms / tot_ms, "alg_GBps": gbs, "alg_TFLOPs": tfl})
    top = kernels[0]
    t_hbm = prof[top["kernel"]]["bytes"] / (hbm_peak * 1e9)
    t_alu = prof[top["kernel"]]["flops"] / (FP64_PEAK_TFLOPS * 1e12)
    if t_alu >= t_hbm:
        roof = {"bound": "alu", "achieved": top["alg_TFLOPs"], "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                "frac": top["alg_TFLOPs"] / FP64_PEAK_TFLOPS, "traffic": None, "peak_source": "derived: 148 SM x 64 DFMA/clk x 1965 MHz"}
    else:
        roof = {"bound": "hbm", "achieved": top["alg_GBps"], "peak": hbm_peak, "unit": "GB/s",
                "frac": top["alg_GBps"] / hbm_peak, "traffic": None, "peak_source": peak_src}
    roof["kernel"] = top["kernel"]; roof["share_of_step"] = top["share"]
    # measured DRAM traffic of that kernel class from the committed ncu capture (ratio to its algorithmic bytes), per launch
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "r01d_traffic.csv")) as fh:
            for row in csv.DictReader(fh):
                if row["kernel"] == top["kernel"]:
                    ratio = float(row["dram_bytes_per_launch"]) / float(row["alg_bytes_per_launch"])
                    v = prof[top["kernel"]]
                    roof["traffic"] = ratio * v["bytes"] / v["count"]
                    roof["alg_bytes_per_launch"] = v["bytes"] / v["count"]
                    roof["traffic_source"] = row["capture"]
    except Exception:
        pass

    # ---- batched DST-I side measurement (metric's second half): n = 2^p - 1, batch 128, buffers rotate beyond L2
    dst = None
    try:
        nd, bd = (1 << args.dst_p) - 1, 128
        xs = [torch.randn((bd, nd), dtype=torch.float64, device=dev) for _ in range(2)]
        ys = [torch.empty_like(xs[0]) for _ in range(2)]
        for i in range(3):
            ctx.dst1_batched(xs[i % 2], out=ys[i % 2])
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        reps = 10
        d0.record(stream)
        for i in range(reps):
            ctx.dst1_batched(xs[i % 2], out=ys[i % 2])
        d1.record(stream); torch.cuda.synchronize(dev)
        dms = d0.elapsed_time(d1) / reps
        gbs = 16.0 * nd * bd / (dms * 1e-3) / 1e9
        dst = {"n": nd, "batch": bd, "ms": dms, "alg_GBps": gbs, "frac_of_hbm_peak": gbs / hbm_peak, "peak": hbm_peak,
               "peak_source": peak_src, "alg_bytes": "16*n*batch (read once + write once)"}
        del xs, ys
    except Exception as ex:                       # never lose the main line because of the side measurement
        dst = {"error": str(ex)}

    # ---- the oracle timed beside it (rank 0, N = 1 only): bounded sample of the same recipe
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        ws_ = W.make(args.workload, 0, min(CPU_SAMPLE_N, n))
        t, _ = oracle_step(ws_)
        cpu = {"value": float(ws_.n) ** 2 / t, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle",
               "sample": f"one full oracle solve (numpy fp64) of the {args.workload} recipe at n={ws_.n}: {t:.1f} s"}

    if rank == 0:
        info = res["info"]
        line = {"metric": METRIC, "value": agg["per_s"], "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
                "ms_per_step": agg["ms"] / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"{w.name}: n={n}, rF={rF}, tol={w.tol}, max_rank={w.max_rank}, oversample={w.oversample}",
                           "l2": f"inputs larger than L2 ({in_bytes / 1e6:.0f} MB of factors re-read every step)",
                           "parallelism": f"{world} independent replica(s), no data-path collective"},
                "solve": {"rank": res["rank"], "sweeps": res["sweeps"], "converged": res["converged"],
                          "ms": {k: getattr(info, "ms_" + k) for k in ("dst_fwd", "select", "sample", "qr", "core", "rebuild", "stop", "dst_inv", "total")}},
                "clocks": clk,
                "e2e": {"value": agg_e2e["per_s"], "unit": UNIT, "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": d2h,
                        "ms_per_step": agg_e2e["ms"] / steps},
                "gpu_launches": int(launches),
                "roofline": roof, "kernels": kernels[:8], "dst1": dst, "cpu_baseline": cpu}
        print(json.dumps(line))
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
