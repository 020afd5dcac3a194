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
FP64_PEAK_DERIVED = 148 * 64 * 2 * 1.965e9 / 1e12     # fallback only: 148 SMs x 64 DFMA/clk x 2 flop x 1965 MHz; the run measures it
NOMINAL_N = {"C1": 255, "C2": 4095, "C3": 65535, "C4": (1 << 20) - 1, "C5": (1 << 22) - 1}
CPU_SAMPLE_N = (1 << 15) - 1                          # oracle sample: the same recipe at n = 32767 (the method is O(n) per solve)
CPU_SAMPLE_N_1T = (1 << 13) - 1                       # single-thread sample
L2_BYTES = 126e6


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return 6650.0, "fallback"


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def config_dict(name: str, n: int, rF: int, tol: float, max_rank: int, oversample: int, world: int, in_mb: float) -> dict:
    """The same dictionary in both arms (ours / --impl reference): it names the workload, not the implementation."""
    return {"workload": f"{name}: n={n}, rF={rF}, tol={tol}, max_rank={max_rank}, oversample={oversample}",
            "l2": f"inputs larger than L2 ({in_mb:.0f} MB of factors re-read every step)" if in_mb * 1e6 > L2_BYTES
                  else f"inputs of {in_mb:.1f} MB; a buffer larger than L2 is written between timed steps",
            "parallelism": f"{world} independent replica(s), no data-path collective"}


def solve_roofline(n, rF, trace, r_final, hbm_gbs, p64_tflops, ms_measured):
    """Solve-level floor of SURVEY.md 8(d): t_roof = sum over steps of max(algorithmic bytes / measured HBM rate,
    algorithmic flops / measured fp64 rate), with the per-step accounting of its table (what the METHOD must move and
    compute per sweep with the sets it used -- all K fibers sampled and factored, as Alg. 1 states; the driver's reuse
    of unchanged fibers, reading R4, is not credited to the floor).  Small-core and host steps are latency
    items and contribute nothing.  Returns the total, the fraction of the measured solve time and the split by phase."""
    BW, P = hbm_gbs * 1e9, p64_tflops * 1e12
    ph = {"dst": 0.0, "sampling": 0.0, "qr": 0.0, "rebuild": 0.0, "rho": 0.0, "leverage": 0.0}
    bound = {}

    def add(key, nbytes, flops):
        tb, tf = nbytes / BW, flops / P
        ph[key] += max(tb, tf)
        bound.setdefault(key, {"hbm": 0.0, "fp64": 0.0})["hbm" if tb >= tf else "fp64"] += max(tb, tf)

    add("dst", 16.0 * n * 2 * rF, 0.0)                                   # forward DST-I of both RHS factors
    add("dst", 16.0 * n * 2 * r_final, 0.0)                              # inverse DST-I of both solution factors
    r_prev = 0
    sel_cols = rF
    for t in trace:
        K_I, K_J, r = len(t["I"]), len(t["J"]), int(t["rank"])
        for K in (K_I, K_J):
            add("sampling", 8.0 * n * (rF + K), 2.0 * n * rF * K)        # read the factor, write K fibers; fused divide
            add("qr", 24.0 * n * K, 4.0 * n * K * K)                      # thin QR: R and explicit Q
            add("rebuild", 8.0 * n * (K + r), 2.0 * n * K * r)            # U = Q Uc (+ row norms in the epilogue)
            add("leverage", 16.0 * n, 0.0)                                # scores written once, read once by the top-k
        if r_prev > 0:
            for _ in range(2):
                add("rho", 8.0 * n * (r + r_prev), 5.0 * n * r * r)
        else:
            add("leverage", 2 * 8.0 * n * sel_cols, 2 * 4.0 * n * sel_cols * sel_cols)      # QR of the initial guess (k = 0)
        r_prev = r
    t_roof = sum(ph.values())
    return {"t_roof_ms": 1e3 * t_roof, "t_measured_ms": ms_measured, "frac": 1e3 * t_roof / ms_measured if ms_measured else None,
            "by_phase_ms": {k: 1e3 * v for k, v in ph.items()},
            "bound_by_phase": {k: max(v, key=v.get) for k, v in bound.items()},
            "peaks": {"hbm_GBps": hbm_gbs, "fp64_TFLOPs": p64_tflops},
            "accounting": "SURVEY.md 8(d) per-step table; latency-bound steps (small core, host set logic) count as 0"}


# dram__bytes_read.sum + dram__bytes_write.sum per launch over the algorithmic bytes of the same launch, from this round's
# `ncu --set full` captures (summaries with their commands under profiles/r02_*_ncu.md); None -> "traffic": null
_SRC = "profiles/r02_solve_ncu.md (ncu --set full, one C4 solve)"
NCU_TRAFFIC = {"panel_qr": {"dram_over_alg": 0.77, "source": _SRC}, "panel_apply": {"dram_over_alg": 0.81, "source": _SRC},
               "dst1_fused": {"dram_over_alg": 1.74, "source": _SRC + ", final-state addendum"}, "tall_gemm_t": {"dram_over_alg": 0.89, "source": _SRC},
               "tall_gemm_subtract": {"dram_over_alg": 0.97, "source": _SRC + ", all tall_gemm modes together"},
               "tall_gemm_plain": {"dram_over_alg": 0.97, "source": _SRC + ", all tall_gemm modes together"},
               "tall_gemm_sample": {"dram_over_alg": 0.97, "source": _SRC + ", all tall_gemm modes together"}}

# kernel class -> (phase, roofline SURVEY.md 8(d) assigns to it)
PHASE_OF = {"dst1_small": ("dst", "hbm"), "dst1_naive": ("dst", "hbm"), "dst1_fused": ("dst", "hbm"), "dst1_bluestein": ("dst", "hbm"),
            "tall_gemm_sample": ("sampling", "hbm"), "tall_gemm_plain": ("rebuild", "fp64"),
            "tall_gemm_subtract": ("qr", "fp64"), "tall_gemm_t": ("qr", "fp64"), "panel_qr": ("qr", "fp64"),
            "panel_apply": ("qr", "fp64"), "add_block": ("qr", "fp64"), "conditional_refactor": ("qr", "fp64"), "tall_resid_gram": ("rho", "fp64"),
            "rho": ("rho", "latency"), "eta": ("core", "latency"), "scross_core": ("core", "latency"),
            "rownorm2": ("leverage", "hbm"), "topk_chunk": ("leverage", "hbm"), "topk_merge": ("leverage", "latency"),
            "topk": ("leverage", "hbm"), "deim_step": ("leverage", "hbm"), "colmask": ("leverage", "latency"), "copy_tall": ("leverage", "hbm"),
            "gather_rows": ("core", "latency"), "lowrank_entries": ("core", "latency"), "reduce_partials": ("qr", "fp64")}


def phase_rooflines(prof, nprof, hbm_gbs, p64_tflops):
    """Per phase: serialised kernel time (events around every launch), the library's algorithmic bytes / flops of those
    launches, and the fraction of the roofline 8(d) assigns (fp64 pipe for QR / rebuild / rho, HBM for DST, sampling,
    leverage; latency items carry no roofline)."""
    out = {}
    for name, v in prof.items():
        phase, kind = PHASE_OF.get(name, ("other", "latency"))
        o = out.setdefault(phase, {"ms": 0.0, "bytes": 0.0, "flops": 0.0, "bound": kind})
        o["ms"] += v["ms"] / nprof; o["bytes"] += v["bytes"] / nprof; o["flops"] += v["flops"] / nprof
        if kind != "latency" and o["bound"] == "latency":
            o["bound"] = kind
    for phase, o in out.items():
        t = o["ms"] * 1e-3
        if o["bound"] == "hbm" and t > 0:
            o["achieved"] = o["bytes"] / t / 1e9; o["peak"] = hbm_gbs; o["unit"] = "GB/s"; o["frac"] = o["achieved"] / hbm_gbs
        elif o["bound"] == "fp64" and t > 0:
            o["achieved"] = o["flops"] / t / 1e12; o["peak"] = p64_tflops; o["unit"] = "TFLOP/s"; o["frac"] = o["achieved"] / p64_tflops
            o["hbm_GBps"] = o["bytes"] / t / 1e9
        else:
            o["frac"] = None
    return out


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


def oracle_sample(name: str, n_full: int, n_sample: int, threads: int | None = None):
    """The oracle as it stands on a bounded sample: one FULL solve of the same recipe at n_sample <= n_full (the method
    costs O(n) per solve at fixed ranks -- eq. (5), PAPER.md:238-242 -- and these recipes have n-independent rank
    structure), scaled linearly in n to the metric's unit at the full size: DOF/s = n_full^2 / (t_sample n_full / n_sample)."""
    ws_ = W.make(name, 0, min(n_sample, n_full))
    if threads is not None:
        from threadpoolctl import threadpool_limits
        with threadpool_limits(limits=threads):
            t, r = oracle_step(ws_)
    else:
        t, r = oracle_step(ws_)
    t_full = t * n_full / ws_.n
    return {"value": float(n_full) ** 2 / t_full, "unit": UNIT, "sample_n": ws_.n, "sample_seconds": t,
            "ms_per_grid_row": 1e3 * t / ws_.n, "extrapolated_seconds_at_full_n": t_full,
            "sweeps": r.sweeps, "rank": r.rank}


def run_reference(args):
    """--impl reference: the CPU oracle on this arm's config, metric and unit (rank 0 only)."""
    rank, _, world = R.env_world()
    if rank != 0:
        return 0
    name = args.workload
    n = NOMINAL_N[name]
    w0 = W.make(name, 0, min(CPU_SAMPLE_N, n))          # rF, tol, ... of the recipe (the sample the oracle is timed on)
    for _ in range(min(args.warmup, 1)):
        oracle_step(w0)
    samples = [oracle_sample(name, n, CPU_SAMPLE_N) for _ in range(args.steps)]
    t_full = float(np.mean([s_["extrapolated_seconds_at_full_n"] for s_ in samples]))
    val = float(n) ** 2 / t_full
    in_mb = 2 * n * w0.rF * 8 / 1e6
    sample = (f"per step one full oracle solve (numpy fp64) of the {name} recipe at n={w0.n} "
              f"({np.mean([s_['sample_seconds'] for s_ in samples]):.1f} s), scaled linearly in n to n={n}")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t_full, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": config_dict(name, n, w0.rF, w0.tol, w0.max_rank, w0.oversample, max(world, 1), in_mb),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cpu_threads(), "cpu_model": cpu_model(), "kind": "oracle",
                             "sample": sample, "ms_per_grid_row": samples[-1]["ms_per_grid_row"]},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def dst_measure(ctx, torch, dev, stream, p: int, batch: int, inplace: bool, hbm_peak: float, reps: int = 10, library: bool = False):
    """Batched DST-I at n = 2^p - 1: buffer sets rotate over >= 4x the L2 so that every repetition starts L2-cold."""
    nd = (1 << p) - 1
    per_set = batch * nd * 8 * (1 if inplace else 2)
    nsets = max(2, int(np.ceil(4 * L2_BYTES / per_set)))
    nsets = min(nsets, 64)
    xs = [torch.randn((batch, nd), dtype=torch.float64, device=dev) for _ in range(nsets)]
    ys = xs if inplace else [torch.empty_like(xs[0]) for _ in range(nsets)]
    for i in range(3):
        ctx.dst1_batched(xs[i % nsets], out=ys[i % nsets])
    d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    reps = max(reps, nsets)
    d0.record(stream)
    for i in range(reps):
        ctx.dst1_batched(xs[i % nsets], out=ys[i % nsets])
    d1.record(stream); torch.cuda.synchronize(dev)
    dms = d0.elapsed_time(d1) / reps
    gbs = 16.0 * nd * batch / (dms * 1e-3) / 1e9
    out = {"p": p, "n": nd, "batch": batch, "in_place": inplace, "ms": dms, "alg_GBps": gbs, "frac_of_hbm_peak": gbs / hbm_peak,
           "frac_of_8TBps": gbs / 8000.0, "buffer_sets": nsets, "footprint_MB": nsets * per_set / 1e6}
    if library and not inplace:
        x0 = xs[0]; y0 = ys[0].clone()
        del xs, ys
        out["library_route"] = dst_library_route(torch, dev, stream, x0, y0, reps)
    return out


def dst_library_route(torch, dev, stream, x, ours, reps: int):
    """The route the paper itself takes (library FFT calls from PyTorch), timed beside the
    kernel as a baseline, never on the product path: DST-I of every row of x (batch, n) as the imaginary part of a real
    FFT of the odd extension of length 2(n+1), torch.fft.rfft = cuFFT D2Z.  `ms` covers extension + FFT + extraction,
    `rfft_only_ms` the library transform alone; `max_rel_diff` compares its result with lrp_dst1_batched's."""
    batch, nd = x.shape
    N = nd + 1
    def route():
        ext = torch.zeros((batch, 2 * N), dtype=torch.float64, device=dev)
        ext[:, 1:N] = x
        ext[:, N + 1:] = -torch.flip(x, dims=(1,))
        return ext, -0.5 * torch.fft.rfft(ext, dim=1).imag[:, 1:N]
    ext, lib = route()
    diff = float((lib - ours).abs().max() / ours.abs().max())
    del lib
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    torch.cuda.synchronize(dev)
    reps = max(3, min(reps, 10))
    e0.record(stream)
    for _ in range(reps):
        ext, lib = route(); del lib
    e1.record(stream)
    for _ in range(reps):
        f = torch.fft.rfft(ext, dim=1); del f
    e2.record(stream); torch.cuda.synchronize(dev)
    return {"kind": "torch.fft.rfft (cuFFT D2Z) of the odd extension of length 2(n+1): the paper's own route, PAPER.md:226-228",
            "ms": e0.elapsed_time(e1) / reps, "rfft_only_ms": e1.elapsed_time(e2) / reps, "max_rel_diff": diff}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--timeline", default="", help="also write the per-launch timeline (CSV) of one real multi-stream solve here")
    ap.add_argument("--dst-p", default="20,22", help="log2(n+1) values of the batched DST-I side measurement")
    ap.add_argument("--dst-sweep", action="store_true", help="print one JSON line per DST-I size p = 12..22 (batch 128, out of place "
                    "and in place, L2-cold) instead of the solve benchmark")
    ap.add_argument("--seeds", type=int, default=0, help="also solve seeds 0..K-1 of the workload: mean +- std (PAPER.md:280, 325)")
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
    stream = torch.cuda.current_stream(dev)
    hbm_peak, peak_src = measured_peaks()

    if args.dst_sweep:                                   # the C5 config's second half: lengths 2^12-1 .. 2^22-1, batch 128
        if rank == 0:
            for p_ in range(12, 23):
                for inplace in (False, True):
                    print(json.dumps(dst_measure(ctx, torch, dev, stream, p_, 128, inplace, hbm_peak, library=True)), flush=True)
        ctx.close()
        return 0

    pk = ctx.fp64_peak()                                 # measured on this device, this run
    p64 = max(pk["dfma_tflops"], pk["dmma_tflops"])

    w = W.make(args.workload, seed=rank)
    n, rF = w.n, w.rF
    UF = lrp.tall_from_numpy(w.UF, dev); VF = lrp.tall_from_numpy(w.VF, dev); SF = torch.from_numpy(w.SF).to(dev)
    kw = dict(tol=w.tol, max_rank=w.max_rank, oversample=w.oversample, max_sweeps=w.max_sweeps, safeguard=w.safeguard)
    in_bytes = (UF.numel() + VF.numel() + SF.numel()) * 8
    flush = None
    if in_bytes <= L2_BYTES:                             # small configs: write a buffer larger than L2 between timed steps
        flush = torch.empty(int(1.5 * L2_BYTES) // 8, dtype=torch.float64, device=dev)

    def step():
        return ctx.cross_deim_solve(UF, SF, VF, **kw)

    for _ in range(warmup):
        res = step()
    # ---- timed region: K solves, device-resident inputs, CUDA events on the launching stream
    clocks = ClockSampler(local_rank)
    R.barrier(dist); torch.cuda.synchronize(dev)
    clocks.start()
    l0 = ctx.launch_count()
    local_ms = 0.0
    if flush is None:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            res = step()
        e1.record(stream)
        torch.cuda.synchronize(dev)
        local_ms = e0.elapsed_time(e1)
    else:
        for _ in range(steps):
            flush.fill_(1.0)                              # not timed
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); res = step(); e1.record(stream)
            torch.cuda.synchronize(dev)
            local_ms += e0.elapsed_time(e1)
    R.barrier(dist)
    launches = ctx.launch_count() - l0
    agg = R.throughput(dist, local_ms, float(n) ** 2 * steps, dev)
    clk = clocks.stop()

    # ---- end to end through the C-ABI call with HOST buffers (lrp_cross_deim_solve_host): every step's inputs come from
    # pinned host memory and every step's result is read back to pinned host memory inside the timed region; the call
    # overlaps the copies of the neighbouring steps with the solve (two staging slots).  `single_call_ms` is one isolated
    # call (copy in, solve, copy out, nothing to overlap with).
    e2e_error = None
    lanes, d2h, e2e_single_ms, two_lane = 1, 0, None, None
    agg_e2e = {"per_s": None, "ms": None}
    try:
        hprob = tuple(t.pin_memory() for t in (torch.from_numpy(np.ascontiguousarray(w.UF.T)), torch.from_numpy(np.ascontiguousarray(w.SF)),
                                               torch.from_numpy(np.ascontiguousarray(w.VF.T))))
        pool = [(torch.empty((w.max_rank, n), dtype=torch.float64).pin_memory(), torch.empty(w.max_rank, dtype=torch.float64).pin_memory(),
                 torch.empty((w.max_rank, n), dtype=torch.float64).pin_memory()) for _ in range(2)]

        torch.cuda.empty_cache()
        lanes = 2 if ctx.lib.lrp_solve_host_workspace_bytes(n, rF, w.max_rank, w.oversample, 2) < 64e9 else 1      # C5: one lane (2 x 66 GB otherwise)

        def e2e_batch(k):
            return ctx.cross_deim_solve_host([hprob] * k, [pool[p & 1] for p in range(k)], lanes=lanes, **kw)
        e2e_batch(2)                                       # warm-up: workspace, copy streams
        R.barrier(dist); torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        hres = e2e_batch(steps)
        e2e_ms = 1e3 * (time.perf_counter() - t0)
        R.barrier(dist)
        d2h = (2 * n * hres[-1]["rank"] + hres[-1]["rank"]) * 8
        t0 = time.perf_counter()
        e2e_batch(1)
        e2e_single_ms = 1e3 * (time.perf_counter() - t0)
        agg_e2e = R.throughput(dist, e2e_ms, float(n) ** 2 * steps, dev)
        del pool, hprob
        # ---- the same K device-resident solves with two in flight (lrp_cross_deim_solve_batch): what a second solve fills of the
        # SMs the first leaves idle.  Reported beside `value`, which stays one solve after the other.
        if lanes == 2:
            ctx.release_workspace(); torch.cuda.empty_cache()
            bouts = [(torch.empty((w.max_rank, n), dtype=torch.float64, device=dev), torch.empty(w.max_rank, dtype=torch.float64, device=dev),
                      torch.empty((w.max_rank, n), dtype=torch.float64, device=dev)) for _ in range(steps)]
            ctx.cross_deim_solve_batch([(UF, SF, VF)] * 2, lanes=2, outputs=bouts[:2], **kw)
            R.barrier(dist); torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            ctx.cross_deim_solve_batch([(UF, SF, VF)] * steps, lanes=2, outputs=bouts, **kw)
            torch.cuda.synchronize(dev)
            agg2 = R.throughput(dist, 1e3 * (time.perf_counter() - t0), float(n) ** 2 * steps, dev)
            two_lane = {"value": agg2["per_s"], "unit": UNIT, "ms_per_step": agg2["ms"] / steps, "lanes": 2,
                        "call": "lrp_cross_deim_solve_batch, host timer around the synchronous call (outputs preallocated)"}
            del bouts
    except Exception as ex:                            # e.g. no pinned host memory to be had: the device-resident line still prints
        if dist is not None:
            raise
        e2e_error = f"{type(ex).__name__}: {ex}"[:300]
    ctx.release_workspace(); torch.cuda.empty_cache()  # the staging slots are not needed any more (the next call sizes a new workspace)

    if args.timeline and rank == 0:                 # start/end of every launch of one solve, streams NOT serialised
        ctx.profile_reset(); ctx.profile_enable(2)
        step()
        ctx.profile_timeline(args.timeline)
        ctx.profile_enable(False); ctx.profile_reset()

    # ---- per-kernel profile (separate pass: events around every launch), rooflines
    ctx.profile_reset(); ctx.profile_enable(True)
    nprof = 2
    for _ in range(nprof):
        step()
    prof = ctx.profile()
    ctx.profile_enable(False); ctx.profile_reset()
    tot_ms = sum(v["ms"] for v in prof.values()) or 1.0
    kernels = []
    for name, v in sorted(prof.items(), key=lambda kv: -kv[1]["ms"]):
        ms = v["ms"]
        gbs = v["bytes"] / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
        tfl = v["flops"] / (ms * 1e-3) / 1e12 if ms > 0 else 0.0
        kernels.append({"kernel": name, "launches_per_step": v["count"] / nprof, "ms_per_step": ms / nprof,
                        "share": ms / tot_ms, "alg_GBps": gbs, "alg_TFLOPs": tfl})
    # dominant kernel class, on the roofline SURVEY.md 8(d) assigns to it (the larger of its two floor times)
    top = kernels[0]
    t_hbm = prof[top["kernel"]]["bytes"] / (hbm_peak * 1e9)
    t_alu = prof[top["kernel"]]["flops"] / (p64 * 1e12)
    vtop = prof[top["kernel"]]
    if t_alu >= t_hbm:
        roof = {"bound": "alu", "achieved": top["alg_TFLOPs"], "peak": p64, "unit": "TFLOP/s", "frac": top["alg_TFLOPs"] / p64,
                "traffic": None, "peak_source": "measured this run (lrp_fp64_peak: max of DFMA and DMMA register-only loops)"}
    else:
        roof = {"bound": "hbm", "achieved": top["alg_GBps"], "peak": hbm_peak, "unit": "GB/s", "frac": top["alg_GBps"] / hbm_peak,
                "traffic": None, "peak_source": peak_src}
    roof["kernel"] = top["kernel"]; roof["share_of_step"] = top["share"]
    roof["alg_bytes_per_launch"] = vtop["bytes"] / vtop["count"]; roof["alg_flops_per_launch"] = vtop["flops"] / vtop["count"]
    tr = NCU_TRAFFIC.get(top["kernel"])                  # dram__bytes read + write per launch / algorithmic bytes, this round's ncu capture
    if tr is not None:
        roof["traffic"] = tr["dram_over_alg"] * roof["alg_bytes_per_launch"]; roof["traffic_source"] = tr["source"]
    trace = [dict(I=t["I"], J=t["J"], rank=t["rank"]) for t in res["trace"]]
    solve_roof = solve_roofline(n, rF, trace, res["rank"], hbm_peak, p64, agg["ms"] / steps)
    phases = phase_rooflines(prof, nprof, hbm_peak, p64)

    # ---- batched DST-I side measurement (metric's second half): batch 128, L2-cold rotation
    dst = []
    try:
        for p_ in [int(v) for v in args.dst_p.split(",") if v]:
            dst.append(dst_measure(ctx, torch, dev, stream, p_, 128, False, hbm_peak, library=True))
    except Exception as ex:                       # never lose the main line because of the side measurement
        dst.append({"error": str(ex)})

    # ---- mean +- std over seeds, optional
    seeds = None
    if args.seeds > 0 and rank == 0:
        rows = []
        for sd in range(args.seeds):
            ws_ = W.make(args.workload, seed=sd)
            a_, b_, c_ = lrp.tall_from_numpy(ws_.UF, dev), torch.from_numpy(ws_.SF).to(dev), lrp.tall_from_numpy(ws_.VF, dev)
            kws = dict(tol=ws_.tol, max_rank=ws_.max_rank, oversample=ws_.oversample, max_sweeps=ws_.max_sweeps, safeguard=ws_.safeguard)
            ctx.cross_deim_solve(a_, b_, c_, **kws)                       # warm-up with the same seed
            ts = []
            for _ in range(3):
                torch.cuda.synchronize(dev); t0 = time.perf_counter()
                r_ = ctx.cross_deim_solve(a_, b_, c_, **kws)
                torch.cuda.synchronize(dev); ts.append(1e3 * (time.perf_counter() - t0))
            rows.append({"seed": sd, "ms": float(np.mean(ts)), "rank": r_["rank"], "sweeps": r_["sweeps"], "converged": r_["converged"]})
            del a_, b_, c_
        ms_ = np.array([r_["ms"] for r_ in rows])
        seeds = {"count": args.seeds, "ms_mean": float(ms_.mean()), "ms_std": float(ms_.std()),
                 "rank_mean": float(np.mean([r_["rank"] for r_ in rows])), "rank_std": float(np.std([r_["rank"] for r_ in rows])),
                 "sweeps_mean": float(np.mean([r_["sweeps"] for r_ in rows])), "sweeps_std": float(np.std([r_["sweeps"] for r_ in rows])),
                 "per_seed": rows, "protocol": "warm-up solve with the same seed, then 3 timed solves (host timer around the synchronous call)"}

    # ---- the oracle timed beside it (rank 0, N = 1 only): bounded sample of the same recipe, scaled to the full size
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        a_ = oracle_sample(args.workload, n, CPU_SAMPLE_N)
        one = oracle_sample(args.workload, n, CPU_SAMPLE_N_1T, threads=1)
        # the GPU on the very sample the oracle was timed on (same n): the like-for-like pair
        wsmp = W.make(args.workload, 0, a_["sample_n"])
        a2, b2, c2 = lrp.tall_from_numpy(wsmp.UF, dev), torch.from_numpy(wsmp.SF).to(dev), lrp.tall_from_numpy(wsmp.VF, dev)
        kws = dict(tol=wsmp.tol, max_rank=wsmp.max_rank, oversample=wsmp.oversample, max_sweeps=wsmp.max_sweeps, safeguard=wsmp.safeguard)
        ctx.cross_deim_solve(a2, b2, c2, **kws)
        torch.cuda.synchronize(dev); t0 = time.perf_counter()
        ctx.cross_deim_solve(a2, b2, c2, **kws)
        torch.cuda.synchronize(dev); gpu_sample_ms = 1e3 * (time.perf_counter() - t0)
        cpu = {"value": a_["value"], "unit": UNIT, "cores": cpu_threads(), "cpu_model": cpu_model(), "kind": "oracle",
               "sample": f"one full oracle solve (numpy fp64) of the {args.workload} recipe at n={a_['sample_n']}: {a_['sample_seconds']:.1f} s on "
                         f"{cpu_threads()} threads, scaled linearly in n (O(n) method, PAPER.md:238-242) to n={n}: {a_['extrapolated_seconds_at_full_n']:.0f} s",
               "ms_per_grid_row": a_["ms_per_grid_row"], "gpu_ms_per_grid_row": (agg["ms"] / steps) / n,
               "same_n_pair": {"n": a_["sample_n"], "oracle_ms": 1e3 * a_["sample_seconds"], "gpu_ms": gpu_sample_ms},
               "single_thread": {"sample_n": one["sample_n"], "sample_seconds": one["sample_seconds"], "ms_per_grid_row": one["ms_per_grid_row"],
                                 "value": one["value"]}}

    if rank == 0:
        info = res["info"]
        line = {"metric": METRIC, "value": agg["per_s"], "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
                "ms_per_step": agg["ms"] / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": config_dict(w.name, n, rF, w.tol, w.max_rank, w.oversample, world, in_bytes / 1e6),
                "solve": {"rank": res["rank"], "sweeps": res["sweeps"], "converged": res["converged"],
                          "ms": {k: getattr(info, "ms_" + k) for k in ("dst_fwd", "select", "sample", "qr", "core", "rebuild", "stop", "dst_inv", "total")}},
                "clocks": clk,
                "e2e": {"value": agg_e2e["per_s"], "unit": UNIT, "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": d2h,
                        "ms_per_step": (agg_e2e["ms"] / steps) if agg_e2e["ms"] is not None else None, "single_call_ms": e2e_single_ms, "error": e2e_error,
                        "lanes": lanes,
                        "call": "lrp_cross_deim_solve_host: one call for all steps; per lane the copies of its previous / next step overlap its solve"},
                "gpu_launches": int(launches), "two_solves_in_flight": two_lane,
                "roofline": roof, "solve_roofline": solve_roof, "phases": phases, "fp64_peak_measured": pk,
                "kernels": kernels, "dst1": dst, "seeds": seeds, "cpu_baseline": cpu}
        print(json.dumps(line))
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
