"""Writes tests/golden/solve_<cfg>_n<n>_s<seed>.npz (+ a .txt header beside it): the CPU oracle's FREE RUN of the
Cross-DEIM low-rank Poisson solve (Alg. 4; section 3.2) on one seeded workload
at a size where the oracle is too slow to be called from a test (C3/C4/C5 at BASELINE.json's full sizes, C5-shaped
cases at n = 65535, 2^18-1 and 2^20-1), reduced to what the `-m gpu` parity tests need:

  * the trace of discrete decisions (I_k, J_k, prune masks, rank, rho, ind, eta, S_min per sweep, the leverage
    selections I*, J* and the sorted top scores that decide them) -- the GPU free run is compared with it and the
    GPU is then REPLAYED on it (the oracle's trace is an input of the CUDA path, never the other way round);
  * the final singular values (all r_k of the untruncated iterate), final rank, |diag R_C|, |diag R_R| of every sweep;
  * 4096 physical-space entries W(i,j) at `workloads.sample_pairs(n, 4096, seed=1)`;
  * the selected fibers of the final spectral iterate -- columns J_k and rows I_k of U_k S_k V_k^T -- at 1024 positions
    (the 256 lowest frequencies + 768 seeded random ones; a full fiber is n doubles) plus the 2-norm of each whole fiber
    and max |What| over them.

Only `oracle/` and the input generators `paper_2607_06021_b200/workloads.py` are imported; nothing here (and nothing
it writes) comes from the CUDA path.

Run (from the repo root; wall time and peak memory end up in the .txt header):
    python tests/golden/make_solve_golden.py C4 --seed 0
    python tests/golden/make_solve_golden.py C5 --seed 0 --n 65535
    python tests/golden/make_solve_golden.py C5 --seed 0 --n 1048575      # 86 min, 13.8 GB on 8 cores
"""
import argparse
import os
import resource
import subprocess
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import lrp_oracle as O                      # noqa: E402
from paper_2607_06021_b200 import workloads as W        # noqa: E402

FIBER_POS_LOW = 256
FIBER_POS_RANDOM = 768


def fiber_positions(n: int, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed + 777)
    low = np.arange(min(FIBER_POS_LOW, n), dtype=np.int64)
    rnd = rng.integers(0, n, FIBER_POS_RANDOM).astype(np.int64)
    return np.concatenate([low, rnd])


def golden_name(cfg: str, n: int, seed: int) -> str:
    return f"solve_{cfg}_n{n}_s{seed}"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--n", type=int, default=None)
    ap.add_argument("--max-sweeps", type=int, default=None)
    ap.add_argument("--out-dir", default=HERE)
    a = ap.parse_args()
    w = W.make(a.config, a.seed, a.n)
    if a.max_sweeps:
        w.max_sweeps = a.max_sweeps
    n = w.n
    t0 = time.time()
    ref = O.cross_deim_solve(n, w.UF, w.SF, w.VF, **w.opts())
    wall = time.time() - t0
    out = dict(n=np.int64(n), seed=np.int64(a.seed), sweeps=np.int64(ref.sweeps), rank=np.int64(ref.rank),
               converged=np.int64(ref.converged), tol=np.float64(w.tol), max_rank=np.int64(w.max_rank),
               oversample=np.int64(w.oversample), max_sweeps=np.int64(w.max_sweeps),
               SW=ref.SW, Shat=ref.Shat)
    for s, t in enumerate(ref.trace):
        out[f"I_{s}"] = t.I.astype(np.int32)
        out[f"J_{s}"] = t.J.astype(np.int32)
        out[f"keepI_{s}"] = t.keepI.astype(np.uint8)
        out[f"keepJ_{s}"] = t.keepJ.astype(np.uint8)
        out[f"Istar_{s}"] = np.asarray(t.Istar, dtype=np.int32)
        out[f"Jstar_{s}"] = np.asarray(t.Jstar, dtype=np.int32)
        out[f"topU_{s}"] = np.sort(t.scoresU)[::-1][:len(t.Istar) + 1].copy()
        out[f"topV_{s}"] = np.sort(t.scoresV)[::-1][:len(t.Jstar) + 1].copy()
        out[f"rC_{s}"] = t.rC
        out[f"rR_{s}"] = t.rR
        out[f"scalars_{s}"] = np.array([t.rank, t.rho, t.ind, t.eta1, t.eta2, t.smin_full, t.snorm], dtype=np.float64)
    rows, cols = W.sample_pairs(n, 4096, seed=1)
    out["W_rows"] = rows
    out["W_cols"] = cols
    out["W_vals"] = O.lowrank_entries(ref.UW, ref.SW, ref.VW, rows, cols)
    I = ref.trace[-1].I.astype(np.int64)
    J = ref.trace[-1].J.astype(np.int64)
    pos = fiber_positions(n, a.seed)
    colsR = (ref.Uhat * ref.Shat) @ ref.Vhat[J].T           # n x |J|: columns J of the spectral iterate
    rowsR = (ref.Vhat * ref.Shat) @ ref.Uhat[I].T           # n x |I|: rows I, transposed
    out["fiber_pos"] = pos
    out["fiber_cols"] = colsR[pos]
    out["fiber_rows"] = rowsR[pos]
    out["fiber_cols_norm"] = np.linalg.norm(colsR, axis=0)
    out["fiber_rows_norm"] = np.linalg.norm(rowsR, axis=0)
    out["ghat"] = np.float64(max(np.abs(colsR).max(), np.abs(rowsR).max()))
    # orthonormality of the oracle's own factors at this size (the property the GPU factors are held to as well)
    out["orth_U"] = np.float64(np.abs(ref.Uhat.T @ ref.Uhat - np.eye(ref.Uhat.shape[1])).max())
    out["orth_V"] = np.float64(np.abs(ref.Vhat.T @ ref.Vhat - np.eye(ref.Vhat.shape[1])).max())
    name = golden_name(a.config, n, a.seed)
    np.savez_compressed(os.path.join(a.out_dir, name + ".npz"), **out)
    try:
        commit = subprocess.run(["git", "-C", ROOT, "log", "-1", "--format=%h", "--", "oracle/"],
                                capture_output=True, text=True).stdout.strip()
    except Exception:
        commit = "?"
    with open(os.path.join(a.out_dir, name + ".txt"), "w") as f:
        f.write(f"# {name}.npz -- oracle free run, written by tests/golden/make_solve_golden.py "
                f"{' '.join(sys.argv[1:])}\n")
        f.write(f"# source: oracle/lrp_oracle.py (last oracle commit {commit}); method: PAPER.md:129-192 (Alg. 4), "
                f"26-51 (Alg. 1), 105-114 (Alg. 3), 222-236 (section 3.2); readings DESIGN.md section 2\n")
        f.write(f"config {a.config} seed {a.seed} n {n} tol {w.tol} max_rank {w.max_rank} oversample {w.oversample} "
                f"max_sweeps {w.max_sweeps}\n")
        f.write(f"sweeps {ref.sweeps} rank {ref.rank} converged {int(ref.converged)}\n")
        f.write(f"oracle_wall_s {wall:.1f} cores {os.cpu_count()} "
                f"peak_rss_gb {resource.getrusage(resource.RUSAGE_SELF).ru_maxrss / 1048576:.1f}\n")
        for s, t in enumerate(ref.trace):
            f.write(f"sweep {s}: nI {len(t.I)} nJ {len(t.J)} rank {t.rank} rho/|S| {t.rho / t.snorm:.3e} "
                    f"ind/|S| {t.ind / t.snorm:.3e} eta1 {t.eta1:.3e} eta2 {t.eta2:.3e} "
                    f"pruned {int((~t.keepI).sum())}/{int((~t.keepJ).sum())}\n")
    print(open(os.path.join(a.out_dir, name + ".txt")).read())


if __name__ == "__main__":
    main()
