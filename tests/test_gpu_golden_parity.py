"""GPU <-> oracle parity at the sizes the oracle cannot reach inside a test: BASELINE.json's C3 and C4 at full size
and C5-shaped cases at n = 65535 / 2^18-1 / 2^20-1.  The oracle's FREE RUN was computed once by
tests/golden/make_solve_golden.py (oracle + input generators only) and reduced to the trace of discrete decisions, the
singular values, 4096 physical-space entries and the selected fibers at 1024 positions (+ whole-fiber norms).

Per case: (1) the GPU free run is compared with the oracle's decisions wherever the deciding gaps are clear
(north_star: index sets equal where the leverage gap exceeds 1e-12; sweep count within one when rho or the indicator is
within 10x of the threshold); (2) the GPU is REPLAYED on the oracle's trace and compared entry by entry at 1e-10
(north_star) -- for a run the sweep cap ended before the stop test passed (C3 as configured), reading R1
applies and the bound is stated there.  The solve runs in the launch configuration bench.py times."""
import os

import numpy as np
import pytest

from paper_2607_06021_b200 import workloads as W

pytestmark = pytest.mark.gpu

GOLDEN_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
TOL = 1e-10

# (config, seed, n) -- n = None: the config's own size.  C5 at its own size (n = 2^22 - 1) has no stored oracle run: scaled
# from the n = 2^20 - 1 case (5162 s, 13.8 GB on 8 cores) it needs ~5.7 h and ~55 GB of the build box's 62 GB; C5 is covered
# by its three smaller shapes here (the largest a quarter of its size: four-step DST-I, five-level TSQR tree, several
# waves of row slabs, K up to 95 of K_cap = 272) and by the size-independent properties of tests/test_gpu_full_size.py.
CASES = [("C3", 0, None), ("C5", 0, 65535), ("C5", 0, (1 << 18) - 1), ("C5", 0, (1 << 20) - 1), ("C4", 0, None)]


@pytest.fixture(scope="module")
def ctx():
    from paper_2607_06021_b200 import build, lrp
    build.build()
    c = lrp.Context(0)
    yield c
    c.close()


def _load(cfg, seed, n):
    w_n = n if n is not None else {"C3": 65535, "C4": (1 << 20) - 1, "C5": (1 << 22) - 1}[cfg]
    path = os.path.join(GOLDEN_DIR, f"solve_{cfg}_n{w_n}_s{seed}.npz")
    if not os.path.exists(path):
        pytest.skip(f"{os.path.basename(path)} not generated (tests/golden/make_solve_golden.py {cfg} --seed {seed}"
                    f"{'' if n is None else ' --n ' + str(n)})")
    return np.load(path)


def _gpu_solve(ctx, w, **kw):
    import torch
    from paper_2607_06021_b200 import lrp
    return ctx.cross_deim_solve(lrp.tall_from_numpy(w.UF), torch.from_numpy(w.SF).cuda(), lrp.tall_from_numpy(w.VF),
                                tol=w.tol, max_rank=w.max_rank, oversample=w.oversample, max_sweeps=w.max_sweeps,
                                safeguard=w.safeguard, want_spectral=True, **kw)


@pytest.mark.parametrize("cfg,seed,n", CASES)
def test_free_run_decisions_and_replay_parity(ctx, cfg, seed, n):
    import torch
    g = _load(cfg, seed, n)
    w = W.make(cfg, seed, n)
    assert w.n == int(g["n"]) and w.max_sweeps == int(g["max_sweeps"]) and w.tol == float(g["tol"])
    sweeps_or, rank_or, conv_or = int(g["sweeps"]), int(g["rank"]), bool(g["converged"])

    # ---------------------------------------------------------------- (1) free run: discrete decisions
    res = _gpu_solve(ctx, w)
    nchk = min(res["sweeps"], sweeps_or)
    compared = 0
    for s in range(nchk):
        clear = True
        for top in (g[f"topU_{s}"], g[f"topV_{s}"]):
            clear &= bool(np.abs(np.diff(top)).min() > 1e-12)          # every gap that decides membership / order
        rr = g[f"rR_{s}"] / g[f"rR_{s}"].max(); rc = g[f"rC_{s}"] / g[f"rC_{s}"].max()
        clear &= not (((rr > 1e-13) & (rr < 1e-11)).any() or ((rc > 1e-13) & (rc < 1e-11)).any())
        if not clear:
            break
        t = res["trace"][s]
        assert t["I"].tolist() == g[f"I_{s}"].tolist() and t["J"].tolist() == g[f"J_{s}"].tolist(), f"sweep {s}"
        assert t["keepI"].tolist() == g[f"keepI_{s}"].astype(bool).tolist(), f"sweep {s}"
        assert t["keepJ"].tolist() == g[f"keepJ_{s}"].astype(bool).tolist(), f"sweep {s}"
        assert t["rank"] == int(g[f"scalars_{s}"][0]), f"sweep {s}"
        compared += 1
    print(f"{cfg} n={w.n}: free run {res['sweeps']} sweeps (oracle {sweeps_or}), decisions compared on {compared} sweeps, "
          f"GPU rank {res['rank']} (oracle {rank_or}), GPU converged {res['converged']} (oracle {conv_or})")
    assert compared >= 1
    assert abs(res["sweeps"] - sweeps_or) <= 1
    last = g[f"scalars_{sweeps_or - 1}"]
    margin = max(last[1], last[2]) / (w.tol * last[6])                  # max(rho, ind) / threshold in the oracle's last sweep
    if compared == sweeps_or and (margin < 0.1 or margin > 10.0):
        assert res["sweeps"] == sweeps_or and res["converged"] == conv_or and res["rank"] == rank_or
    del res

    # ---------------------------------------------------------------- (2) replay of the oracle's trace: continuous parity
    rep = [dict(I=g[f"I_{s}"], J=g[f"J_{s}"], keepI=g[f"keepI_{s}"], keepJ=g[f"keepJ_{s}"]) for s in range(sweeps_or)]
    rep[-1]["final_rank"] = rank_or
    res = _gpu_solve(ctx, w, replay=rep)
    assert res["sweeps"] == sweeps_or and res["rank"] == rank_or
    # Singular values, selected fibers and fiber norms: 1e-10 flat.  Physical-space entries of a run the sweep cap ended
    # before the stop test passed (C3 as configured): DESIGN.md reading R1 -- the final truncation cuts an iterate whose
    # trailing singular values (~rho) are not yet resolved, and two fp64 implementations then differ by a fraction of
    # rho/||S|| on W; bound max(1e-10, 0.1 rho/||S||) = 2.7e-10 at C3 (measured 1.4e-10, printed below).
    tol = TOL
    tolW = TOL if conv_or else max(TOL, 0.1 * last[1] / last[6])
    Sh = res["Shat"].cpu().numpy()
    assert Sh.shape[0] == g["Shat"].shape[0]
    errS = np.abs(Sh - g["Shat"]).max() / g["Shat"][0]
    rows = torch.from_numpy(g["W_rows"]).cuda(); cols = torch.from_numpy(g["W_cols"]).cuda()
    got = ctx.lowrank_entries(res["UW"], res["SW"], res["VW"], rows, cols).cpu().numpy()
    errW = np.abs(got - g["W_vals"]).max() / np.abs(g["W_vals"]).max()
    # selected fibers of the spectral iterate at the stored positions, and whole-fiber norms
    pos = torch.from_numpy(g["fiber_pos"]).cuda()
    I = torch.from_numpy(g[f"I_{sweeps_or - 1}"].astype(np.int64)).cuda()
    J = torch.from_numpy(g[f"J_{sweeps_or - 1}"].astype(np.int64)).cuda()
    Uh, Vh, S = res["Uhat"], res["Vhat"], res["Shat"]                   # tall tensors (r, n)
    colsG = ((Uh[:, pos] * S[:, None]).T @ Vh[:, J]).cpu().numpy()       # (npos, |J|)
    rowsG = ((Vh[:, pos] * S[:, None]).T @ Uh[:, I]).cpu().numpy()
    ghat = float(g["ghat"])
    errF = max(np.abs(colsG - g["fiber_cols"]).max(), np.abs(rowsG - g["fiber_rows"]).max()) / ghat
    ncol = torch.linalg.vector_norm((Uh * S[:, None]).T @ Vh[:, J], dim=0).cpu().numpy()
    nrow = torch.linalg.vector_norm((Vh * S[:, None]).T @ Uh[:, I], dim=0).cpu().numpy()
    errN = max(np.abs(ncol - g["fiber_cols_norm"]).max(), np.abs(nrow - g["fiber_rows_norm"]).max()) / g["fiber_cols_norm"].max()
    dev = lambda F: float((F @ F.T - torch.eye(F.shape[0], dtype=F.dtype, device=F.device)).abs().max().item())
    orth = max(dev(res["Uhat"]), dev(res["Vhat"]))                      # spectral iterate: Q (thin QR) times the core's factors
    orth_phys = max(dev(res["UW"]), dev(res["VW"]))                     # after the inverse DST-I
    print(f"{cfg} n={w.n}: replay parity  S {errS:.2e}  W {errW:.2e}  fibers {errF:.2e}  fiber norms {errN:.2e}  "
          f"(tol {tol:.1e})  orthonormality {orth:.1e} / physical {orth_phys:.1e} (oracle {max(float(g['orth_U']), float(g['orth_V'])):.1e})")
    assert errS <= tol and errW <= tolW and errF <= tol and errN <= tol
    # 1e-13, widened by the rounding of the check itself (n-term fp64 Gram sums: eps sqrt(n) = 2.3e-13 at n = 2^20)
    floor = max(1.0, np.sqrt(w.n / float(1 << 18)))
    assert orth <= 1e-13 * floor and orth_phys <= 1e-12 * floor
