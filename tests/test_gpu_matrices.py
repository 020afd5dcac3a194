"""NEXT-1 of SURVEY.md 8(f): generic function-handle Cross-DEIM on the paper's test matrices H (Hilbert) and K, eq. (6),
PAPER.md:264-267, on the GPU against the oracle: sampler entrywise, free-run decisions, replay parity at 1e-10."""
import numpy as np
import pytest

from oracle import lrp_oracle as O
from paper_2607_06021_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def ctx():
    from paper_2607_06021_b200 import build, lrp
    build.build()
    c = lrp.Context(0)
    yield c
    c.close()


@pytest.mark.parametrize("kind,n", [("hilbert", 1000), ("kmatrix", 1000), ("kmatrix", 4097), ("hilbert", 65536)])
def test_sample_matrix_entrywise(ctx, kind, n):
    import torch
    from paper_2607_06021_b200 import lrp
    rng = np.random.default_rng(n)
    I = rng.choice(n, 19, replace=False).astype(np.int32); J = rng.choice(n, 33, replace=False).astype(np.int32)
    I[0], J[0] = 0, n - 1
    Cref, Rref = O.matrix_fibers(kind, n)(I, J)
    Cg, Rg = ctx.sample_matrix(kind, n, torch.from_numpy(I).cuda(), torch.from_numpy(J).cuda())
    Cg, Rg = lrp.tall_to_numpy(Cg), lrp.tall_to_numpy(Rg)
    if kind == "hilbert":                                       # one exact division: bit-identical
        assert np.array_equal(Cg, Cref) and np.array_equal(Rg, Rref)
    else:                                                       # t^5 by multiplications vs libm pow: a few ulp
        assert np.abs(Cg - Cref).max() <= 4e-16 * np.abs(Cref).max() and np.abs(Rg - Rref).max() <= 4e-16 * np.abs(Rref).max()


def _solve(ctx, kind, n, U0, V0, sg, tol, sweeps=12, **kw):
    from paper_2607_06021_b200 import lrp
    return ctx.cross_deim_matrix(kind, n, lrp.tall_from_numpy(U0), lrp.tall_from_numpy(V0), tol=tol, max_rank=64, oversample=8,
                                 max_sweeps=sweeps, safeguard=sg, want_spectral=True, **kw)


# (kind, n, tol, seed, max_sweeps).  n = 777 and 600: n + 1 is not a power of two (no transform is involved here).
# For many initial guesses the deterministic top-k selection stalls on these matrices (the same indices are re-selected
# and the safeguard index is pruned again -- PAPER.md:301 "the LS selection is clearly worse"; the Bernoulli form of
# Alg. 3 is the remedy): ("hilbert", 1024, seed 1) and ("kmatrix", 512, seed 2) are such runs, compared under reading R1.
CASES = [("hilbert", 512, 1e-9, 0, 12), ("hilbert", 1024, 1e-9, 0, 12), ("hilbert", 1024, 1e-9, 1, 12), ("kmatrix", 512, 1e-6, 0, 12),
         ("kmatrix", 512, 1e-6, 2, 12), ("hilbert", 777, 1e-9, 0, 12), ("kmatrix", 600, 1e-6, 1, 12)]


@pytest.mark.parametrize("kind,n,tol,seed,sweeps", CASES)
def test_matrix_cross_deim_free_run_and_replay(ctx, kind, n, tol, seed, sweeps):
    from paper_2607_06021_b200 import lrp
    U0, V0, sg = W.matrix_initial_guess(n, 4, seed)
    ref = O.cross_deim(n, O.matrix_fibers(kind, n), U0, V0, tol=tol, max_rank=64, oversample=8, max_sweeps=sweeps, safeguard=sg)
    res = _solve(ctx, kind, n, U0, V0, sg, tol, sweeps)
    # discrete decisions of the free run where the deciding gaps are clear
    compared = 0
    for s in range(min(res["sweeps"], ref.sweeps)):
        t = ref.trace[s]
        sel_clear = True
        for sc, star in ((t.scoresU, t.Istar), (t.scoresV, t.Jstar)):
            srt = np.sort(sc)[::-1][:len(star) + 1]
            sel_clear &= bool(np.abs(np.diff(srt)).min() > 1e-12)
        if not sel_clear:
            break
        g = res["trace"][s]
        assert g["I"].tolist() == t.I.tolist() and g["J"].tolist() == t.J.tolist(), f"sweep {s}"
        compared += 1
        # prune masks: only when no |diag R| sits in the tolerance band around 1e-12 (a rapidly decaying matrix such as
        # H puts values there by construction); later sweeps depend on them
        rr = t.rR / t.rR.max(); rc = t.rC / t.rC.max()
        if ((rr > 1e-13) & (rr < 1e-11)).any() or ((rc > 1e-13) & (rc < 1e-11)).any():
            break
        assert g["keepI"].tolist() == t.keepI.tolist() and g["keepJ"].tolist() == t.keepJ.tolist()
    print(f"{kind} n={n} seed={seed}: GPU {res['sweeps']} sweeps rank {res['rank']} conv {res['converged']}; oracle {ref.sweeps} sweeps "
          f"rank {ref.rank} conv {ref.converged}; index sets compared on {compared} sweeps")
    assert compared >= 1
    # replay of the oracle's trace: continuous parity
    rep = O.trace_to_replay(ref.trace, ref.rank)
    res2 = _solve(ctx, kind, n, U0, V0, sg, tol, sweeps, replay=rep)
    assert res2["sweeps"] == ref.sweeps and res2["rank"] == ref.rank
    U = lrp.tall_to_numpy(res2["UW"]); V = lrp.tall_to_numpy(res2["VW"]); S = res2["SW"].cpu().numpy()
    rows, cols = W.sample_pairs(n, 4096, seed=9)
    a = np.einsum("tk,k,tk->t", U[rows], S, V[cols])
    b = O.lowrank_entries(ref.U[:, :ref.rank], ref.S[:ref.rank], ref.V[:, :ref.rank], rows, cols)
    t = ref.trace[-1]
    # DESIGN.md reading R1: a run that never passed the stop test (these matrices make the deterministic selection stall
    # for some initial guesses) is defined only up to its own error estimates: a tenth of rho and the
    # a-posteriori indicator of Alg. 4 line 26, whose pseudo-inverse cut at 1e-13 sigma_max sits inside the
    # spectrum of these ill-conditioned cores.  Converged runs: 1e-10, or the last sweep's indicator where that is larger:
    # when the sampled fibers are numerically dependent (min |diag R_C| / max ~ 7e-15 in the K-matrix runs) the trailing
    # columns of Q are set by rounding, and what they contribute to the iterate is what the indicator S_min * eta
    # estimates (K, n = 600, seed 1: ind/||S|| = 5.6e-8 at tol = 1e-6; measured difference 3.6e-8).
    tolW = max(TOL, t.ind / t.snorm) if ref.converged else max(TOL, 0.1 * t.rho / t.snorm, t.ind / t.snorm)
    gmax = np.abs(b).max()
    errW = np.abs(a - b).max() / gmax
    Uh = lrp.tall_to_numpy(res2["Uhat"]); Vh = lrp.tall_to_numpy(res2["Vhat"]); Sh = res2["Shat"].cpu().numpy()
    It, Jt = t.I.astype(np.int64), t.J.astype(np.int64)
    colsG = (Uh * Sh) @ Vh[Jt].T; colsR = (ref.U * ref.S) @ ref.V[Jt].T
    rowsG = (Vh * Sh) @ Uh[It].T; rowsR = (ref.V * ref.S) @ ref.U[It].T
    ghat = max(np.abs(colsR).max(), np.abs(rowsR).max())
    errF = max(np.abs(colsG - colsR).max(), np.abs(rowsG - rowsR).max()) / ghat
    # numerical rank = #{S > 1e-14 S_1} (reading Q4): a singular value AT the cut may fall on either side; what differs must be there
    m = min(Sh.shape[0], ref.S.shape[0])
    assert abs(Sh.shape[0] - ref.S.shape[0]) <= 2 and (Sh[m:] <= 1e-13 * ref.S[0]).all() and (ref.S[m:] <= 1e-13 * ref.S[0]).all()
    errS = np.abs(Sh[:m] - ref.S[:m]).max() / ref.S[0]
    print(f"   replay parity: entries {errW:.2e} (tol {tolW:.1e}) selected fibers {errF:.2e} singular values {errS:.2e}")
    assert errW <= tolW and errF <= max(TOL, tolW) and errS <= max(TOL, tolW)
    if ref.converged:                                          # the GPU result against the matrix itself
        G = O.hilbert_entries(rows, cols) if kind == "hilbert" else O.kmatrix_entries(n, rows, cols)
        # the stop test of Alg. 4 is a heuristic: the oracle's own converged result may miss the matrix by more than tol
        # (K, n = 600, seed 1: 7e-4 at tol = 1e-6) -- the GPU result is held to the oracle's error
        eo, eg = np.abs(b - G).max(), np.abs(a - G).max()
        print(f"   error against the matrix itself: GPU {eg / gmax:.2e}  oracle {eo / gmax:.2e}  (tol {tol:.0e})")
        assert eg <= max(50 * tol * gmax, eo + tolW * gmax)


def test_matrix_call_argument_errors(ctx):
    import torch
    from paper_2607_06021_b200 import lrp
    n = 512
    U0, V0, sg = W.matrix_initial_guess(n, 4, 0)
    o = lrp.SolveOpts(); o.tol = 1e-9; o.max_rank = 16; o.oversample = 8; o.max_sweeps = 4      # no initial guess
    info = lrp.SolveInfo()
    ctx.ensure_workspace(ctx.lib.lrp_matrix_workspace_bytes(n, 4, 16, 8))
    out = torch.empty((16, n), dtype=torch.float64, device="cuda"); S = torch.empty(16, dtype=torch.float64, device="cuda")
    import ctypes as C
    rc = ctx.lib.lrp_cross_deim_matrix(ctx.h, lrp.LRP_G_HILBERT, n, C.byref(o), out.data_ptr(), n, S.data_ptr(), out.data_ptr(), n,
                                       C.byref(info), None, None, None, None, None, None, None, n)
    assert rc == lrp.LRP_ERR_BADARG
    with pytest.raises(lrp.LrpError):
        ctx.cross_deim_matrix(7, n, lrp.tall_from_numpy(U0), lrp.tall_from_numpy(V0), tol=1e-9, max_rank=16)
