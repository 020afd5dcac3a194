"""GPU parity of lrp_cross_deim_solve against the CPU oracle: free-running (discrete decisions compared)
and under replay in both directions (continuous parity <= 1e-10 on reconstructed entries and selected fibers)."""
import numpy as np
import pytest

from oracle import lrp_oracle as O
from paper_2607_06021_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-10          # north_star: relative error <= 1e-10 on reconstructed solution entries


@pytest.fixture(scope="module")
def ctx():
    from paper_2607_06021_b200 import build, lrp
    build.build()
    c = lrp.Context(0)
    yield c
    c.close()


def _gpu_solve(ctx, w, **kw):
    import torch
    from paper_2607_06021_b200 import lrp
    return ctx.cross_deim_solve(lrp.tall_from_numpy(w.UF), torch.from_numpy(w.SF).cuda(), lrp.tall_from_numpy(w.VF),
                                tol=w.tol, max_rank=w.max_rank, oversample=w.oversample, max_sweeps=w.max_sweeps,
                                safeguard=w.safeguard, want_spectral=True, **kw)


def _entries(U, S, V, rows, cols):
    return np.einsum("tk,k,tk->t", U[rows], S, V[cols])


def _parity_tol(ref):
    """Tolerance on PHYSICAL-space entries: 1e-10 when the stop test passed.  A run that the sweep cap ends first (C3 as
    configured: 5 sweeps) still has a residual of size rho; the final truncation then cuts singular values that are not
    yet resolved, and two fp64 implementations differ by a fraction of rho / ||S|| on W -- DESIGN.md reading R1, shown on
    the oracle itself (Householder vs LAPACK QR under replay) in
    tests/test_oracle_solve.py::test_unconverged_run_sensitivity.  Bound: max(1e-10, 0.1 rho/||S||) (C3: 2.7e-10,
    measured 1.4e-10).  Singular values and selected fibers are held to 1e-10 in every case."""
    t = ref.trace[-1]
    return TOL if ref.converged else max(TOL, 0.1 * t.rho / t.snorm)


def _continuous_parity(res, ref, w, replay_sets, tol=None):
    from paper_2607_06021_b200 import lrp
    n = w.n
    tolW = tol if tol is not None else _parity_tol(ref)
    UW, VW, SW = lrp.tall_to_numpy(res["UW"]), lrp.tall_to_numpy(res["VW"]), res["SW"].cpu().numpy()
    assert res["rank"] == ref.rank
    rows, cols = W.sample_pairs(n, 4096, seed=1)
    a = _entries(UW, SW, VW, rows, cols); b = _entries(ref.UW, ref.SW, ref.VW, rows, cols)
    wmax = np.abs(b).max()                                   # max |W| over the 4096 samples of the smooth solution
    assert np.abs(a - b).max() <= tolW * wmax, (np.abs(a - b).max() / wmax, tolW)
    # all selected fibers of the spectral iterate
    Uh, Vh, Sh = lrp.tall_to_numpy(res["Uhat"]), lrp.tall_to_numpy(res["Vhat"]), res["Shat"].cpu().numpy()
    assert Uh.shape[1] == ref.Uhat.shape[1]
    I, J = replay_sets
    colsG = (Uh * Sh) @ Vh[J].T; colsR = (ref.Uhat * ref.Shat) @ ref.Vhat[J].T
    rowsG = (Vh * Sh) @ Uh[I].T; rowsR = (ref.Vhat * ref.Shat) @ ref.Uhat[I].T
    ghat = max(np.abs(colsR).max(), np.abs(rowsR).max())      # max |What| (the selected fibers carry it)
    assert np.abs(colsG - colsR).max() <= TOL * ghat and np.abs(rowsG - rowsR).max() <= TOL * ghat
    assert np.abs(Sh - ref.Shat).max() <= TOL * ref.Shat[0]


# (config, seed, n override, max_sweeps override).  C3 is run as configured (5 sweeps: the cap ends it unconverged;
# with more sweeps the oracle itself stagnates at rho ~ 2e-10 ||S||).
CASES = [("C1", 0, None, None), ("C1", 3, None, None), ("C2", 0, None, None), ("C2", 1, None, None),
         ("C3", 0, None, None), ("C2", 2, None, None), ("C4", 0, (1 << 14) - 1, None)]


@pytest.mark.parametrize("name,seed,n,sweeps", CASES)
def test_solve_free_run_and_replay(ctx, name, seed, n, sweeps):
    w = W.make(name, seed, n)
    if sweeps:
        w.max_sweeps = sweeps
    ref = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, **w.opts())
    res = _gpu_solve(ctx, w)
    # ---- discrete parity of the free run: ordered selections equal where the deciding leverage gaps exceed 1e-12
    same = res["sweeps"] == ref.sweeps
    nchk = min(res["sweeps"], ref.sweeps)
    clear = True
    for s in range(nchk):
        t = ref.trace[s]
        for sc, star in ((t.scoresU, t.Istar), (t.scoresV, t.Jstar)):
            srt = np.sort(sc)[::-1][:len(star) + 1]
            clear &= bool(np.abs(np.diff(srt)).min() > 1e-12)
        rr = t.rR / t.rR.max(); rc = t.rC / t.rC.max()
        clear &= not (((rr > 1e-13) & (rr < 1e-11)).any() or ((rc > 1e-13) & (rc < 1e-11)).any())
        if not clear:
            break
        g = res["trace"][s]
        assert g["I"].tolist() == t.I.tolist() and g["J"].tolist() == t.J.tolist(), f"sweep {s}"
        assert g["keepI"].tolist() == t.keepI.tolist() and g["keepJ"].tolist() == t.keepJ.tolist()
        assert g["rank"] == t.rank
    # sweep count may differ by one when rho / indicator sits within 10x of the threshold
    assert abs(res["sweeps"] - ref.sweeps) <= 1
    if clear and same:
        assert res["converged"] == ref.converged
        _continuous_parity(res, ref, w, (ref.trace[-1].I, ref.trace[-1].J))
    else:       # decisions inside the tolerance bands: the free runs took different (equally valid) index sets
        print(f"{name} seed {seed}: free-run continuous comparison not applicable (clear={clear}, same sweeps={same}); "
              f"replay parity below covers it")
    # ---- replay oracle -> GPU
    rep = O.trace_to_replay(ref.trace, ref.rank)
    res2 = _gpu_solve(ctx, w, replay=rep)
    assert res2["sweeps"] == ref.sweeps
    _continuous_parity(res2, ref, w, (ref.trace[-1].I, ref.trace[-1].J))
    # ---- replay GPU -> oracle
    rep_g = [dict(I=t["I"], J=t["J"], keepI=t["keepI"], keepJ=t["keepJ"]) for t in res["trace"]]
    rep_g[-1]["final_rank"] = res["rank"]
    ref2 = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, replay=rep_g, **w.opts())
    _continuous_parity(res, ref2, w, (res["trace"][-1]["I"], res["trace"][-1]["J"]), tol=_parity_tol(ref))


def test_c1_closed_form_on_gpu(ctx):
    """sin(k pi x) sin(l pi y) forcing: exact solution f / (d_k + d_l), exact rank 4 (north_star pin, on the GPU path)."""
    import math
    from paper_2607_06021_b200 import lrp
    w = W.config1(5)
    res = _gpu_solve(ctx, w)
    assert res["rank"] == 4 and res["converged"]
    x = W.grid(w.n)
    dk = lambda k: 4.0 * (w.n + 1) ** 2 * math.sin(math.pi * k / (2 * (w.n + 1))) ** 2
    Wex = sum(w.meta["a"][m] * np.outer(np.sin(math.pi * w.meta["k"][m] * x), np.sin(math.pi * w.meta["l"][m] * x))
              / (dk(int(w.meta["k"][m])) + dk(int(w.meta["l"][m]))) for m in range(4))
    Wg = (lrp.tall_to_numpy(res["UW"]) * res["SW"].cpu().numpy()) @ lrp.tall_to_numpy(res["VW"]).T
    assert np.abs(Wg - Wex).max() < 5e-12 * np.abs(Wex).max()


def test_solve_argument_errors(ctx):
    import torch
    from paper_2607_06021_b200 import lrp
    w = W.config1(0)
    UF = lrp.tall_from_numpy(w.UF); VF = lrp.tall_from_numpy(w.VF); SF = torch.from_numpy(w.SF).cuda()
    with pytest.raises(lrp.LrpError) as e:
        ctx.cross_deim_solve(UF, SF, VF, tol=-1.0, max_rank=16)
    assert e.value.code == lrp.LRP_ERR_BADARG
    # general n is supported (Bluestein); beyond n + 1 = 2^23 it is not
    assert ctx.lib.lrp_dst1_workspace_bytes((1 << 23) + 1, 1) == 0
    # max_sweeps = 1 cannot pass the stop test -> warning code, outputs still valid
    r = ctx.cross_deim_solve(UF, SF, VF, tol=1e-12, max_rank=16, max_sweeps=1, safeguard=w.safeguard)
    assert r["code"] == lrp.LRP_WARN_NOCONV and r["rank"] >= 1


def test_rank_cap_returns_noconv_warning(ctx):
    """r* > r_max (Alg. 4 line 31): the result is truncated to r_max and the tolerance is not met --
    reading Q20: LRP_WARN_NOCONV and converged = 0, as the oracle's rank_capped flag."""
    from paper_2607_06021_b200 import lrp
    w = W.make("C2", 0)
    w.max_rank = 6
    ref = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, **w.opts())
    assert ref.rank == 6 and ref.rank_capped
    res = _gpu_solve(ctx, w)
    assert res["rank"] == 6 and res["code"] == lrp.LRP_WARN_NOCONV and not res["converged"]
    assert np.abs(res["SW"].cpu().numpy() - ref.SW).max() <= 1e-6 * ref.SW[0]


def test_first_selection_must_fit_the_set_cap(ctx):
    """K_cap = 2 (r_max + p_os) (reading Q10) as in the oracle; a right-hand side whose first selection
    (rF + p_os indices + safeguard) does not fit is rejected instead of silently enlarging the cap."""
    import torch
    from paper_2607_06021_b200 import lrp
    w = W.make("C4", 0, 1023)                  # rF = 32
    UF = lrp.tall_from_numpy(w.UF); VF = lrp.tall_from_numpy(w.VF); SF = torch.from_numpy(w.SF).cuda()
    assert ctx.lib.lrp_workspace_bytes(w.n, w.rF, 8, 8) == 0           # 2 (8 + 8) = 32 < 32 + 8 + 1
    with pytest.raises(lrp.LrpError) as e:
        ctx.cross_deim_solve(UF, SF, VF, tol=1e-8, max_rank=8, oversample=8)
    assert e.value.code == lrp.LRP_ERR_BADARG
    ok = ctx.cross_deim_solve(UF, SF, VF, tol=1e-8, max_rank=13, oversample=8, safeguard=w.safeguard)   # 42 >= 41
    assert ok["rank"] <= 13
