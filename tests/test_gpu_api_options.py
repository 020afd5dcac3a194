"""Options of lrp_cross_deim_solve on the GPU: warm start (U0, V0), absolute tolerance mode, padded leading dimensions,
a non-default stream, the K_cap truncation, and the trace/replay hook with the GPU's own trace."""
import numpy as np
import pytest

from oracle import lrp_oracle as O
from paper_2607_06021_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _entries(U, S, V, rows, cols):
    return np.einsum("tk,k,tk->t", U[rows], S, V[cols])


@pytest.fixture(scope="module")
def ctx():
    from paper_2607_06021_b200 import build, lrp
    build.build()
    c = lrp.Context(0)
    yield c
    c.close()


def _solve(ctx, w, **kw):
    import torch
    from paper_2607_06021_b200 import lrp
    args = dict(tol=w.tol, max_rank=w.max_rank, oversample=w.oversample, max_sweeps=w.max_sweeps, safeguard=w.safeguard)
    args.update(kw)
    return ctx.cross_deim_solve(lrp.tall_from_numpy(w.UF), torch.from_numpy(w.SF).cuda(), lrp.tall_from_numpy(w.VF), **args)


def test_warm_start_matches_oracle_and_saves_sweeps(ctx):
    """Alg. 4 takes U0, V0: restarting from a converged spectral iterate selects the same
    well-placed indices at once (warm start)."""
    from paper_2607_06021_b200 import lrp
    w = W.make("C2", 0)
    cold = _solve(ctx, w, want_spectral=True)
    warm = _solve(ctx, w, U0=cold["Uhat"], V0=cold["Vhat"], want_spectral=True)
    assert warm["converged"] and warm["sweeps"] <= cold["sweeps"]
    ref = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, U0=lrp.tall_to_numpy(cold["Uhat"]), V0=lrp.tall_to_numpy(cold["Vhat"]), **w.opts())
    assert abs(warm["sweeps"] - ref.sweeps) <= 1 and abs(warm["rank"] - ref.rank) <= 1
    rows, cols = W.sample_pairs(w.n, 4096, seed=2)
    a = _entries(lrp.tall_to_numpy(warm["UW"]), warm["SW"].cpu().numpy(), lrp.tall_to_numpy(warm["VW"]), rows, cols)
    b = O.lowrank_entries(ref.UW, ref.SW, ref.VW, rows, cols)
    assert np.abs(a - b).max() <= 20 * w.tol * np.abs(b).max()


def test_absolute_tolerance_mode(ctx):
    """tol_mode = 1: the thresholds of Alg. 4 lines 26 and 30 exactly as printed (absolute), reading Q15."""
    from paper_2607_06021_b200 import lrp
    w = W.make("C1", 1)
    kw = dict(tol=1e-9, tol_mode=1)
    res = _solve(ctx, w, **kw)
    opts = w.opts(); opts["tol"] = 1e-9
    ref = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, tol_mode=1, **opts)
    assert res["converged"] == ref.converged and res["rank"] == ref.rank and res["sweeps"] == ref.sweeps
    Wg = (lrp.tall_to_numpy(res["UW"]) * res["SW"].cpu().numpy()) @ lrp.tall_to_numpy(res["VW"]).T
    Wo = (ref.UW * ref.SW) @ ref.VW.T
    assert np.abs(Wg - Wo).max() <= 1e-10 * np.abs(Wo).max()


def test_padded_leading_dimensions_and_side_stream(ctx):
    import torch
    from paper_2607_06021_b200 import lrp
    w = W.make("C1", 2)
    n, rF = w.n, w.rF
    base = _solve(ctx, w)
    big_u = torch.zeros((rF, n + 13), dtype=torch.float64, device="cuda"); big_u[:, :n] = lrp.tall_from_numpy(w.UF)
    big_v = torch.zeros((rF, n + 5), dtype=torch.float64, device="cuda"); big_v[:, :n] = lrp.tall_from_numpy(w.VF)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        c2 = lrp.Context(0)                      # bound to the side stream
        res = c2.cross_deim_solve(big_u[:, :n], torch.from_numpy(w.SF).cuda(), big_v[:, :n], tol=w.tol, max_rank=w.max_rank,
                                  oversample=w.oversample, max_sweeps=w.max_sweeps, safeguard=w.safeguard)
        c2.close()
    s.synchronize()
    assert res["rank"] == base["rank"] and res["sweeps"] == base["sweeps"]
    assert torch.equal(res["SW"], base["SW"])     # same kernels, same inputs: bit-identical singular values
    assert float((res["UW"] - base["UW"]).abs().max().item()) == 0.0


def test_set_cap_truncation_and_gpu_trace_replay(ctx):
    """A tiny rank cap forces the K_cap = 2 (r_max + p_os) truncation of reading Q10; the GPU's own trace replays
    bit-for-bit on the GPU (the replay hook takes exactly the recorded decisions)."""
    import torch
    w = W.make("C2", 1)
    w.max_rank, w.oversample, w.max_sweeps = 4, 2, 6
    res = _solve(ctx, w, want_spectral=True)
    kcap = 2 * (w.max_rank + w.oversample)
    assert all(len(t["I"]) <= kcap and len(t["J"]) <= kcap for t in res["trace"])
    assert res["rank"] <= w.max_rank
    ref = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, **w.opts())
    assert [len(t.I) for t in ref.trace][:2] == [len(t["I"]) for t in res["trace"]][:2]
    rep = [dict(I=t["I"], J=t["J"], keepI=t["keepI"], keepJ=t["keepJ"]) for t in res["trace"]]
    rep[-1]["final_rank"] = res["rank"]
    again = _solve(ctx, w, replay=rep, want_spectral=True)
    assert again["sweeps"] == res["sweeps"] and again["rank"] == res["rank"]
    assert torch.equal(again["Shat"], res["Shat"])


def test_fused_and_two_sweep_stop_test_agree(ctx):
    """rho (Alg. 4 line 24) through the fused residual-Gram kernel (E = U_{k-1} - U_k A never written)
    and through the update sweep + Gram sweep it replaces (shapes outside the fused kernel's range take that path):
    the same sweeps, ranks and index decisions, rho equal to rounding of a sum of squares."""
    w = W.make("C2", 3)
    from paper_2607_06021_b200 import lrp
    a = _solve(ctx, w)
    b = _solve(ctx, w, flags=lrp.LRP_FLAG_NO_FUSED_RHO)
    assert a["sweeps"] == b["sweeps"] and a["rank"] == b["rank"] and a["converged"] == b["converged"]
    ia, ib = a["info"], b["info"]
    for k in range(a["sweeps"]):
        ra, rb = ia.rho_per_sweep[k], ib.rho_per_sweep[k]
        assert abs(ra - rb) <= 1e-9 * max(abs(ra), abs(rb)) + 1e-13 * ia.snorm
        assert ia.rank_per_sweep[k] == ib.rank_per_sweep[k] and ia.nI[k] == ib.nI[k] and ia.nJ[k] == ib.nJ[k]


@pytest.mark.parametrize("cfg,seed,nred", [("C2", 0, None), ("C2", 3, None), ("C3", 0, 16383), ("C4", 0, 32767)])
def test_qr_prefix_reuse_matches_full_factorization(ctx, cfg, seed, nred):
    """Fibers of surviving indices do not change between sweeps (G-hat is fixed, eq. (4)) and the QR of a
    column prefix is the prefix of the QR, so the driver keeps the Q columns of the common prefix of consecutive index
    lists and factors only the new fibers.  Against factoring every block from scratch (LRP_FLAG_NO_QR_REUSE): the same
    index decisions in the first sweeps, the same rank, and reconstructed entries equal to the parity tolerance."""
    from paper_2607_06021_b200 import lrp
    w = W.make(cfg, seed) if nred is None else W.make(cfg, seed, nred)
    a = _solve(ctx, w)
    b = _solve(ctx, w, flags=lrp.LRP_FLAG_NO_QR_REUSE)
    assert abs(a["sweeps"] - b["sweeps"]) <= 1 and a["rank"] == b["rank"]
    for ta, tb in list(zip(a["trace"], b["trace"]))[:2]:
        assert list(ta["I"]) == list(tb["I"]) and list(ta["J"]) == list(tb["J"])
    rows, cols = W.sample_pairs(w.n, 4096, seed=5)
    ea = _entries(lrp.tall_to_numpy(a["UW"]), a["SW"].cpu().numpy(), lrp.tall_to_numpy(a["VW"]), rows, cols)
    eb = _entries(lrp.tall_to_numpy(b["UW"]), b["SW"].cpu().numpy(), lrp.tall_to_numpy(b["VW"]), rows, cols)
    tol = 1e-10 if (a["converged"] and b["converged"]) else max(1e-10, 0.1 * max(a["info"].rho, b["info"].rho) / a["info"].snorm)
    assert np.abs(ea - eb).max() <= tol * np.abs(eb).max()
    assert a["info"].launches < b["info"].launches


@pytest.mark.parametrize("cfg,seed,nred", [("C2", 0, None), ("C3", 0, 16383), ("C4", 0, 32767), ("C4", 1, 262143)])
def test_cholesky_qr_leverage_of_the_initial_guess_matches_householder(ctx, cfg, seed, nred):
    """Leverage scores are the diagonal of the projector onto span(U_0) (Alg. 3 lines 1-3): whichever
    orthonormal basis is used.  The driver takes CholeskyQR2 for a well-conditioned initial guess (reading R8)
    and the Householder TSQR otherwise (LRP_FLAG_NO_CHOLQR_LEVERAGE forces it): same first selection, same run."""
    from paper_2607_06021_b200 import lrp
    w = W.make(cfg, seed) if nred is None else W.make(cfg, seed, nred)
    a = _solve(ctx, w)
    b = _solve(ctx, w, flags=lrp.LRP_FLAG_NO_CHOLQR_LEVERAGE)
    assert list(a["trace"][0]["I"]) == list(b["trace"][0]["I"]) and list(a["trace"][0]["J"]) == list(b["trace"][0]["J"])
    assert a["sweeps"] == b["sweeps"] and a["rank"] == b["rank"] and a["converged"] == b["converged"]
    rows, cols = W.sample_pairs(w.n, 4096, seed=5)
    ea = _entries(lrp.tall_to_numpy(a["UW"]), a["SW"].cpu().numpy(), lrp.tall_to_numpy(a["VW"]), rows, cols)
    eb = _entries(lrp.tall_to_numpy(b["UW"]), b["SW"].cpu().numpy(), lrp.tall_to_numpy(b["VW"]), rows, cols)
    tol = 1e-10 if (a["converged"] and b["converged"]) else max(1e-10, 0.1 * max(a["info"].rho, b["info"].rho) / a["info"].snorm)
    assert np.abs(ea - eb).max() <= tol * np.abs(eb).max()
    assert a["info"].launches < b["info"].launches


@pytest.mark.parametrize("cfg,seed,nred", [("C2", 3, None), ("C4", 0, 32767)])
def test_nested_stop_test_matches_tall_contractions(ctx, cfg, seed, nred):
    """rho (Alg. 4 line 24) when last sweep's index lists are prefixes of this sweep's: U_{k-1} lies in
    span(Q_k), so rho follows from the small core factors alone; with a few dropped trailing indices (the pruned
    safeguard of sweep 0) U_{k-1} = Q_k Y + P Uc_rest with the dropped Q columns set aside (three narrow passes).
    Against the general path (contractions over the tall
    iterates, LRP_FLAG_NO_NESTED_RHO): same decisions, rho equal up to the orthonormality of the GPU's Q.  Both forms assume
    Q^T Q = I, which the thin QR delivers to ~1e-15 (every panel is re-orthogonalised after its factorization, DESIGN.md
    "Thin QR"), so the two rho agree to rounding of ||S||."""
    w = W.make(cfg, seed) if nred is None else W.make(cfg, seed, nred)
    from paper_2607_06021_b200 import lrp
    a = _solve(ctx, w)
    b = _solve(ctx, w, flags=lrp.LRP_FLAG_NO_NESTED_RHO)
    assert a["sweeps"] == b["sweeps"] and a["rank"] == b["rank"] and a["converged"] == b["converged"]
    ia, ib = a["info"], b["info"]
    for k in range(a["sweeps"]):
        ra, rb = ia.rho_per_sweep[k], ib.rho_per_sweep[k]
        assert abs(ra - rb) <= 1e-6 * max(abs(ra), abs(rb)) + 2e-13 * ia.snorm
        assert ia.rank_per_sweep[k] == ib.rank_per_sweep[k] and ia.nI[k] == ib.nI[k] and ia.nJ[k] == ib.nJ[k]
