"""Index selection on the GPU: the sort-based top-k at sizes spanning several chunks and levels, and the randomized
(Bernoulli) leverage sampling of Alg. 3 lines 4-5 (NEXT-2 of SURVEY.md 8(f)) against the oracle:
the same counter-based uniforms on both sides, selections equal as ordered lists, solve parity under replay."""
import numpy as np
import pytest

from oracle import lrp_oracle as O
from paper_2607_06021_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from paper_2607_06021_b200 import build, lrp
    build.build()
    c = lrp.Context(0)
    yield c
    c.close()


@pytest.mark.parametrize("n,num", [(100, 100), (8192, 17), (8193, 50), (65535, 300), ((1 << 20) - 1, 49), ((1 << 20) + 5, 2000),
                                   ((1 << 22) - 1, 545)])
def test_topk_matches_full_sort(ctx, n, num):
    """(score desc, index asc) order, bit-exact, with heavy ties (quantised scores) and several reduction levels."""
    import torch
    from paper_2607_06021_b200 import lrp
    rng = np.random.default_rng(n + num)
    sc = np.floor(rng.random(n) * 1000.0) / 1000.0 * np.exp(-np.arange(n) / (n / 3.0))       # ties + decay
    sc[rng.integers(0, n, 5)] = 2.0                                                            # a few exact ties at the top
    A = np.sqrt(sc)[:, None]                                                                   # one column: row norm^2 = sc
    idx, got_sc = ctx.leverage_select(lrp.tall_from_numpy(A), num, assume_orthonormal=True)
    got_sc = got_sc.cpu().numpy()
    ref = O.top_select(got_sc, num)                          # the oracle's order on the SAME scores (sqrt/square round trip)
    assert idx.cpu().numpy().tolist() == ref.tolist()


@pytest.mark.parametrize("n,num,kind", [(100_000, 50, "flat"), ((1 << 20) - 1, 300, "flat"), (300_000, 4096, "two_levels"),
                                        (50_000, 64, "narrow"), (9000, 9000 // 3, "flat")])
def test_topk_flat_distributions_take_the_multi_level_sort(ctx, n, num, kind):
    """More than 4096 keys share the threshold bin of the histogram pass (equal scores; scores within one 2^(1/4) band):
    the device-side flag routes the call to the multi-level sort.  Same bit-exact order."""
    from paper_2607_06021_b200 import lrp
    rng = np.random.default_rng(n)
    if kind == "flat":
        sc = np.full(n, 0.25)
    elif kind == "narrow":
        sc = 0.5 + 0.01 * rng.random(n)                                   # all inside one bin, no ties
    else:
        sc = np.where(np.arange(n) % 7 == 0, 0.5, 0.25 + 1e-3 * rng.random(n))   # 1/7 in a higher bin (> 4096 of them), rest flat
    A = np.sqrt(sc)[:, None]
    idx, got_sc = ctx.leverage_select(lrp.tall_from_numpy(A), num, assume_orthonormal=True)
    ref = O.top_select(got_sc.cpu().numpy(), num)
    assert idx.cpu().numpy().tolist() == ref.tolist()


def _solve(ctx, w, **kw):
    import torch
    from paper_2607_06021_b200 import lrp
    return ctx.cross_deim_solve(lrp.tall_from_numpy(w.UF), torch.from_numpy(w.SF).cuda(), lrp.tall_from_numpy(w.VF),
                                tol=w.tol, max_rank=w.max_rank, oversample=w.oversample, max_sweeps=w.max_sweeps,
                                safeguard=w.safeguard, want_spectral=True, **kw)


@pytest.mark.parametrize("cfg,n,seed,ls_seed", [("C2", None, 0, 11), ("C3", 16383, 0, 3), ("C4", 16383, 0, 5)])
def test_bernoulli_selection_free_run_and_replay(ctx, cfg, n, seed, ls_seed):
    from paper_2607_06021_b200 import lrp
    w = W.make(cfg, seed, n)
    w.max_sweeps = 12
    ref = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, selection="bernoulli", ls_seed=ls_seed, **w.opts())
    res = _solve(ctx, w, selection="bernoulli", ls_seed=ls_seed)
    # sweep 0: the draws depend on the leverage scores of the RHS factors only.  A decision u < p is "clear" unless |u - p|
    # is at rounding level; with clear decisions the ordered lists must be equal
    t0 = ref.trace[0]
    for side, (sc, star) in enumerate(((t0.scoresU, t0.Istar), (t0.scoresV, t0.Jstar))):
        cols = w.rF
        p = np.minimum(1.0, (cols + w.oversample) * (sc / cols))
        u = O.counter_uniforms(ls_seed, 0, side, w.n)
        assert np.abs(u - p)[p > 0].min() > 1e-12
    g0 = res["trace"][0]
    assert g0["I"].tolist() == t0.I.tolist() and g0["J"].tolist() == t0.J.tolist()
    print(f"{cfg} n={w.n}: bernoulli GPU {res['sweeps']} sweeps rank {res['rank']} conv {res['converged']}; oracle {ref.sweeps} "
          f"sweeps rank {ref.rank} conv {ref.converged}; |I_0| = {len(t0.I)}")
    assert abs(res["sweeps"] - ref.sweeps) <= 1
    # replay of the oracle's trace on the GPU: continuous parity at 1e-10
    rep = O.trace_to_replay(ref.trace, ref.rank)
    res2 = _solve(ctx, w, replay=rep)
    rows, cols_ = W.sample_pairs(w.n, 4096, seed=1)
    UW, VW, SW = lrp.tall_to_numpy(res2["UW"]), lrp.tall_to_numpy(res2["VW"]), res2["SW"].cpu().numpy()
    a = np.einsum("tk,k,tk->t", UW[rows], SW, VW[cols_]); b = O.lowrank_entries(ref.UW, ref.SW, ref.VW, rows, cols_)
    t = ref.trace[-1]
    tolW = 1e-10 if ref.converged else max(1e-10, 0.1 * t.rho / t.snorm, t.ind / t.snorm)
    assert np.abs(a - b).max() <= tolW * np.abs(b).max()
    assert np.abs(res2["Shat"].cpu().numpy() - ref.Shat).max() <= 1e-10 * ref.Shat[0]


def test_bernoulli_escapes_the_stall_on_the_gpu(ctx):
    """Same statement as tests/test_oracle_options.py::test_bernoulli_selection_escapes_the_deterministic_stall, on the
    GPU path: the deterministic form stalls on this Hilbert case, the Bernoulli form converges."""
    from paper_2607_06021_b200 import lrp
    n = 1024
    U0, V0, sg = W.matrix_initial_guess(n, 4, 1)
    kw = dict(tol=1e-9, max_rank=64, oversample=8, max_sweeps=12, safeguard=sg)
    det = ctx.cross_deim_matrix("hilbert", n, lrp.tall_from_numpy(U0), lrp.tall_from_numpy(V0), **kw)
    rnd = ctx.cross_deim_matrix("hilbert", n, lrp.tall_from_numpy(U0), lrp.tall_from_numpy(V0), selection="bernoulli", ls_seed=7, **kw)
    assert not det["converged"] and rnd["converged"] and rnd["sweeps"] <= 8
    rows, cols = W.sample_pairs(n, 4096, seed=2)
    U, V, S = lrp.tall_to_numpy(rnd["UW"]), lrp.tall_to_numpy(rnd["VW"]), rnd["SW"].cpu().numpy()
    a = np.einsum("tk,k,tk->t", U[rows], S, V[cols])
    assert np.abs(a - O.hilbert_entries(rows, cols)).max() <= 5e-8


@pytest.mark.parametrize("sel", ["qdeim", "deim"])
@pytest.mark.parametrize("kind,n,seed", [("hilbert", 1024, 1), ("hilbert", 777, 0), ("kmatrix", 512, 0)])
def test_deim_variants_on_test_matrices(ctx, sel, kind, n, seed):
    """NEXT-3 of SURVEY.md 8(f): QDEIM (column-pivoted QR of U^T) and DEIM (pivoted LU) selection, Alg. 2, as
    hand-written kernels (the paper had to leave them to JAX / MAGMA).  Free run: the ordered pivot lists
    of the first sweeps equal the oracle's (pivot gaps of these generic matrices are far above rounding); replay: 1e-10."""
    from paper_2607_06021_b200 import lrp
    tol = 1e-9 if kind == "hilbert" else 1e-6
    U0, V0, sg = W.matrix_initial_guess(n, 4, seed)
    kw = dict(tol=tol, max_rank=64, oversample=8, max_sweeps=10, safeguard=sg)
    ref = O.cross_deim(n, O.matrix_fibers(kind, n), U0, V0, selection=sel, **kw)
    res = ctx.cross_deim_matrix(kind, n, lrp.tall_from_numpy(U0), lrp.tall_from_numpy(V0), selection=sel, want_spectral=True, **kw)
    same = 0
    for s in range(min(res["sweeps"], ref.sweeps)):
        if res["trace"][s]["I"].tolist() != ref.trace[s].I.tolist() or res["trace"][s]["J"].tolist() != ref.trace[s].J.tolist():
            break
        same += 1
    print(f"{kind} n={n} {sel}: GPU {res['sweeps']} sweeps rank {res['rank']} conv {res['converged']}; oracle {ref.sweeps} sweeps rank "
          f"{ref.rank} conv {ref.converged}; identical index lists on the first {same} sweeps")
    assert same >= 2                                           # sweep 0 (random initial guess) and sweep 1 at least
    assert abs(res["sweeps"] - ref.sweeps) <= 1
    rep = O.trace_to_replay(ref.trace, ref.rank)
    res2 = ctx.cross_deim_matrix(kind, n, lrp.tall_from_numpy(U0), lrp.tall_from_numpy(V0), replay=rep, want_spectral=True, **kw)
    rows, cols = W.sample_pairs(n, 4096, seed=4)
    U, V, S = lrp.tall_to_numpy(res2["UW"]), lrp.tall_to_numpy(res2["VW"]), res2["SW"].cpu().numpy()
    a = np.einsum("tk,k,tk->t", U[rows], S, V[cols])
    b = O.lowrank_entries(ref.U[:, :ref.rank], ref.S[:ref.rank], ref.V[:, :ref.rank], rows, cols)
    t = ref.trace[-1]
    tolW = 1e-10 if ref.converged else max(1e-10, 0.1 * t.rho / t.snorm, t.ind / t.snorm)
    assert np.abs(a - b).max() <= tolW * np.abs(b).max(), (np.abs(a - b).max() / np.abs(b).max(), tolW)


@pytest.mark.parametrize("sel", ["qdeim", "deim"])
def test_deim_variants_on_the_poisson_solve(ctx, sel):
    from paper_2607_06021_b200 import lrp
    w = W.make("C4", 0, 16383)
    w.max_sweeps = 6
    ref = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, selection=sel, **w.opts())
    res = _solve(ctx, w, selection=sel)
    for s in range(2):
        assert res["trace"][s]["I"].tolist() == ref.trace[s].I.tolist() and res["trace"][s]["J"].tolist() == ref.trace[s].J.tolist()
    rep = O.trace_to_replay(ref.trace, ref.rank)
    res2 = _solve(ctx, w, replay=rep)
    rows, cols_ = W.sample_pairs(w.n, 4096, seed=1)
    UW, VW, SW = lrp.tall_to_numpy(res2["UW"]), lrp.tall_to_numpy(res2["VW"]), res2["SW"].cpu().numpy()
    a = np.einsum("tk,k,tk->t", UW[rows], SW, VW[cols_]); b = O.lowrank_entries(ref.UW, ref.SW, ref.VW, rows, cols_)
    t = ref.trace[-1]
    tolW = 1e-10 if ref.converged else max(1e-10, 0.1 * t.rho / t.snorm, t.ind / t.snorm)
    assert np.abs(a - b).max() <= tolW * np.abs(b).max()
