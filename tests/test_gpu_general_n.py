"""NEXT-4 of SURVEY.md 8(f): general n (n + 1 not a power of two -- the paper's own grids are n = 2^10 .. 2^18,
PAPER.md:274), the paper's eq. (7) workload, and the dense full-rank DST solver of section 3.1
 as an on-GPU baseline."""
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


@pytest.mark.parametrize("n", [2, 5, 100, 127, 1000, 1024, 4095 + 1, 4097, 8000, 16384, 50000, 65536, 100003, 262144])
def test_dst1_general_n(ctx, n):
    """Bluestein DST-I: the shared-memory regime (P <= 8192, n <= 4095), the four-step regime above, primes and 2^p."""
    from paper_2607_06021_b200 import lrp
    x = W.dst_batch(n, 3, seed=n)
    got = lrp.tall_to_numpy(ctx.dst1_batched(lrp.tall_from_numpy(x), scale=0.5))
    ref = O.dst1(x, 0.5)                                       # definition sum for n <= 4095, odd-extension numpy.fft above
    assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max()
    # involution: the orthonormal transform applied twice is the identity
    sc = O.orthonormal_scale(n)
    t = lrp.tall_from_numpy(x)
    back = ctx.dst1_batched(ctx.dst1_batched(t, scale=sc), scale=sc)
    assert float((back - t).abs().max().item()) <= 1e-11 * np.abs(x).max()


def test_dst1_general_n_in_place_and_padded(ctx):
    import torch
    from paper_2607_06021_b200 import lrp
    n = 30000
    x = W.dst_batch(n, 5, seed=1)
    big = torch.zeros((5, n + 7), dtype=torch.float64, device="cuda"); big[:, :n] = lrp.tall_from_numpy(x)
    view = big[:, :n]
    ctx.dst1_batched(view, out=view)
    ref = O.dst1(x)
    assert np.abs(view.cpu().numpy().T - ref).max() <= 1e-11 * np.abs(ref).max()
    assert float(big[:, n:].abs().max().item()) == 0.0


def _solve(ctx, w, **kw):
    import torch
    from paper_2607_06021_b200 import lrp
    return ctx.cross_deim_solve(lrp.tall_from_numpy(w.UF), torch.from_numpy(w.SF).cuda(), lrp.tall_from_numpy(w.VF),
                                tol=w.tol, max_rank=w.max_rank, oversample=w.oversample, max_sweeps=w.max_sweeps,
                                safeguard=w.safeguard, want_spectral=True, **kw)


@pytest.mark.parametrize("n", [1000, 1 << 10, 1 << 14])
def test_paper_eq7_workload_at_general_n(ctx, n):
    """The paper's rank-1 Gaussian forcing (eq. (7)) on its own grid sizes: free-run decisions and replay parity vs the oracle."""
    from paper_2607_06021_b200 import lrp
    w = W.paper_eq7(n)
    ref = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, **w.opts())
    res = _solve(ctx, w)
    assert abs(res["sweeps"] - ref.sweeps) <= 1
    assert res["trace"][0]["I"].tolist() == ref.trace[0].I.tolist() and res["trace"][0]["J"].tolist() == ref.trace[0].J.tolist()
    rep = O.trace_to_replay(ref.trace, ref.rank)
    res2 = _solve(ctx, w, replay=rep)
    assert res2["rank"] == ref.rank
    rows, cols = W.sample_pairs(n, 4096, seed=1)
    UW, VW, SW = lrp.tall_to_numpy(res2["UW"]), lrp.tall_to_numpy(res2["VW"]), res2["SW"].cpu().numpy()
    a = np.einsum("tk,k,tk->t", UW[rows], SW, VW[cols]); b = O.lowrank_entries(ref.UW, ref.SW, ref.VW, rows, cols)
    t = ref.trace[-1]
    tolW = 1e-10 if ref.converged else max(1e-10, 0.1 * t.rho / t.snorm, t.ind / t.snorm)
    err = np.abs(a - b).max() / np.abs(b).max()
    print(f"eq7 n={n}: GPU {res['sweeps']} sweeps rank {res['rank']} conv {res['converged']}; oracle {ref.sweeps} sweeps rank {ref.rank} "
          f"conv {ref.converged}; replay parity {err:.2e}")
    assert err <= tolW
    # discrete residual of the returned solution at interior samples (meaningful for small n: it amplifies by 8/h^2)
    if n <= 1024:
        Wg = (UW * SW) @ VW.T
        F = (w.UF * w.SF) @ w.VF.T
        h2 = 1.0 / (n + 1) ** 2
        rng = np.random.default_rng(0)
        ii = rng.integers(1, n - 1, 300); jj = rng.integers(1, n - 1, 300)
        lap = (4 * Wg[ii, jj] - Wg[ii - 1, jj] - Wg[ii + 1, jj] - Wg[ii, jj - 1] - Wg[ii, jj + 1]) / h2
        assert np.abs(lap - F[ii, jj]).max() <= 8 * 50 * w.tol / h2 * np.linalg.norm(Wg)


@pytest.mark.parametrize("n", [255, 1000, 1023])
def test_dense_full_rank_solver_matches_oracle(ctx, n):
    """Section 3.1: W = Z (Z F Z ./ (d_i + d_j)) Z on the GPU vs the oracle's dense_poisson."""
    import torch
    rng = np.random.default_rng(n)
    F = rng.standard_normal((n, n))
    Wd = ctx.dense_poisson(torch.from_numpy(np.ascontiguousarray(F.T)).cuda()).cpu().numpy().T
    ref = O.dense_poisson(n, F)
    assert np.abs(Wd - ref).max() <= 1e-11 * np.abs(ref).max()


def test_low_rank_solve_agrees_with_the_dense_baseline_on_gpu(ctx):
    """The low-rank solve against the full-rank DST solve of the same right-hand side, both on the GPU (n = 4095, C2)."""
    import torch
    from paper_2607_06021_b200 import lrp
    w = W.make("C2", 0)
    res = _solve(ctx, w)
    F = (w.UF * w.SF) @ w.VF.T
    Wd = ctx.dense_poisson(torch.from_numpy(np.ascontiguousarray(F.T)).cuda())          # Wd[j, i] = W(i, j)
    Wl = (res["VW"].T * res["SW"]) @ res["UW"]                                              # (n, n) with [j, i] = sum_k V(j,k) S_k U(i,k)
    nrm = float(torch.linalg.matrix_norm(Wd).item())
    assert float(torch.linalg.matrix_norm(Wl - Wd).item()) <= 20 * w.tol * nrm
