"""Edge and degenerate cases of the C-ABI calls on the GPU (empty / minimal / ragged inputs, argument errors, the
paper's own rank-1 separable Gaussian right-hand side)."""
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


def test_sample_fibers_minimal_sets(ctx):
    import torch
    from paper_2607_06021_b200 import lrp
    n, r = 1023, 3
    rng = np.random.default_rng(1)
    Uh = rng.standard_normal((n, r)); Vh = rng.standard_normal((n, r)); S = np.array([3.0, 2.0, 1.0])
    d = O.eigenvalues_d(n)
    I = np.array([n - 1], dtype=np.int32); J = np.array([0], dtype=np.int32)
    Cref, Rref = O.sample_fibers(Uh, S, Vh, d, I, J)
    Cg, Rg = ctx.sample_fibers(lrp.tall_from_numpy(Uh), torch.from_numpy(S).cuda(), lrp.tall_from_numpy(Vh),
                               torch.from_numpy(I).cuda(), torch.from_numpy(J).cuda())
    assert np.abs(lrp.tall_to_numpy(Cg) - Cref).max() < 1e-13 * np.abs(Cref).max()
    assert np.abs(lrp.tall_to_numpy(Rg) - Rref).max() < 1e-13 * np.abs(Rref).max()
    # empty index lists produce empty outputs and no error
    e = torch.zeros(0, dtype=torch.int32, device="cuda")
    Cg, Rg = ctx.sample_fibers(lrp.tall_from_numpy(Uh), torch.from_numpy(S).cuda(), lrp.tall_from_numpy(Vh), e, e)
    assert Cg.shape == (0, n) and Rg.shape == (0, n)


def test_leverage_select_extremes(ctx):
    from paper_2607_06021_b200 import lrp
    n = 255
    rng = np.random.default_rng(2)
    A = rng.standard_normal((n, 1))
    idx, sc = ctx.leverage_select(lrp.tall_from_numpy(A), n)            # select everything: a full sort
    ref_idx, ref_sc = O.leverage_select(A, n)
    assert np.abs(sc.cpu().numpy() - ref_sc).max() < 1e-13
    assert idx.cpu().numpy().tolist() == ref_idx.tolist()
    idx0, _ = ctx.leverage_select(lrp.tall_from_numpy(A), 0)
    assert idx0.numel() == 0
    with pytest.raises(lrp.LrpError) as e:
        ctx.leverage_select(lrp.tall_from_numpy(A), n + 1)
    assert e.value.code == lrp.LRP_ERR_BADARG


def test_scross_single_fiber_and_bad_indices(ctx):
    import torch
    from paper_2607_06021_b200 import lrp
    n = 511
    x = W.grid(n)
    u = np.exp(-3 * x)[:, None]; v = np.cos(2 * x)[:, None]
    I = np.array([7], dtype=np.int32); J = np.array([5], dtype=np.int32)
    Cm = u * v[J].T; Rt = v * u[I].T                                     # rank-1 G = u v^T
    out = ctx.scross(lrp.tall_from_numpy(Cm), lrp.tall_from_numpy(Rt), torch.from_numpy(I).cuda(), torch.from_numpy(J).cuda())
    U = lrp.tall_to_numpy(out["U"]); V = lrp.tall_to_numpy(out["V"]); S = out["S"].cpu().numpy()
    assert out["rank"] == 1
    assert np.abs((U * S) @ V.T - u @ v.T).max() < 1e-13 * np.abs(u @ v.T).max()
    dup = torch.tensor([3, 3], dtype=torch.int32, device="cuda")
    C2 = lrp.tall_from_numpy(np.hstack([Cm, Cm]))
    with pytest.raises(lrp.LrpError) as e:
        ctx.scross(C2, C2, dup, dup)
    assert e.value.code == lrp.LRP_ERR_BADARG


@pytest.mark.parametrize("n", [1023, 65535])
def test_rank_one_gaussian_rhs(ctx, n):
    """The paper's Poisson experiment uses a separable (rank-1) Gaussian forcing (eq. (7))."""
    import torch
    from paper_2607_06021_b200 import lrp
    x = W.grid(n)
    g1 = np.exp(-36 * (x - 0.55) ** 2); g2 = np.exp(-36 * (x - 0.45) ** 2)
    UF = (g1 / np.linalg.norm(g1))[:, None]; VF = (g2 / np.linalg.norm(g2))[:, None]
    SF = np.array([np.linalg.norm(g1) * np.linalg.norm(g2)])
    sg = np.random.default_rng(0).integers(0, n, 64).astype(np.int32)
    kw = dict(tol=1e-10, max_rank=48, oversample=8, max_sweeps=20, safeguard=sg)
    ref = O.cross_deim_solve(n, UF, SF, VF, **kw)
    res = ctx.cross_deim_solve(lrp.tall_from_numpy(UF), torch.from_numpy(SF).cuda(), lrp.tall_from_numpy(VF),
                               want_spectral=True, **kw)
    assert ref.converged and res["converged"]
    assert abs(res["rank"] - ref.rank) <= 1 and abs(res["sweeps"] - ref.sweeps) <= 1
    rows, cols = W.sample_pairs(n, 4096, seed=5)
    UW, VW, SW = lrp.tall_to_numpy(res["UW"]), lrp.tall_to_numpy(res["VW"]), res["SW"].cpu().numpy()
    a = np.einsum("tk,k,tk->t", UW[rows], SW, VW[cols]); b = O.lowrank_entries(ref.UW, ref.SW, ref.VW, rows, cols)
    # two converged free runs may stop one sweep apart: both are within the certified tolerance of the same solution
    assert np.abs(a - b).max() <= 20 * 1e-10 * np.abs(b).max()
    if n == 1023:                                                      # dense truth, eq. (4)
        Wd = O.dense_poisson(n, (UF * SF) @ VF.T)
        assert np.abs(a - Wd[rows, cols]).max() <= 20 * 1e-10 * np.abs(Wd).max()
