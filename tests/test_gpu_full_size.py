"""Full BASELINE sizes (C4: n = 2^20-1, C5: n = 2^22-1) in the launch configuration bench.py times.  The oracle cannot
run a whole solve at these sizes in test time, so the GPU result is checked on sampled outputs the oracle computes
one by one -- exact spectral entries G(i,j) = (Uh S Vh^T)(i,j)/(d_i+d_j) from the oracle's own DST of the factors --
and on properties that hold at any size (orthonormal factors, DST involution of the returned factors)."""
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


@pytest.mark.parametrize("name", ["C4", "C5"])
def test_full_size_solve_against_exact_spectral_entries(ctx, name):
    import torch
    from paper_2607_06021_b200 import lrp
    w = W.make(name, 0)
    n = w.n
    UF = lrp.tall_from_numpy(w.UF); VF = lrp.tall_from_numpy(w.VF); SF = torch.from_numpy(w.SF).cuda()
    res = ctx.cross_deim_solve(UF, SF, VF, tol=w.tol, max_rank=w.max_rank, oversample=w.oversample,
                               max_sweeps=w.max_sweeps, safeguard=w.safeguard, want_spectral=True)
    assert res["rank"] >= 1 and res["sweeps"] <= w.max_sweeps
    info = res["info"]
    # oracle side: spectral RHS factors by the oracle's own DST, exact entries at sampled (i, j)
    sc = O.orthonormal_scale(n)
    UhF = O.dst1_fft(w.UF, sc); VhF = O.dst1_fft(w.VF, sc)
    d = O.eigenvalues_d(n)
    # the RHS factors in sine space agree (forward DST at full size, every column)
    got = lrp.tall_to_numpy(ctx.dst1_batched(UF, scale=sc))
    assert np.abs(got - UhF).max() <= 1e-11 * np.abs(UhF).max()
    del got
    active = int(4 * max(max(t["I"].max(), t["J"].max()) for t in res["trace"])) + 64
    rows, cols = W.sample_pairs(n, 4096, seed=3, active=active)
    exact = O.G_entries(UhF, w.SF, VhF, d, rows, cols)
    r = res["rank"]
    Uh = res["Uhat"][:r]; Vh = res["Vhat"][:r]; Sh = res["Shat"][:r]
    approx = ctx.lowrank_entries(Uh, Sh, Vh, torch.from_numpy(rows).cuda(), torch.from_numpy(cols).cuda()).cpu().numpy()
    snorm = float(torch.linalg.vector_norm(res["Shat"]).item())
    # error of the truncated iterate, normalised by ||S||_2 (SURVEY.md 8(c) pin (iii)); the stop test certifies ~tol
    err = np.abs(approx - exact).max() / snorm
    bound = 50 * w.tol if res["converged"] else 50 * max(w.tol, max(info.rho, info.indicator) / snorm)
    assert err <= bound, (err, bound, res["converged"], info.rho / snorm, info.indicator / snorm)
    # properties at any size: orthonormal spectral and physical factors, Z Z = I on the returned factors
    # bar 1e-13, widened by the rounding of the check itself: a Gram entry is an n-term fp64 sum, eps sqrt(n) = 2.3e-13 at n = 2^20
    floor = max(1.0, np.sqrt(n / float(1 << 18)))
    for F, bar in ((res["Uhat"], 1e-13), (res["Vhat"], 1e-13), (res["UW"], 1e-12), (res["VW"], 1e-12)):
        G = (F @ F.T).cpu().numpy()
        assert np.abs(G - np.eye(G.shape[0])).max() <= bar * floor, np.abs(G - np.eye(G.shape[0])).max()
    back = ctx.dst1_batched(res["UW"], scale=sc)
    # two transforms in a row; the odd outputs are a prefix sum over N/2 terms, whose rounding error grows with N
    # (2-5e-11 of max|X| per transform at N = 2^22 on smooth columns)
    assert float((back - Uh).abs().max().item()) <= 2e-10 * float(Uh.abs().max().item())


def test_scross_rank_deficient_block_at_full_size(ctx):
    """Thin QR of fiber blocks whose columns are dependent to rounding (Alg. 4 lines 14-23, rely on
    it) at n = 2^20-1: exactly-rank-20 G sampled on 40 columns / 37 rows.  The factors must stay orthonormal to 1e-13
    (every panel is re-orthogonalised after its Householder factorization, decided and repeated on the device) and
    reproduce G (skeleton theorem)."""
    import torch
    from paper_2607_06021_b200 import lrp
    n, rank, k, l = (1 << 20) - 1, 20, 40, 37
    gen = torch.Generator(device="cuda"); gen.manual_seed(7)
    decay = torch.exp(-torch.arange(n, dtype=torch.float64, device="cuda") / (n / 8.0))
    A = torch.randn((rank, n), dtype=torch.float64, device="cuda", generator=gen) * decay      # tall tensors (cols, n)
    B = torch.randn((rank, n), dtype=torch.float64, device="cuda", generator=gen) * decay
    sig = 2.0 ** (-torch.arange(rank, dtype=torch.float64, device="cuda"))
    rng = np.random.default_rng(11)
    I = torch.from_numpy(rng.choice(n // 8, l, replace=False).astype(np.int32)).cuda()
    J = torch.from_numpy(rng.choice(n // 8, k, replace=False).astype(np.int32)).cuda()
    Cm = (B[:, J.long()].T * sig) @ A                      # (k, n): column c = G(:, J[c])
    Rt = (A[:, I.long()].T * sig) @ B                      # (l, n): column c = G(I[c], :)^T
    out = ctx.scross(Cm.contiguous(), Rt.contiguous(), I, J)
    U, V, S = out["U"], out["V"], out["S"]
    assert out["rank"] >= rank
    eye = torch.eye(U.shape[0], dtype=torch.float64, device="cuda")
    # 1e-13 x 2: the check's own n-term fp64 Gram sums round at eps sqrt(n) = 2.3e-13 for n = 2^20
    assert float((U @ U.T - eye).abs().max().item()) <= 2e-13 and float((V @ V.T - eye).abs().max().item()) <= 2e-13
    rows = torch.from_numpy(rng.integers(0, n, 4096)).cuda(); cols = torch.from_numpy(rng.integers(0, n // 4, 4096)).cuda()
    got = ctx.lowrank_entries(U, S, V, rows, cols)
    truth = ((A[:, rows] * sig[:, None]) * B[:, cols]).sum(0)
    assert float((got - truth).abs().max().item()) <= 1e-10 * float(Cm.abs().max().item())
    rC = out["rC"].cpu().numpy()
    assert (rC[rank:] < 1e-12 * rC.max()).all()
