"""GPU parity of the per-step C-ABI calls against the CPU oracle (same seeded inputs, element by element)."""
import math

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


def _rel(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


# ------------------------------------------------------------------------------------------------ DST-I
# tolerance: FFT rounding eps*log2(N) plus the sqrt(N) growth of the odd-output prefix sum
@pytest.mark.parametrize("n", [1, 3, 7, 31, 63, 127, 255, 511, 1023, 2047, 4095, 8191, 16383])
def test_dst1_one_pass_regime(ctx, n):
    from paper_2607_06021_b200 import lrp
    x = W.dst_batch(n, 5, seed=n)
    ref = O.dst1(x, 1.0) if n <= 4095 else O.dst1_fft(x, 1.0)
    got = lrp.tall_to_numpy(ctx.dst1_batched(lrp.tall_from_numpy(x)))
    assert _rel(got, ref) < 1e-12
    # orthonormal scaling, in place, and the involution Z Z = I
    t = lrp.tall_from_numpy(x)
    sc = O.orthonormal_scale(n)
    ctx.dst1_batched(t, out=t, scale=sc)
    assert _rel(lrp.tall_to_numpy(t), sc * ref) < 1e-12
    ctx.dst1_batched(t, out=t, scale=sc)
    assert _rel(lrp.tall_to_numpy(t), x) < 1e-12


@pytest.mark.parametrize("n", [32767, 65535, (1 << 18) - 1])
def test_dst1_four_step_regime(ctx, n):
    from paper_2607_06021_b200 import lrp
    x = W.dst_batch(n, 3, seed=7)
    x[:, 1] = np.exp(-((W.grid(n) - 0.37) ** 2) / (2 * 0.01 ** 2))      # a smooth column like the bump factors
    ref = O.dst1_fft(x, 1.0)
    got = lrp.tall_to_numpy(ctx.dst1_batched(lrp.tall_from_numpy(x)))
    for c in range(3):
        assert _rel(got[:, c], ref[:, c]) < 1e-12          # exact per-chunk anchors: no growth with N
    t = lrp.tall_from_numpy(x)
    ctx.dst1_batched(t, out=t, scale=1.0)
    ctx.dst1_batched(t, out=t, scale=2.0 / (n + 1))                       # twice = (n+1)/2 I
    assert _rel(lrp.tall_to_numpy(t), x) < 1e-12


@pytest.mark.parametrize("p", [17, 19, 20, 21, 22, 23, 24, 25])
def test_dst1_full_size_sampled(ctx, p):
    """BASELINE sizes n = 2^20-1, 2^22-1, the largest sizes the call accepts (2^24-1, 2^25-1) and the sizes in between
    whose four-step split is not met elsewhere (every instantiation of the persistent kernel from L = 2^16 = 256 x 256 to
    2^24 = 4096 x 4096 is run by this test or by test_dst1_four_step_regime): sampled outputs against the O(n) definition
    sum per entry."""
    import torch
    from paper_2607_06021_b200 import lrp
    n = (1 << p) - 1
    batch = 3 if p <= 22 else (2 if p == 24 else 1)
    x = W.dst_batch(n, batch, seed=p)
    t = lrp.tall_from_numpy(x)
    out = ctx.dst1_batched(t)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    rng = np.random.default_rng(p)
    ks = np.concatenate([[1, 2, 3, n - 1, n, (n + 1) // 2, (n + 1) // 2 + 1], rng.integers(1, n + 1, 25 if p <= 22 else 3)])
    for c in range(batch):
        ref = O.dst1_entries(x[:, c], ks)
        scale = np.abs(got[c]).max()
        assert np.abs(got[c, ks - 1] - ref).max() < 1e-12 * scale
    # Parseval with the orthonormal scaling (holds at any size)
    y = ctx.dst1_batched(t, scale=O.orthonormal_scale(n))
    nx = torch.linalg.vector_norm(t, dim=1).cpu().numpy()
    ny = torch.linalg.vector_norm(y, dim=1).cpu().numpy()
    assert np.abs(nx - ny).max() < 1e-12 * nx.max()


def test_dst1_leading_dimension_and_errors(ctx):
    import torch
    from paper_2607_06021_b200 import lrp
    n, b = 1023, 4
    x = W.dst_batch(n, b, seed=3)
    big = torch.zeros((b, n + 9), dtype=torch.float64, device="cuda")
    big[:, :n] = lrp.tall_from_numpy(x)
    view = big[:, :n]
    out = ctx.dst1_batched(view)
    assert _rel(lrp.tall_to_numpy(out), O.dst1(x)) < 1e-12
    # n + 1 need not be a power of two (Bluestein, tests/test_gpu_general_n.py); beyond 2^23 it is refused
    import ctypes as C
    rc = ctx.lib.lrp_dst1_batched(ctx.h, (1 << 23) + 1, 1, C.c_void_p(big.data_ptr()), (1 << 23) + 1, C.c_void_p(big.data_ptr()),
                                  (1 << 23) + 1, 1.0)
    assert rc == lrp.LRP_ERR_UNSUPPORTED_N
    empty = torch.zeros((0, n), dtype=torch.float64, device="cuda")
    assert ctx.dst1_batched(empty).shape == (0, n)


# ------------------------------------------------------------------------------------------------ fibers
@pytest.mark.parametrize("n,r,nI,nJ", [(255, 4, 12, 13), (4095, 3, 19, 11), (4095, 37, 70, 33), (65535, 8, 40, 41)])
def test_sample_fibers(ctx, n, r, nI, nJ):
    import torch
    from paper_2607_06021_b200 import lrp
    rng = np.random.default_rng(n + r)
    Uh = rng.standard_normal((n, r)); Vh = rng.standard_normal((n, r)); S = np.abs(rng.standard_normal(r)) + 0.1
    I = rng.choice(n, nI, replace=False).astype(np.int32); J = rng.choice(n, nJ, replace=False).astype(np.int32)
    I[0], J[0] = 0, n - 1
    d = O.eigenvalues_d(n)
    Cref, Rref = O.sample_fibers(Uh, S, Vh, d, I, J)
    Cg, Rg = ctx.sample_fibers(lrp.tall_from_numpy(Uh), torch.from_numpy(S).cuda(), lrp.tall_from_numpy(Vh),
                               torch.from_numpy(I).cuda(), torch.from_numpy(J).cuda())
    # entrywise: r-term dot product + one divide; error relative to the sum of magnitudes (cancellation-free bound)
    boundC = ((np.abs(Uh) * S) @ np.abs(Vh[J]).T) / (d[:, None] + d[J][None, :])
    boundR = ((np.abs(Vh) * S) @ np.abs(Uh[I]).T) / (d[:, None] + d[I][None, :])
    assert (np.abs(lrp.tall_to_numpy(Cg) - Cref) <= 1e-14 * r * boundC + 1e-300).all()
    assert (np.abs(lrp.tall_to_numpy(Rg) - Rref) <= 1e-14 * r * boundR + 1e-300).all()
    # one side only
    Cg2, none = ctx.sample_fibers(lrp.tall_from_numpy(Uh), torch.from_numpy(S).cuda(), lrp.tall_from_numpy(Vh),
                                  None, torch.from_numpy(J).cuda())
    assert none is None and torch.equal(Cg2, Cg)


# ------------------------------------------------------------------------------------------------ leverage
@pytest.mark.parametrize("n,k", [(255, 4), (4095, 7), (4095, 40), (65535, 33)])
def test_leverage_select(ctx, n, k):
    from paper_2607_06021_b200 import lrp
    rng = np.random.default_rng(k * 1000 + n)
    x = W.grid(n)
    # smooth decaying columns (like spectral factors): leverage concentrated on few rows, well separated
    A = np.stack([np.exp(-(c + 1) * 3.0 * x) * np.cos((c + 1) * 2.0 * x + c) for c in range(k)], axis=1)
    A = A + 1e-3 * rng.standard_normal((n, k)) * np.exp(-5 * x)[:, None]
    num = min(k + 8, n)
    idx_ref, sc_ref = O.leverage_select(A, num)
    idx, sc = ctx.leverage_select(lrp.tall_from_numpy(A), num)
    sc = sc.cpu().numpy(); idx = idx.cpu().numpy()
    assert abs(sc.sum() - k) < 1e-10 and sc.min() >= -1e-15 and sc.max() <= 1 + 1e-12      # sum of leverage = k
    assert np.abs(sc - sc_ref).max() < 1e-11
    # selected sets equal as ordered lists wherever the deciding gaps exceed 1e-12 (north_star)
    s_sorted = np.sort(sc_ref)[::-1]
    gaps = np.abs(np.diff(s_sorted[:num + 1]))
    if gaps.min() > 1e-12:
        assert idx.tolist() == idx_ref.tolist()
    else:
        assert set(idx.tolist()) == set(idx_ref.tolist()) or np.abs(np.sort(sc[idx]) - np.sort(sc_ref[idx_ref])).max() < 1e-11
    # orthonormal shortcut: scores are the plain squared row norms
    Q, _ = np.linalg.qr(A)
    idx2, sc2 = ctx.leverage_select(lrp.tall_from_numpy(Q), num, assume_orthonormal=True)
    assert np.abs(sc2.cpu().numpy() - (Q * Q).sum(1)).max() < 1e-13


def test_leverage_ties_are_broken_by_index(ctx):
    import torch
    from paper_2607_06021_b200 import lrp
    n = 4095
    A = np.zeros((n, 2)); A[[5, 77, 900, 4000], 0] = 0.5; A[[6, 78, 901, 4001], 1] = 0.5
    idx, sc = ctx.leverage_select(lrp.tall_from_numpy(A), 6, assume_orthonormal=True)
    assert idx.cpu().numpy().tolist() == [5, 6, 77, 78, 900, 901]


# ------------------------------------------------------------------------------------------------ scross
def _recon(U, S, V, rows, cols):
    return np.einsum("tk,k,tk->t", U[rows], S, V[cols])


def _kahan(m, c):
    sn = np.sqrt(1.0 - c * c)
    return (sn ** np.arange(m))[:, None] * (np.eye(m) - c * np.triu(np.ones((m, m)), 1))


@pytest.mark.parametrize("m,c", [(64, 0.6), (100, 0.45)])
def test_scross_numerically_singular_selected_rows_with_a_harmless_r_diagonal(ctx, m, c):
    """Q(I,:) = a scaled Kahan matrix: numerically singular (sigma_min / sigma_max ~ 1e-20, below the 1e-13 cut of reading
    Q4) while the diagonal of its unpivoted R spans only 1e-6.  The Householder least-squares shortcut of the core must not
    be taken on the strength of that diagonal: its condition test is ||R||_F ||R^-1||_F, and the SVD pseudo-inverse (which
    drops the singular direction, like the oracle) takes over.  m = 64: the shortcut's size range; m = 100: beyond it."""
    import torch
    from paper_2607_06021_b200 import lrp
    n = 4095
    rng = np.random.default_rng(m)
    X0 = _kahan(m, c); X0 *= 0.5 / np.linalg.norm(X0, 2)
    sv = np.linalg.svd(X0, compute_uv=False)
    d = np.abs(np.diag(np.linalg.qr(X0)[1]))
    assert sv[-1] < 1e-15 * sv[0] and sv[-2] > 1e-8 * sv[0] and d.min() > 1e-7 * d.max()      # the construction holds
    w, V = np.linalg.eigh(np.eye(m) - X0.T @ X0)
    comp = np.linalg.qr(rng.standard_normal((n - m, m)))[0] @ ((V * np.sqrt(w)) @ V.T)       # completes X0 to orthonormal columns
    I = np.sort(rng.choice(n, m, replace=False)).astype(np.int32)
    J = np.sort(rng.choice(n, m, replace=False)).astype(np.int32)
    Cm = np.empty((n, m)); rest = np.ones(n, bool); rest[I] = False
    Cm[I] = X0; Cm[rest] = comp
    Rt = rng.standard_normal((n, m)) * np.exp(-np.arange(n) / (n / 6))[:, None]
    ref = O.scross(Cm, Rt, I, J)
    out = ctx.scross(lrp.tall_from_numpy(Cm), lrp.tall_from_numpy(Rt), torch.from_numpy(I).cuda(), torch.from_numpy(J).cuda())
    U = lrp.tall_to_numpy(out["U"]); Vg = lrp.tall_to_numpy(out["V"]); S = out["S"].cpu().numpy()
    assert out["rank"] == ref.rank
    tol = 1e-9                                          # measured 1e-11; eps * sigma_1 / sigma_kept,min = 1e-9 .. 1e-10
    errS = np.abs(S - ref.S).max() / ref.S[0]
    rows = rng.integers(0, n, 4096); cols = rng.integers(0, n, 4096)
    a = _recon(U, S, Vg, rows, cols); b = _recon(ref.U, ref.S, ref.V, rows, cols)
    errW = np.abs(a - b).max() / np.abs(b).max()
    print(f"Kahan m={m}: rank {out['rank']}, S {errS:.2e}, entries {errW:.2e} (tol {tol:.1e})")
    assert errS <= tol and errW <= tol


@pytest.mark.parametrize("n,rank,k,l", [(255, 4, 12, 13), (4095, 9, 20, 17), (4095, 30, 45, 45), (16383, 12, 33, 40)])
def test_scross_exact_low_rank(ctx, n, rank, k, l):
    """Skeleton theorem pin carried to the GPU: rank(G) <= #I,#J and rank G(I,J) = rank  =>  U S V^T = G."""
    import torch
    from paper_2607_06021_b200 import lrp
    rng = np.random.default_rng(n + rank)
    A = rng.standard_normal((n, rank)) * np.exp(-np.arange(n) / (n / 8))[:, None]
    B = rng.standard_normal((n, rank)) * np.exp(-np.arange(n) / (n / 8))[:, None]
    sig = 2.0 ** (-np.arange(rank))
    G = lambda rows, cols: np.einsum("tk,k,tk->t", A[rows], sig, B[cols])
    I = rng.choice(n // 8, l, replace=False).astype(np.int32); J = rng.choice(n // 8, k, replace=False).astype(np.int32)
    Cm = (A * sig) @ B[J].T; Rt = (B * sig) @ A[I].T
    ref = O.scross(Cm, Rt, I, J)
    out = ctx.scross(lrp.tall_from_numpy(Cm), lrp.tall_from_numpy(Rt), torch.from_numpy(I).cuda(), torch.from_numpy(J).cuda())
    U = lrp.tall_to_numpy(out["U"]); V = lrp.tall_to_numpy(out["V"]); S = out["S"].cpu().numpy()
    rows = rng.integers(0, n, 4096); cols = rng.integers(0, n, 4096)
    truth = G(rows, cols)
    scale = np.abs(Cm).max()
    assert np.abs(_recon(U, S, V, rows, cols) - truth).max() < 1e-10 * scale
    assert np.abs(_recon(U, S, V, rows, cols) - _recon(ref.U, ref.S, ref.V, rows, cols)).max() < 1e-10 * scale
    Sf = out["S_full"].cpu().numpy()
    assert np.abs(Sf[:rank] - ref.S_full[:rank]).max() < 1e-10 * ref.S_full[0]
    # |diag R| of the unpivoted QR is unique for the numerically independent columns
    rC = out["rC"].cpu().numpy(); rR = out["rR"].cpu().numpy()
    assert np.abs(rC[:rank] - ref.rC[:rank]).max() < 1e-10 * ref.rC.max()
    assert np.abs(rR[:rank] - ref.rR[:rank]).max() < 1e-10 * ref.rR.max()
    assert (rC[rank:] < 1e-12 * rC.max()).all() and (rR[rank:] < 1e-12 * rR.max()).all()
    # orthonormal factors
    assert np.abs(U.T @ U - np.eye(U.shape[1])).max() <= 1e-13 and np.abs(V.T @ V - np.eye(V.shape[1])).max() <= 1e-13
