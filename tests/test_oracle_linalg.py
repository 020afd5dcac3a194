"""Pins for the oracle's Householder QR, Jacobi SVD / pinv, leverage scores + top-k, scross and the
stopping-test pieces.  LAPACK (numpy.linalg) is used here only as an independent check."""
import math

import numpy as np
import pytest

from oracle import lrp_oracle as O


@pytest.mark.parametrize("shape", [(40, 7), (9, 9), (200, 33), (5, 8)])
def test_householder_qr(shape):
    rng = np.random.default_rng(sum(shape))
    A = rng.standard_normal(shape)
    Q, R = O.householder_qr(A)
    p = min(shape)
    assert Q.shape == (shape[0], p) and R.shape == (p, shape[1])
    assert np.abs(Q.T @ Q - np.eye(p)).max() < 1e-14
    assert np.abs(Q @ R - A).max() < 1e-14 * np.abs(A).max() * 10
    assert np.abs(np.tril(R, -1)).max() == 0.0
    Qn, Rn = np.linalg.qr(A)                       # |diag R| is unique for full-rank A
    assert np.abs(np.abs(np.diag(R)) - np.abs(np.diag(Rn))).max() < 1e-13
    sgn = np.sign(np.diag(R)) * np.sign(np.diag(Rn))
    assert np.abs(R - sgn[:, None] * Rn).max() < 1e-13


def test_householder_qr_rank_deficient_keeps_q_orthonormal():
    rng = np.random.default_rng(2)
    B = rng.standard_normal((120, 4))
    A = np.hstack([B, B @ rng.standard_normal((4, 3)), rng.standard_normal((120, 2))])
    Q, R = O.householder_qr(A)
    assert np.abs(Q.T @ Q - np.eye(9)).max() < 1e-14
    assert np.abs(Q @ R - A).max() < 1e-13
    dg = np.abs(np.diag(R))
    assert (dg[4:7] < 1e-13 * dg.max()).all() and (dg[:4] > 1e-3).all() and (dg[7:] > 1e-3).all()
    Z = np.zeros((10, 3))
    Q0, R0 = O.householder_qr(Z)                   # all-zero input must not produce NaN
    assert np.isfinite(Q0).all() and np.abs(R0).max() == 0.0


@pytest.mark.parametrize("shape", [(30, 6), (6, 30), (12, 12), (1, 5), (7, 1)])
def test_jacobi_svd(shape):
    rng = np.random.default_rng(shape[0] * 31 + shape[1])
    M = rng.standard_normal(shape) * np.logspace(0, -6, shape[1])[None, :]
    U, s, V = O.jacobi_svd(M)
    p = min(shape)
    assert U.shape == (shape[0], p) and V.shape == (shape[1], p) and s.shape == (p,)
    assert (np.diff(s) <= 0).all() and (s >= 0).all()
    assert np.abs(U.T @ U - np.eye(p)).max() < 1e-13
    assert np.abs(V.T @ V - np.eye(p)).max() < 1e-13
    assert np.abs((U * s) @ V.T - M).max() < 1e-14 * max(1.0, np.abs(M).max()) * 10
    sn = np.linalg.svd(M, compute_uv=False)
    assert np.abs(s - sn).max() < 1e-14 * sn[0] * 10
    # against the eigenvalues of M^T M on the well-conditioned part
    ev = np.sort(np.linalg.eigvalsh(M.T @ M if shape[0] >= shape[1] else M @ M.T))[::-1]
    assert abs(math.sqrt(ev[0]) - s[0]) < 1e-13 * s[0]


def test_jacobi_svd_special_cases():
    D = np.diag([3.0, 0.5, 7.0])
    U, s, V = O.jacobi_svd(D)
    assert np.allclose(s, [7.0, 3.0, 0.5], atol=0, rtol=1e-15)
    M = np.array([[3.0, 0.0], [4.0, 5.0]])        # textbook 2x2: singular values sqrt(45), sqrt(5)
    _, s, _ = O.jacobi_svd(M)
    assert np.allclose(s, [math.sqrt(45.0), math.sqrt(5.0)], rtol=1e-15)
    R1 = np.outer([1.0, 2.0, 2.0], [3.0, 4.0])     # rank one: sigma = 3 * 5
    U, s, V = O.jacobi_svd(R1)
    assert abs(s[0] - 15.0) < 1e-14 and s[1] < 1e-15
    assert np.isfinite(U).all() and np.isfinite(V).all()


def test_pinv_moore_penrose():
    rng = np.random.default_rng(11)
    A = rng.standard_normal((25, 8))
    P = O.pinv_svd(A)
    assert np.abs(P - np.linalg.pinv(A)).max() < 1e-13
    for lhs, rhs in ((A @ P @ A, A), (P @ A @ P, P), ((A @ P).T, A @ P), ((P @ A).T, P @ A)):
        assert np.abs(lhs - rhs).max() < 1e-13
    # rank deficient: cut at 1e-13 * sigma_max
    B = np.hstack([A, A[:, :2] @ rng.standard_normal((2, 2))])
    P = O.pinv_svd(B)
    assert np.abs(P - np.linalg.pinv(B, rcond=1e-13)).max() < 1e-11
    assert np.abs(B @ P @ B - B).max() < 1e-12
    assert abs(O.sigma_min(A) - np.linalg.svd(A, compute_uv=False)[-1]) < 1e-14


def test_leverage_scores_and_topk():
    rng = np.random.default_rng(4)
    n, k = 300, 6
    A = rng.standard_normal((n, k)) * np.logspace(0, 2, k)[None, :]
    sc = O.leverage_scores(A)
    assert abs(sc.sum() - k) < 1e-12                       # sums to k (north_star)
    assert (sc >= 0).all() and (sc <= 1 + 1e-14).all()
    H = A @ np.linalg.solve(A.T @ A, A.T)                  # diag of the orthogonal projector
    assert np.abs(sc - np.diag(H)).max() < 1e-10
    B = rng.standard_normal((k, k)) + 3 * np.eye(k)        # invariance under right-multiplication
    assert np.abs(O.leverage_scores(A @ B) - sc).max() < 1e-11
    # unit-vector columns => indicator (C1 gives exactly this)
    E = np.zeros((50, 3))
    E[[4, 17, 30], [0, 1, 2]] = [2.0, -1.0, 0.5]
    assert np.array_equal(O.leverage_scores(E), (np.abs(E).sum(1) > 0).astype(float))
    # dependent column is excluded, the score sum drops to the rank
    A2 = np.hstack([A, A[:, :1] * 2.0])
    assert abs(O.leverage_scores(A2).sum() - k) < 1e-10
    # orthonormal input: skipping the QR gives the same scores
    Q, _ = O.householder_qr(A)
    assert np.abs(O.leverage_scores(Q, assume_orthonormal=True) - sc).max() < 1e-13
    # top-k = full sort with (score desc, index asc)
    s2 = np.array([0.5, 0.9, 0.5, 0.1, 0.9, 0.0])
    assert O.top_select(s2, 4).tolist() == [1, 4, 0, 2]
    assert O.top_select(s2, 10).tolist() == [1, 4, 0, 2, 3, 5]
    idx, _ = O.leverage_select(A, 9)
    assert idx.tolist() == sorted(range(n), key=lambda i: (-sc[i], i))[:9]


def _random_lowrank(rng, m, n, r):
    return rng.standard_normal((m, r)) @ np.diag(np.logspace(0, -3, r)) @ rng.standard_normal((r, n))


@pytest.mark.parametrize("kl", [(6, 9), (9, 6), (5, 5)])
def test_scross_is_exact_on_exactly_low_rank_matrices(kl):
    # skeleton theorem (eq. (1), refs [12,13]): rank(G) = r <= min(k,l) and
    # rank G(I,J) = r  =>  U S V^T = G exactly.
    k, l = kl
    rng = np.random.default_rng(10 * k + l)
    n, r = 80, 4
    G = _random_lowrank(rng, n, n, r)
    I = rng.choice(n, l, replace=False)
    J = rng.choice(n, k, replace=False)
    res = O.scross(G[:, J], G[I, :].T, I, J)
    assert res.rank == r
    assert np.abs((res.U * res.S) @ res.V.T - G).max() < 1e-10 * np.abs(G).max()
    assert np.abs(res.S - np.linalg.svd(G, compute_uv=False)[:r]).max() < 1e-10 * res.S[0]
    assert np.abs(res.U.T @ res.U - np.eye(r)).max() < 1e-12
    assert res.rC.shape == (k,) and res.rR.shape == (l,)
    assert res.smin_full < 1e-12 * res.S[0]
    # r_C is the distance of column c of C from the span of the previous ones
    Cm = G[:, J]
    for c in (0, 2, k - 1):
        if c == 0:
            dist = np.linalg.norm(Cm[:, 0])
        else:
            coef, *_ = np.linalg.lstsq(Cm[:, :c], Cm[:, c], rcond=None)
            dist = np.linalg.norm(Cm[:, c] - Cm[:, :c] @ coef)
        assert abs(res.rC[c] - dist) < 1e-10 * np.abs(G).max() * 10


def test_scross_on_hilbert_matrix_decays_like_singular_values():
    # H(i,j) = 1/(1+i+j), eq. (6)
    n = 256
    i = np.arange(n)
    H = 1.0 / (1.0 + i[:, None] + i[None, :])
    sv = np.linalg.svd(H, compute_uv=False)
    errs = []
    for k in (4, 8, 12):
        idx = np.unique(np.round(np.geomspace(1, n, k + 2)).astype(int) - 1)[:k]
        res = O.scross(H[:, idx], H[idx, :].T, idx, idx)
        err = np.linalg.norm((res.U * res.S) @ res.V.T - H, 2)
        errs.append(err)
        assert err < 1e4 * sv[len(idx)]
    assert errs[2] < errs[1] < errs[0]


def test_rho_eta_indicator_final_rank():
    rng = np.random.default_rng(8)
    n = 60
    Uk, _ = np.linalg.qr(rng.standard_normal((n, 5)))
    Vk, _ = np.linalg.qr(rng.standard_normal((n, 5)))
    Up, _ = np.linalg.qr(Uk[:, :4] + 1e-6 * rng.standard_normal((n, 4)))
    Vp, _ = np.linalg.qr(Vk[:, :4] + 1e-6 * rng.standard_normal((n, 4)))
    Sk = np.array([5.0, 3.0, 1.0, 0.1, 1e-7])
    Sp = Sk[:4] * (1 + 1e-7)
    dense = np.linalg.norm((Uk * Sk) @ Vk.T - (Up * Sp) @ Vp.T, "fro")
    assert abs(O.rho_factored(Uk, Sk, Vk, Up, Sp, Vp) - dense) < 1e-12
    # a difference far below sqrt(eps) is still resolved (no Gram expansion)
    Up2, Vp2 = Uk.copy(), Vk.copy()
    Sp2 = Sk + 1e-12
    assert abs(O.rho_factored(Uk, Sk, Vk, Up2, Sp2, Vp2) - math.sqrt(5) * 1e-12) < 1e-14
    assert abs(O.rho_factored(Uk, Sk, Vk, None, None, None) - np.linalg.norm(Sk)) < 1e-15
    idx = np.array([1, 7, 20, 33, 41, 50])
    assert abs(O.eta_of(Uk, idx) - 1.0 / np.linalg.svd(Uk[idx], compute_uv=False)[-1]) < 1e-9
    assert O.eta_of(Uk, np.array([], dtype=int)) == math.inf
    assert O.indicator(math.inf, 2.0, 0.0) == 0.0
    assert O.indicator(2.0, 3.0, 0.5) == min(2 * 4, 3 * 3) * 0.5
    S = np.array([1.0, 1e-3, 1e-6, 1e-9])
    assert O.final_rank(S, 1e-5, 10) == 2           # tail {1e-6, 1e-9} < 1e-5 * ||S||
    assert O.final_rank(S, 1e-5, 1) == 1            # capped by r_max
    assert O.final_rank(S, 1e-12, 10) == 4
    assert O.final_rank(S, 10.0, 10) == 1           # never below 1
    assert O.final_rank(S, 2e-6, 10, tol_mode=1) == 2
