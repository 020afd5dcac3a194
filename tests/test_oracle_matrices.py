"""Pins for the generic (function-handle) Cross-DEIM of the oracle on the paper's test matrices, eq. (6),
PAPER.md:264-267: entries by hand and against an independent library construction, fibers against slices of the
dense matrix, and the converged approximation against the dense SVD (Hilbert to 1e-9; 309: K to 1e-6)."""
import numpy as np
import pytest

from oracle import lrp_oracle as O
from paper_2607_06021_b200 import workloads as W


def _dense(kind, n):
    i = np.arange(n)
    return O.hilbert_entries(i[:, None], i[None, :]) if kind == "hilbert" else O.kmatrix_entries(n, i[:, None], i[None, :])


def test_hilbert_entries_are_the_hilbert_matrix():
    from scipy.linalg import hilbert
    n = 64
    H = _dense("hilbert", n)
    assert np.array_equal(H, hilbert(n))                     # 1/(i + j + 1), 0-based: the classical Hilbert matrix
    assert H[0, 0] == 1.0 and H[2, 3] == 1.0 / 6.0 and H[n - 1, n - 1] == 1.0 / (2 * n - 1)


def test_kmatrix_entries_by_hand():
    # n = 5: x = y = [-1, -0.5, 0, 0.5, 1]
    K = _dense("kmatrix", 5)
    assert K[0, 0] == 1.0 and K[4, 4] == 1.0                  # (|-2|/2)^5, (|2|/2)^5
    assert K[3, 4] == 0.75 ** 5 and K[4, 3] == 0.75 ** 5      # (|0.5 + 1|/2)^5
    assert K[1, 2] == 0.25 ** 5                                # (|-0.5 + 0|/2)^5
    for i in range(5):
        assert K[i, 4 - i] == 0.0                              # the kink x + y = 0 (C^4 only)
    n = 33
    K = _dense("kmatrix", n)
    assert np.array_equal(K, K.T)
    # closed form on the grid: ((i + j) / (n - 1) - 1)^5 in absolute value
    i = np.arange(n)
    ref = np.abs((i[:, None] + i[None, :]) / (n - 1.0) - 1.0) ** 5
    assert np.abs(K - ref).max() < 1e-15


@pytest.mark.parametrize("kind", ["hilbert", "kmatrix"])
def test_fibers_are_slices_of_the_dense_matrix(kind):
    n = 100
    G = _dense(kind, n) + 0.0
    if kind == "kmatrix":
        G = G.copy()
    I = np.array([3, 99, 0, 41]); J = np.array([7, 0, 98])
    C, Rt = O.matrix_fibers(kind, n)(I, J)
    assert C.shape == (n, 3) and Rt.shape == (n, 4)
    assert np.array_equal(C, G[:, J]) and np.array_equal(Rt, G[I, :].T)


@pytest.mark.parametrize("kind,n,tol,seed", [("hilbert", 512, 1e-9, 0), ("hilbert", 1024, 1e-9, 0), ("kmatrix", 512, 1e-6, 0)])
def test_cross_deim_on_test_matrices_against_dense_svd(kind, n, tol, seed):
    U0, V0, sg = W.matrix_initial_guess(n, 4, seed)
    r = O.cross_deim(n, O.matrix_fibers(kind, n), U0, V0, tol=tol, max_rank=64, oversample=8, max_sweeps=12, safeguard=sg)
    assert r.converged and r.sweeps <= 8                       # LS needs a few more sweeps than (Q)DEIM's 6-7
    G = _dense(kind, n)
    A = (r.U[:, :r.rank] * r.S[:r.rank]) @ r.V[:, :r.rank].T
    sv = np.linalg.svd(G, compute_uv=False)
    nrm = np.linalg.norm(G)
    best = np.sqrt((sv[r.rank:] ** 2).sum())
    err = np.linalg.norm(A - G)
    if kind == "hilbert":                                      # fast decay: the cross approximation is quasi-optimal
        assert err <= 2.0 * best + 1e-12 * nrm and err <= 5 * tol * nrm
        assert abs(r.rank - O.final_rank(sv, tol, 64)) <= 1
        assert np.abs(r.S[:r.rank] - sv[:r.rank]).max() <= 10 * tol * sv[0]
    else:                                                      # slow decay: error within the DEIM-type factor of the best one
        assert err <= 10.0 * best and err <= 20 * tol * nrm
        assert np.abs(r.S[:r.rank] - sv[:r.rank]).max() <= 100 * tol * sv[0]
    # orthonormal factors, descending singular values
    assert np.abs(r.U.T @ r.U - np.eye(r.U.shape[1])).max() < 1e-12 and (np.diff(r.S) <= 0).all()
    # the iterate interpolates G on the selected cross (exact up to the discarded pinv/rank cuts)
    t = r.trace[-1]
    It, Jt = t.I.astype(np.int64), t.J.astype(np.int64)
    full = (r.U * r.S) @ r.V.T
    assert np.abs(full[np.ix_(It, Jt)] - G[np.ix_(It, Jt)]).max() <= 50 * tol * np.abs(G).max()
