"""Pins for the oracle's DEIM / QDEIM index selection (Alg. 2): the pivots of LAPACK's pivoted
factorizations (scipy), the interpolation property the methods exist for, unit-vector inputs, and the paper's
qualitative statement about the Hilbert matrix."""
import numpy as np
import pytest
import scipy.linalg as sl

from oracle import lrp_oracle as O
from paper_2607_06021_b200 import workloads as W


def _basis(n, r, seed):
    rng = np.random.default_rng(seed)
    Q, _ = np.linalg.qr(rng.standard_normal((n, r)) * np.exp(-np.arange(n) / (n / 5.0))[:, None])
    return Q


@pytest.mark.parametrize("n,r,seed", [(50, 3, 0), (200, 7, 1), (5000, 20, 2), (4095, 33, 3)])
def test_pivots_are_lapacks(n, r, seed):
    U = _basis(n, r, seed)
    p_qr = sl.qr(U.T, pivoting=True, mode="r")[1][:r]                     # dgeqp3: column-pivoted QR of U^T
    assert O.qdeim_select(U).tolist() == p_qr.tolist()
    P, _, _ = sl.lu(U)                                                    # dgetrf: U = P L U', pivot rows in order
    assert O.deim_select(U).tolist() == np.argmax(P, axis=0)[:r].tolist()


def test_unit_vector_columns_select_their_rows():
    n = 300
    U = np.zeros((n, 4)); rows = [17, 3, 250, 99]
    U[rows, np.arange(4)] = [1.0, -1.0, 1.0, 1.0]
    assert O.qdeim_select(U).tolist() == [3, 17, 99, 250]                 # equal norms: lowest index first
    assert O.deim_select(U).tolist() == rows                              # column by column


@pytest.mark.parametrize("sel", ["qdeim", "deim"])
def test_interpolation_property(sel):
    """The selected rows make U(I,:) invertible with a moderate inverse: the DEIM error constant ||U(I,:)^-1||_2
    (refs [8], [11] of the paper), far below the trivial bound and far better than random rows."""
    n, r = 3000, 12
    U = _basis(n, r, 5)
    I = O.qdeim_select(U) if sel == "qdeim" else O.deim_select(U)
    assert len(set(I.tolist())) == r
    c_sel = 1.0 / np.linalg.svd(U[I], compute_uv=False)[-1]
    rng = np.random.default_rng(0)
    c_rand = np.median([1.0 / np.linalg.svd(U[rng.choice(n, r, replace=False)], compute_uv=False)[-1] for _ in range(20)])
    assert c_sel < 50 and c_sel < 0.1 * c_rand


@pytest.mark.parametrize("sel", ["qdeim", "deim"])
def test_hilbert_converges_in_six_or_seven_sweeps(sel):
    """'fast convergence to the tolerance of 1e-9 in 6-7 Cross-DEIM iterations for the DEIM-variations'."""
    n = 1024
    U0, V0, sg = W.matrix_initial_guess(n, 4, 1)
    r = O.cross_deim(n, O.matrix_fibers("hilbert", n), U0, V0, tol=1e-9, max_rank=64, oversample=8, max_sweeps=12, safeguard=sg,
                     selection=sel)
    assert r.converged and r.sweeps <= 7
    i = np.arange(n)
    G = O.hilbert_entries(i[:, None], i[None, :])
    A = (r.U[:, :r.rank] * r.S[:r.rank]) @ r.V[:, :r.rank].T
    assert np.linalg.norm(A - G) <= 5e-9 * np.linalg.norm(G)
    # the index sets grow by the (Q)DEIM points of the previous iterate: |I*| = its rank (Alg. 2 line 2: "of size l")
    for k in range(1, r.sweeps):
        assert len(r.trace[k].Istar) == r.trace[k - 1].rank
