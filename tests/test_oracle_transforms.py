"""Pins for the oracle's eigenvalues (O1), DST-I (O2) and fiber sampling (O4).
Every check is against something other than the oracle: closed forms, the definition written
as an explicit loop, invariants, scipy's DST, brute force on the full matrix."""
import math
import os

import numpy as np
import pytest
import scipy.fft

from oracle import lrp_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "eigenvalues_d.txt")


def test_eigenvalues_against_decimal_golden():
    # golden values: 60-digit decimal Taylor series (tests/golden/make_eigenvalues_golden.py)
    rows = [l.split() for l in open(GOLDEN) if not l.startswith("#")]
    cache = {}
    for n, k, val in rows:
        n, k, val = int(n), int(k), float(val)
        if n not in cache:
            cache[n] = O.eigenvalues_d(n)
        assert abs(cache[n][k - 1] - val) <= 2.5e-16 * val, (n, k)


@pytest.mark.parametrize("n", [7, 31, 64])
def test_eigenpairs_of_T(n):
    # T z_k = lambda_k z_k with lambda = h^2 d
    T = O.tridiag_T(n)
    h2 = 1.0 / (n + 1) ** 2
    d = O.eigenvalues_d(n)
    i = np.arange(1, n + 1)
    for k in (1, 2, n // 2, n):
        z = math.sqrt(2.0 / (n + 1)) * np.sin(i * k * math.pi / (n + 1))
        assert np.abs(T @ z - h2 * d[k - 1] * z).max() < 1e-14
    assert abs(h2 * d.sum() - 2 * n) < 1e-12 * n          # trace of T
    # 4 sin^2(theta/2) == 2 (1 - cos theta) (the paper's form) where the latter is still accurate
    lam = 2.0 * (1.0 - np.cos(np.pi * i / (n + 1)))
    assert np.abs(lam - h2 * d).max() < 1e-13


def _dst1_loop(x):
    n = len(x)
    return [sum(x[j - 1] * math.sin(j * k * math.pi / (n + 1)) for j in range(1, n + 1))
            for k in range(1, n + 1)]


def test_dst_naive_is_the_definition():
    rng = np.random.default_rng(1)
    x = rng.standard_normal(9)
    assert np.abs(O.dst1_naive(x) - np.array(_dst1_loop(x))).max() < 1e-14
    X = rng.standard_normal((9, 3))
    got = O.dst1_naive(X, scale=0.5)
    for c in range(3):
        assert np.abs(got[:, c] - 0.5 * np.array(_dst1_loop(X[:, c]))).max() < 1e-14


@pytest.mark.parametrize("n", [15, 255, 1023])
def test_dst_against_scipy_and_invariants(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal((n, 2))
    X = O.dst1_naive(x)
    # scipy's DST-I is 2 * sum x_j sin(pi j k/(n+1))
    ref = scipy.fft.dst(x, type=1, axis=0) / 2.0
    assert np.abs(X - ref).max() < 1e-12 * np.abs(ref).max()
    # unnormalised involution: twice = (n+1)/2 * I  (north_star); orthonormal twice = I
    assert np.abs(O.dst1_naive(X) - (n + 1) / 2.0 * x).max() < 1e-11 * n
    sc = O.orthonormal_scale(n)
    Zx = O.dst1_naive(x, sc)
    assert np.abs(O.dst1_naive(Zx, sc) - x).max() < 1e-12
    # Parseval for the orthonormal transform
    assert abs(np.linalg.norm(Zx) - np.linalg.norm(x)) < 1e-12 * np.linalg.norm(x)
    # closed form: DST-I of sin(j m pi/(n+1)) = (n+1)/2 e_m
    m = 3
    s = np.sin(np.arange(1, n + 1) * m * math.pi / (n + 1))
    e = np.zeros(n)
    e[m - 1] = (n + 1) / 2.0
    assert np.abs(O.dst1_naive(s) - e).max() < 1e-11 * n
    # eigen-relation Z (T x) = lambda .* (Z x)
    T = O.tridiag_T(n)
    lam = O.eigenvalues_d(n) / (n + 1) ** 2
    assert np.abs(O.dst1_naive(T @ x, sc) - lam[:, None] * Zx).max() < 1e-12


@pytest.mark.parametrize("n", [255, 4095])
def test_dst_fft_route_matches_definition(n):
    rng = np.random.default_rng(7)
    x = rng.standard_normal((n, 2))
    a = O.dst1_naive(x)
    b = O.dst1_fft(x)
    assert np.abs(a - b).max() < 1e-13 * np.abs(a).max() * math.log2(n + 1)
    ks = np.array([1, 2, n // 3, n])
    e = O.dst1_entries(x[:, 1], ks, scale=2.0)
    assert np.abs(e - 2.0 * a[ks - 1, 1]).max() < 1e-12 * np.abs(a).max()


def test_dst_fft_large_n_invariants():
    n = (1 << 16) - 1
    rng = np.random.default_rng(3)
    x = rng.standard_normal(n)
    sc = O.orthonormal_scale(n)
    Zx = O.dst1(x, sc)
    assert np.abs(O.dst1(Zx, sc) - x).max() < 1e-12
    ks = np.array([1, 77, n])
    assert np.abs(O.dst1_entries(x, ks, sc) - Zx[ks - 1]).max() < 1e-12


def test_fibers_bruteforce_and_symmetry():
    n, r = 63, 5
    rng = np.random.default_rng(0)
    Uh = rng.standard_normal((n, r))
    Vh = rng.standard_normal((n, r))
    S = rng.uniform(0.5, 2.0, r)
    d = O.eigenvalues_d(n)
    # brute force: explicit loops for the whole G (eq. (4))
    G = np.zeros((n, n))
    for i in range(n):
        for j in range(n):
            G[i, j] = sum(Uh[i, t] * S[t] * Vh[j, t] for t in range(r)) / (d[i] + d[j])
    I = np.array([3, 10, 0, 62])
    J = np.array([5, 1, 44])
    C, Rt = O.sample_fibers(Uh, S, Vh, d, I, J)
    assert C.shape == (n, 3) and Rt.shape == (n, 4)
    assert np.abs(C - G[:, J]).max() < 1e-15 * np.abs(G).max() * 10
    assert np.abs(Rt - G[I, :].T).max() < 1e-15 * np.abs(G).max() * 10
    # symmetry: C from (Uh, Vh) equals Rt from (Vh, Uh)
    C2, Rt2 = O.sample_fibers(Vh, S, Uh, d, J, I)
    assert np.array_equal(C, Rt2) and np.array_equal(Rt, C2)
    rows = np.array([0, 5, 62])
    cols = np.array([1, 5, 0])
    assert np.abs(O.G_entries(Uh, S, Vh, d, rows, cols) - G[rows, cols]).max() < 1e-14 * np.abs(G).max()
    L = (Uh * S) @ Vh.T
    assert np.abs(O.lowrank_entries(Uh, S, Vh, rows, cols) - L[rows, cols]).max() < 1e-13


def test_dense_poisson_solves_the_matrix_equation():
    # eq. (3):  T W + W T^T = h^2 F
    n = 31
    rng = np.random.default_rng(5)
    F = rng.standard_normal((n, n))
    W = O.dense_poisson(n, F)
    T = O.tridiag_T(n)
    h2 = 1.0 / (n + 1) ** 2
    assert np.abs(T @ W + W @ T.T - h2 * F).max() < 1e-13
    Z = O.dst1_matrix(n)
    assert np.abs(Z @ Z - np.eye(n)).max() < 1e-14 and np.abs(Z - Z.T).max() == 0.0
