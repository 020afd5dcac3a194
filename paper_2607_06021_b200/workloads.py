"""Seeded synthetic inputs for the five BASELINE.json configs (C1..C5) and the DST-I sweep.

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU oracle's tests.
It holds none of the method's arithmetic (no DST, no sampling, no QR-of-fibers, no SVD core):
it only draws the right-hand-side factors  F = UF diag(SF) VF^T  as numpy arrays, following the
recipe of SURVEY.md §8(d) / DESIGN.md "Input recipe".  numpy.linalg (LAPACK) is used here for
the *input preparation* of C2/C3/C5 (orthonormalising a separable bump expansion).

The paper measures on no public dataset: its Poisson workload is an analytic separable Gaussian
(PAPER.md:271-274); these configs stand in for it.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

SAFEGUARD_LEN = 64


@dataclass
class Workload:
    name: str
    n: int
    UF: np.ndarray          # (n, rF) column-major friendly (Fortran order)
    SF: np.ndarray          # (rF,)
    VF: np.ndarray          # (n, rF)
    tol: float
    max_rank: int
    oversample: int
    max_sweeps: int
    safeguard: np.ndarray   # int32 pre-drawn random indices (Alg. 4 lines 7-12 randomness as data)
    meta: dict

    @property
    def rF(self) -> int:
        return int(self.SF.shape[0])

    def opts(self) -> dict:
        return dict(tol=self.tol, max_rank=self.max_rank, oversample=self.oversample,
                    max_sweeps=self.max_sweeps, safeguard=self.safeguard)


def grid(n: int) -> np.ndarray:
    """x_i = i h, i = 1..n, h = 1/(n+1) on (0,1)."""
    return np.arange(1, n + 1, dtype=np.float64) / (n + 1)


def _fortran(a: np.ndarray) -> np.ndarray:
    return np.asfortranarray(a, dtype=np.float64)


def _orthonormalise(Gx: np.ndarray, Gy: np.ndarray, amp: np.ndarray, cut: float):
    """F = Gx diag(amp) Gy^T  ->  orthonormal UF, SF, VF (truncated at cut * S_1)."""
    Qx, Rx = np.linalg.qr(Gx)
    Qy, Ry = np.linalg.qr(Gy)
    Uc, S, Vct = np.linalg.svd((Rx * amp[None, :]) @ Ry.T)
    r = max(int(np.sum(S > cut * S[0])), 1)
    return _fortran(Qx @ Uc[:, :r]), S[:r].copy(), _fortran(Qy @ Vct[:r, :].T)


def _bumps(n, rng, nb, sig_lo, sig_hi, c_lo, c_hi, cut=1e-10):
    x = grid(n)
    sig = np.full(nb, sig_lo) if sig_lo == sig_hi else rng.uniform(sig_lo, sig_hi, nb)
    cx = rng.uniform(c_lo, c_hi, nb)
    cy = rng.uniform(c_lo, c_hi, nb)
    Gx = np.exp(-((x[:, None] - cx[None, :]) ** 2) / (2.0 * sig[None, :] ** 2))
    Gy = np.exp(-((x[:, None] - cy[None, :]) ** 2) / (2.0 * sig[None, :] ** 2))
    UF, SF, VF = _orthonormalise(Gx, Gy, np.ones(nb), cut)
    return UF, SF, VF, dict(sigma=sig, cx=cx, cy=cy)


def config1(seed: int = 0, n: int = 255) -> Workload:
    """C1: f = sum_{m=1..4} a_m sin(k_m pi x) sin(l_m pi y), exact rank 4, closed-form solution."""
    rng = np.random.default_rng(seed)
    while True:
        k = rng.integers(1, 17, 4)
        if len(set(k.tolist())) == 4:
            break
    while True:
        l = rng.integers(1, 17, 4)
        if len(set(l.tolist())) == 4:
            break
    a = rng.standard_normal(4)
    x = grid(n)
    sc = np.sqrt(2.0 / (n + 1))
    UF = sc * np.sin(np.pi * np.outer(x, k))
    VF = sc * np.sin(np.pi * np.outer(x, l)) * np.sign(a)[None, :]
    SF = np.abs(a) * (n + 1) / 2.0
    order = np.argsort(-SF, kind="stable")
    safeguard = rng.integers(0, n, SAFEGUARD_LEN).astype(np.int32)
    meta = dict(k=k[order], l=l[order], a=a[order])
    return Workload("C1", n, _fortran(UF[:, order]), SF[order].copy(), _fortran(VF[:, order]),
                    1e-12, 16, 8, 20, safeguard, meta)


def config2(seed: int = 0, n: int = 4095) -> Workload:
    """C2: 3 Gaussian bumps, sigma = 0.05, centres U[0.2,0.8]^2."""
    rng = np.random.default_rng(seed)
    UF, SF, VF, meta = _bumps(n, rng, 3, 0.05, 0.05, 0.2, 0.8)
    safeguard = rng.integers(0, n, SAFEGUARD_LEN).astype(np.int32)
    return Workload("C2", n, UF, SF, VF, 1e-10, 64, 8, 20, safeguard, meta)


def config3(seed: int = 0, n: int = 65535) -> Workload:
    """C3: 8 bumps, sigma U[0.01,0.1], centres U[0.1,0.9]^2, at most 5 sweeps."""
    rng = np.random.default_rng(seed)
    UF, SF, VF, meta = _bumps(n, rng, 8, 0.01, 0.1, 0.1, 0.9)
    safeguard = rng.integers(0, n, SAFEGUARD_LEN).astype(np.int32)
    return Workload("C3", n, UF, SF, VF, 1e-10, 96, 8, 5, safeguard, meta)


def config4(seed: int = 0, n: int = (1 << 20) - 1) -> Workload:
    """C4: random smooth low-rank factors: column c = sum_{k=1..64} g_{k,c} 2^{-k/4} sin(k pi x),
    g ~ N(0,1), 32 columns, S_F(c) = 10^{-c/4}.  Columns deliberately not orthonormal."""
    rng = np.random.default_rng(seed)
    x = grid(n)
    modes = np.arange(1, 65)
    decay = 2.0 ** (-modes / 4.0)
    gU = rng.standard_normal((64, 32)) * decay[:, None]
    gV = rng.standard_normal((64, 32)) * decay[:, None]
    UF = np.zeros((n, 32), order="F")
    VF = np.zeros((n, 32), order="F")
    for k in modes:                                   # column by column to bound temporaries
        s = np.sin(np.pi * k * x)
        UF += np.outer(s, gU[k - 1])
        VF += np.outer(s, gV[k - 1])
    SF = 10.0 ** (-np.arange(32) / 4.0)
    safeguard = rng.integers(0, n, SAFEGUARD_LEN).astype(np.int32)
    return Workload("C4", n, _fortran(UF), SF, _fortran(VF), 1e-10, 64, 8, 20, safeguard,
                    dict(gU=gU, gV=gV))


def config5(seed: int = 0, n: int = (1 << 22) - 1) -> Workload:
    """C5: 32 bumps, sigma U[0.005,0.05], centres U[0.1,0.9]^2, tol 1e-9, 8 sweeps."""
    rng = np.random.default_rng(seed)
    UF, SF, VF, meta = _bumps(n, rng, 32, 0.005, 0.05, 0.1, 0.9, cut=1e-10)
    safeguard = rng.integers(0, n, SAFEGUARD_LEN).astype(np.int32)
    return Workload("C5", n, UF, SF, VF, 1e-9, 128, 8, 8, safeguard, meta)


CONFIGS = {"C1": config1, "C2": config2, "C3": config3, "C4": config4, "C5": config5}


def make(name: str, seed: int = 0, n: int | None = None) -> Workload:
    f = CONFIGS[name]
    return f(seed) if n is None else f(seed, n)


def dst_batch(n: int, batch: int, seed: int = 0) -> np.ndarray:
    """iid N(0,1) columns for the batched DST-I sweep (C5's second half)."""
    rng = np.random.default_rng(seed)
    return np.asfortranarray(rng.standard_normal((n, batch)))


def sample_pairs(n: int, count: int, seed: int = 0, active: int | None = None):
    """`count` random (i, j) pairs; half of them from the low-frequency block [0, active)^2
    when `active` is given (SURVEY.md §8(c) pin (iii))."""
    rng = np.random.default_rng(seed + 12345)
    i = rng.integers(0, n, count)
    j = rng.integers(0, n, count)
    if active is not None:
        h = count // 2
        a = min(active, n)
        i[:h] = rng.integers(0, a, h)
        j[:h] = rng.integers(0, a, h)
    return i.astype(np.int64), j.astype(np.int64)


def matrix_initial_guess(n: int, r0: int = 4, seed: int = 0):
    """Initial guess U0, V0 (n x r0, orthonormal columns) and safeguard list for Cross-DEIM on the paper's test matrices
    (eq. (6)): the paper does not say what Alg. 4's U0, V0 are there; seeded Gaussian columns,
    orthonormalised on the host, are handed to both the CUDA path and the oracle as data."""
    rng = np.random.default_rng(seed + 4242)
    U0, _ = np.linalg.qr(rng.standard_normal((n, r0)))
    V0, _ = np.linalg.qr(rng.standard_normal((n, r0)))
    safeguard = rng.integers(0, n, SAFEGUARD_LEN).astype(np.int32)
    return _fortran(U0), _fortran(V0), safeguard


def paper_eq7(n: int, seed: int = 0) -> Workload:
    """The paper's own Poisson workload, eq. (7): f(x,y) = exp(-36 ((x - 0.1)^2 + (y - 0.55)^2)) on
    [-1,1]^2 (the printed minus sign between the squares is a typo -- either way the forcing is rank-1 separable, DESIGN.md
    reading Q19), grids n = 2^10 .. 2^18, i.e. n + 1 NOT a power of two.  In the solver's unit-square convention
    (s = (x+1)/2, h = 1/(n+1)): -Laplace_s u = 4 f, so S_F = 4.  tol 1e-9, r_max 64."""
    rng = np.random.default_rng(seed)
    x = -1.0 + 2.0 * grid(n)
    UF = np.exp(-36.0 * (x - 0.1) ** 2)[:, None]
    VF = np.exp(-36.0 * (x - 0.55) ** 2)[:, None]
    safeguard = rng.integers(0, n, SAFEGUARD_LEN).astype(np.int32)
    return Workload("eq7", n, _fortran(UF), np.array([4.0]), _fortran(VF), 1e-9, 64, 8, 20, safeguard, dict())
