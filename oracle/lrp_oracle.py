"""CPU oracle for the Cross-DEIM low-rank Poisson hot path (arxiv/paper_2607_06021).

TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 numpy restatement of what the hot path
computes, written from PAPER.md (citations are `PAPER.md:<line>` + section/algorithm) under the
readings Q1..Q22 of SURVEY.md §8(c) and Q23..Q26, R1..R7 of DESIGN.md section 2.  It shares no code with the CUDA
path, imports nothing from `paper_2607_06021_b200`, and may only be imported by `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` leg.

Library primitives used as steps: numpy matmul / elementwise ops, `numpy.fft.fft` (only in
`dst1_fft`, the large-n route, which is itself pinned to the O(n^2) definition `dst1_naive`).
QR is an unblocked Householder QR and the SVD is a one-sided (Hestenes) Jacobi SVD written out
below; no LAPACK routine is on the oracle's path (LAPACK is used only by the *tests* as an
independent pin).

Parity pins (tests/test_oracle_*.py, `-m "not gpu"`): every function below is pinned by closed
forms / invariants / brute force as listed in DESIGN.md §"Oracle pins".
Parity unpinned: the *choice* of the constants PINV_RCOND, RANK_RCOND, PRUNE_REL, K_cap, the
initial guess U0=Uhat_F, the Bernoulli constant c = cols + p_os (Q23) and the random initial guess
of the test-matrix runs (Q25) (paper silent; validated only by convergence to the dense
definition), and the paper's seed-dependent iteration counts (figures only).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# ----------------------------------------------------------------------------- constants
# (paper silent on all of them: SURVEY.md §8(c) Q4, Q6, Q10, Q12)
PINV_RCOND = 1e-13      # singular values <= PINV_RCOND * sigma_max are treated as zero in pinv (Q4)
RANK_RCOND = 1e-14      # numerical rank of the core: #{S_c > RANK_RCOND * S_1} (Q4)
LEV_COL_RCOND = 1e-13   # columns of A with |R_cc| < this * max|R_cc| are excluded from leverage (O6)
PRUNE_REL = 1e-12       # PAPER.md:158-177 (Alg. 4 lines 14-23), made relative to max|r| (Q12)
JACOBI_MAX_SWEEPS = 60
_EPS = np.finfo(np.float64).eps
_PI_LD = np.longdouble("3.14159265358979323846264338327950288")


# ----------------------------------------------------------------------------- O1 eigenvalues
def eigenvalues_d(n: int) -> np.ndarray:
    """d_k = lambda_k / h^2 = 4 (n+1)^2 sin^2(pi k / (2(n+1))), k = 1..n.

    PAPER.md:198-200 gives lambda_k = 2(1 - cos(pi k/(n+1))) and h = 1/(n+1);
    eq. (4) divides h^2 Fhat by lambda_i + lambda_j.  Reading Q1: the identical
    form 4 sin^2(theta/2) is used (no cancellation), evaluated in long double and rounded.
    """
    N = n + 1
    k = np.arange(1, n + 1, dtype=np.longdouble)
    s = np.sin(_PI_LD * k / np.longdouble(2 * N))
    d = np.longdouble(4.0) * np.longdouble(N) * np.longdouble(N) * s * s
    return d.astype(np.float64)


# ----------------------------------------------------------------------------- O2 DST-I
def _sin_table(N: int) -> np.ndarray:
    """sin(pi m / N), m = 0..2N-1, evaluated in long double and rounded to fp64."""
    m = np.arange(2 * N, dtype=np.longdouble)
    return np.sin(_PI_LD * m / np.longdouble(N)).astype(np.float64)


def dst1_naive(x: np.ndarray, scale: float = 1.0) -> np.ndarray:
    """DST-I by its definition, O(n^2) per column:  X_k = scale * sum_{j=1}^n x_j sin(j k pi/(n+1)).

    PAPER.md:198-202 (z_k(i) = sqrt(2/(n+1)) sin(i k pi/(n+1))).  The argument
    is reduced exactly in integer arithmetic: sin(pi ((j k) mod 2(n+1)) / (n+1)).
    x is (n,) or (n, batch); columns are transformed independently.
    """
    x = np.asarray(x, dtype=np.float64)
    one_d = x.ndim == 1
    X = x.reshape(x.shape[0], -1)
    n = X.shape[0]
    N = n + 1
    tab = _sin_table(N)
    j = np.arange(1, n + 1, dtype=np.int64)
    out = np.empty_like(X)
    rows_per_block = max(1, (1 << 24) // max(n, 1))     # bound the temporary sine block
    for k0 in range(0, n, rows_per_block):
        k = np.arange(k0 + 1, min(k0 + rows_per_block, n) + 1, dtype=np.int64)
        Sblk = tab[(k[:, None] * j[None, :]) % (2 * N)]
        out[k0:k0 + k.size, :] = Sblk @ X
    out *= scale
    return out[:, 0] if one_d else out


def dst1_fft(x: np.ndarray, scale: float = 1.0) -> np.ndarray:
    """DST-I through the odd extension: y = [0, x_1..x_n, 0, -x_n..-x_1] (length 2(n+1)),
    Y = DFT(y) (numpy.fft.fft used as a library step), X_k = -Im(Y_k)/2.   Used for large n;
    pinned against `dst1_naive` at n = 255 and 4095 (tests).  PAPER.md:202, 216, 226.
    """
    x = np.asarray(x, dtype=np.float64)
    one_d = x.ndim == 1
    X = x.reshape(x.shape[0], -1)
    n, b = X.shape
    N = n + 1
    out = np.empty_like(X)
    for c in range(b):
        y = np.zeros(2 * N, dtype=np.float64)
        y[1:N] = X[:, c]
        y[N + 1:] = -X[::-1, c]
        Y = np.fft.fft(y)
        out[:, c] = -0.5 * Y.imag[1:N]
    out *= scale
    return out[:, 0] if one_d else out


NAIVE_DST_MAX_N = 4095


def dst1(x: np.ndarray, scale: float = 1.0) -> np.ndarray:
    """DST-I: the definition sum for n <= 4095, the odd-extension FFT route above that (O2)."""
    n = np.asarray(x).shape[0]
    return dst1_naive(x, scale) if n <= NAIVE_DST_MAX_N else dst1_fft(x, scale)


def dst1_entries(x: np.ndarray, ks: np.ndarray, scale: float = 1.0) -> np.ndarray:
    """Selected outputs X_k (1-based k in `ks`) of the DST-I of one column x, each by the O(n)
    definition sum with the exact integer argument reduction.  For full-size sampled parity."""
    x = np.asarray(x, dtype=np.float64)
    n = x.shape[0]
    N = n + 1
    j = np.arange(1, n + 1, dtype=np.int64)
    out = np.empty(len(ks), dtype=np.float64)
    for t, k in enumerate(np.asarray(ks, dtype=np.int64)):
        m = (j * int(k)) % (2 * N)
        s = np.sin(_PI_LD * m.astype(np.longdouble) / np.longdouble(N)).astype(np.float64)
        out[t] = math.fsum(s * x) * scale
    return out


def orthonormal_scale(n: int) -> float:
    """sqrt(2/(n+1)): with it DST-I is the symmetric orthogonal Z of PAPER.md:198-200, so
    DST(DST(I)) = I."""
    return math.sqrt(2.0 / (n + 1))


# ----------------------------------------------------------------------------- O4 fibers
def sample_fibers(Uh: np.ndarray, S: np.ndarray, Vh: np.ndarray, d: np.ndarray,
                  I: np.ndarray, J: np.ndarray):
    """C = G(:, J) (n x |J|) and Rt = G(I, :)^T (n x |I|) of
    G(i,j) = (sum_t Uh(i,t) S(t) Vh(j,t)) / (d_i + d_j)       eq. (4), PAPER.md:213, 230;
    Alg. 1 line 3.  O(r) per entry; the n^2 matrix is never formed.
    """
    I = np.asarray(I, dtype=np.int64)
    J = np.asarray(J, dtype=np.int64)
    C = ((Uh * S[None, :]) @ Vh[J, :].T) / (d[:, None] + d[J][None, :])
    Rt = ((Vh * S[None, :]) @ Uh[I, :].T) / (d[:, None] + d[I][None, :])
    return C, Rt


def G_entries(Uh, S, Vh, d, rows, cols) -> np.ndarray:
    """G(rows[t], cols[t]) one by one (pairs, not the outer product)."""
    rows = np.asarray(rows, dtype=np.int64)
    cols = np.asarray(cols, dtype=np.int64)
    num = np.einsum("tk,k,tk->t", Uh[rows, :], S, Vh[cols, :])
    return num / (d[rows] + d[cols])


def lowrank_entries(U, S, V, rows, cols) -> np.ndarray:
    """(U diag(S) V^T)(rows[t], cols[t]) -- X(i,j) = sum_k sigma_k u_k(i) v_k(j)."""
    rows = np.asarray(rows, dtype=np.int64)
    cols = np.asarray(cols, dtype=np.int64)
    return np.einsum("tk,k,tk->t", U[rows, :], S, V[cols, :])


# ----------------------------------------------------------------------------- Householder QR
def householder_qr(A: np.ndarray):
    """Thin, unpivoted Householder QR, A (m x k) = Q (m x p) R (p x k), p = min(m, k).
    Alg. 1 line 4 "Perform QR".  Reflector H_j = I - tau v v^T, v(0) = 1,
    beta = -sign(alpha) ||x||, tau = (beta - alpha)/beta  (textbook / LAPACK dlarfg convention).
    """
    A = np.array(A, dtype=np.float64, copy=True)
    m, k = A.shape
    p = min(m, k)
    vs = []
    taus = np.zeros(p)
    for j in range(p):
        x = A[j:, j]
        alpha = x[0]
        xnorm = np.linalg.norm(x[1:]) if x.size > 1 else 0.0
        if xnorm == 0.0:
            v = np.zeros_like(x)
            v[0] = 1.0
            taus[j] = 0.0
            vs.append(v)
            continue
        beta = -math.copysign(math.hypot(alpha, xnorm), alpha)
        tau = (beta - alpha) / beta
        v = x / (alpha - beta)
        v[0] = 1.0
        taus[j] = tau
        vs.append(v.copy())
        A[j, j] = beta
        A[j + 1:, j] = 0.0
        if j + 1 < k:
            w = v @ A[j:, j + 1:]
            A[j:, j + 1:] -= tau * np.outer(v, w)
    R = np.triu(A[:p, :])
    Q = np.zeros((m, p))
    Q[np.arange(p), np.arange(p)] = 1.0
    for j in range(p - 1, -1, -1):
        v = vs[j]
        w = v @ Q[j:, j:]
        Q[j:, j:] -= taus[j] * np.outer(v, w)
    return Q, R


# ----------------------------------------------------------------------------- Jacobi SVD
def jacobi_svd(M: np.ndarray):
    """One-sided (Hestenes) Jacobi SVD, cyclic-by-rows pair order.  M (m x n) = U diag(s) V^T,
    U (m x p), V (n x p), p = min(m, n), s sorted descending.  Alg. 1 lines 8/12
    "Perform truncated SVD" -- the truncation is applied by the caller.
    Columns of U belonging to exactly-zero singular values are zero vectors.
    """
    M = np.asarray(M, dtype=np.float64)
    transposed = M.shape[0] < M.shape[1]
    A = np.array(M.T if transposed else M, dtype=np.float64, copy=True)
    m, n = A.shape
    V = np.eye(n)
    for _ in range(JACOBI_MAX_SWEEPS):
        rotated = False
        for p in range(n - 1):
            for q in range(p + 1, n):
                ap = A[:, p]
                aq = A[:, q]
                alpha = ap @ ap
                beta = aq @ aq
                gamma = ap @ aq
                if gamma == 0.0 or abs(gamma) <= _EPS * math.sqrt(alpha * beta):
                    continue
                rotated = True
                zeta = (beta - alpha) / (2.0 * gamma)
                t = math.copysign(1.0, zeta) / (abs(zeta) + math.sqrt(1.0 + zeta * zeta))
                c = 1.0 / math.sqrt(1.0 + t * t)
                s = c * t
                A[:, p], A[:, q] = c * ap - s * aq, s * ap + c * aq
                vp = V[:, p].copy()
                vq = V[:, q]
                V[:, p], V[:, q] = c * vp - s * vq, s * vp + c * vq
        if not rotated:
            break
    sv = np.sqrt(np.einsum("ij,ij->j", A, A))
    order = np.argsort(-sv, kind="stable")
    sv = sv[order]
    A = A[:, order]
    V = V[:, order]
    U = np.zeros_like(A)
    nz = sv > 0.0
    U[:, nz] = A[:, nz] / sv[nz]
    if transposed:
        return V, sv, U
    return U, sv, V


def pinv_svd(M: np.ndarray, rcond: float = PINV_RCOND) -> np.ndarray:
    """Moore-Penrose pseudo-inverse through the Jacobi SVD, relative cut `rcond` (reading Q4;
    Alg. 1 lines 6-7 / 11-12: "truncated SVD pseudoinverse" / torch.linalg.pinv)."""
    U, s, V = jacobi_svd(M)
    if s.size == 0 or s[0] == 0.0:
        return np.zeros((M.shape[1], M.shape[0]))
    keep = s > rcond * s[0]
    return (V[:, keep] / s[keep][None, :]) @ U[:, keep].T


def sigma_min(M: np.ndarray) -> float:
    """Smallest of the min(rows, cols) singular values of M (0.0 for an empty matrix)."""
    if M.shape[0] == 0 or M.shape[1] == 0:
        return 0.0
    _, s, _ = jacobi_svd(M)
    return float(s[-1])


# ----------------------------------------------------------------------------- O6 leverage
def leverage_scores(A: np.ndarray, assume_orthonormal: bool = False) -> np.ndarray:
    """l_i = ||Q(i,:)||^2 with A = QR the thin Householder QR (Alg. 3 line 3, without
    the rank-independent 1/k factor: reading Q5).  Columns with |R_cc| < 1e-13 max|R_cc| carry no
    direction of range(A) and are excluded (O6)."""
    if assume_orthonormal:
        return np.einsum("ij,ij->i", A, A)
    Q, R = householder_qr(A)
    dg = np.abs(np.diag(R))
    keep = dg >= LEV_COL_RCOND * dg.max() if dg.size and dg.max() > 0 else np.zeros(dg.size, bool)
    Qk = Q[:, keep]
    return np.einsum("ij,ij->i", Qk, Qk)


def top_select(scores: np.ndarray, num_select: int) -> np.ndarray:
    """The num_select largest scores, ordered by (score desc, index asc) -- deterministic top-k
    form of Alg. 3 lines 4-6 per north_star / reading Q5."""
    n = scores.shape[0]
    num_select = min(num_select, n)
    order = np.lexsort((np.arange(n), -scores))
    return order[:num_select].astype(np.int32)


def leverage_select(A: np.ndarray, num_select: int, assume_orthonormal: bool = False):
    sc = leverage_scores(A, assume_orthonormal)
    return top_select(sc, num_select), sc


# ----------------------------------------------------------------------------- Alg. 3 lines 4-5, randomized form
_M64 = (1 << 64) - 1


def counter_uniforms(seed: int, sweep: int, side: int, n: int) -> np.ndarray:
    """u_i in [0, 1), i = 0..n-1: a counter-based generator (SplitMix64 finaliser of a key built from seed, sweep, side
    and i), so that the CUDA path and this oracle draw the SAME numbers without sharing code or state (the paper's
    randomness is not reproducible across devices):
        x = seed + 0x9E3779B97F4A7C15 (1 + 2 sweep + side);   z = x + 0xD1B54A32D192ED03 (i + 1)        (mod 2^64)
        z = (z xor z>>30) 0xBF58476D1CE4E5B9;  z = (z xor z>>27) 0x94D049BB133111EB;  z = z xor z>>31
        u = (z >> 11) 2^-53."""
    x = (int(seed) + 0x9E3779B97F4A7C15 * (1 + 2 * int(sweep) + int(side))) & _M64
    with np.errstate(over="ignore"):
        z = np.uint64(x) + np.uint64(0xD1B54A32D192ED03) * (np.arange(n, dtype=np.uint64) + np.uint64(1))
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


def bernoulli_select(scores: np.ndarray, cols: int, c: float, u: np.ndarray, cap: int) -> np.ndarray:
    """Alg. 3 lines 3-6 as printed: pi_i = scores_i / cols (the 1/k-normalised leverage, sum = 1),
    keep index i with probability p_i = min{1, c pi_i}: i is kept iff u_i < p_i.  The kept indices are returned in
    (score desc, index asc) order (reading Q8), at most `cap` of them (the best-scoring ones)."""
    p = np.minimum(1.0, c * (scores / cols))
    kept = np.nonzero(u < p)[0]
    order = np.lexsort((kept, -scores[kept]))
    return kept[order][:cap].astype(np.int32)


# ----------------------------------------------------------------------------- Alg. 2: DEIM / QDEIM
def qdeim_select(U: np.ndarray) -> np.ndarray:
    """QDEIM (Alg. 2 lines 7-10): column-pivoted Householder QR of U^T (cols x n); the pivot columns, in
    pivot order, are the selected row indices of U (as many as U has columns).  Written out: at step c the column of
    the trailing block with the largest 2-norm (recomputed exactly, lowest index on ties) is swapped to position c, a
    Householder reflector annihilates it below the diagonal and is applied to the remaining columns."""
    A = np.array(np.asarray(U, dtype=np.float64).T, copy=True)           # cols x n
    r, n = A.shape
    perm = np.arange(n)
    steps = min(r, n)
    for c in range(steps):
        nrm2 = np.einsum("ij,ij->j", A[c:, c:], A[c:, c:])
        j = c + int(np.argmax(nrm2))                                       # first maximum = lowest index on ties
        if j != c:
            A[:, [c, j]] = A[:, [j, c]]
            perm[[c, j]] = perm[[j, c]]
        x = A[c:, c].copy()
        alpha = x[0]
        xnorm = np.linalg.norm(x[1:]) if x.size > 1 else 0.0
        if xnorm != 0.0:
            beta = -math.copysign(math.hypot(alpha, xnorm), alpha)
            tau = (beta - alpha) / beta
            v = x / (alpha - beta)
            v[0] = 1.0
            A[c:, c:] -= tau * np.outer(v, v @ A[c:, c:])
    return perm[:steps].astype(np.int32)


def deim_select(U: np.ndarray) -> np.ndarray:
    """DEIM (Alg. 2 lines 3-6): LU with partial (row) pivoting of U (n x cols); the pivot rows, in pivot
    order, are the selected indices.  Written out: at step c the row with the largest |entry| of column c among the
    rows not yet chosen (lowest index on ties) becomes the pivot, and column c is eliminated from the other unchosen rows."""
    A = np.array(U, dtype=np.float64, copy=True)
    n, r = A.shape
    free = np.ones(n, dtype=bool)
    out = []
    for c in range(min(r, n)):
        col = np.where(free, np.abs(A[:, c]), -1.0)
        p = int(np.argmax(col))
        out.append(p)
        free[p] = False
        if A[p, c] != 0.0 and c + 1 < r:
            m = A[:, c] / A[p, c]
            m[~free] = 0.0
            A[:, c + 1:] -= np.outer(m, A[p, c + 1:])
    return np.asarray(out, dtype=np.int32)


# ----------------------------------------------------------------------------- O8 scross
@dataclass
class ScrossResult:
    U: np.ndarray
    S: np.ndarray
    V: np.ndarray
    rC: np.ndarray
    rR: np.ndarray
    rank: int
    smin_full: float
    S_full: np.ndarray = field(default=None)


def scross(C: np.ndarray, Rt: np.ndarray, I: np.ndarray, J: np.ndarray) -> ScrossResult:
    """Algorithm 1 on already sampled fibers C = G(:,J) (n x k), Rt = G(I,:)^T
    (n x l); k = #J, l = #I (reading Q2).
      line 4 : C = Q R_C, R^T = Z R_R
      k <= l : solve Q(I,:) W = R  by the SVD pseudo-inverse; with R = R_R^T Z^T only the k x l
               core M = Q(I,:)^+ R_R^T is decomposed (reading Q4), W = M Z^T
      k >  l : solve Z(J,:) W = C^T (reading Q3: Z(J,:)), W^T = Q R_C Z(J,:)^+T, M = (Z(J,:)^+ R_C^T)^T
      M = Uh S Vh^T (Jacobi SVD); U = Q Uh, V = Z Vh; r_C = |diag R_C|, r_R = |diag R_R| (line 16).
    smin_full is the smallest singular value of the untruncated core (reading Q11)."""
    I = np.asarray(I, dtype=np.int64)
    J = np.asarray(J, dtype=np.int64)
    k = C.shape[1]
    l = Rt.shape[1]
    Q, RC = householder_qr(C)
    Z, RR = householder_qr(Rt)
    rC = np.abs(np.diag(RC))
    rR = np.abs(np.diag(RR))
    if k <= l:
        P = pinv_svd(Q[I, :])            # k x l
        M = P @ RR.T                     # k x l
    else:
        P = pinv_svd(Z[J, :])            # l x k
        M = (P @ RC.T).T                 # k x l
    Uh, S, Vh = jacobi_svd(M)
    smin_full = float(S[-1])
    rank = max(int(np.sum(S > RANK_RCOND * S[0])), 1) if S[0] > 0 else 1
    U = Q @ Uh[:, :rank]
    V = Z @ Vh[:, :rank]
    return ScrossResult(U=U, S=S[:rank].copy(), V=V, rC=rC, rR=rR, rank=rank,
                        smin_full=smin_full, S_full=S)


# ----------------------------------------------------------------------------- O10 pieces
def rho_factored(Uk, Sk, Vk, Up, Sp, Vp) -> float:
    """rho = || U_k S_k V_k^T - U_{k-1} S_{k-1} V_{k-1}^T ||_F  (Alg. 4 line 24),
    Frobenius, in factored form (reading Q13):  || R_a diag(S_k, -S_{k-1}) R_b^T ||_F with
    [U_k U_{k-1}] = Q_a R_a,  [V_k V_{k-1}] = Q_b R_b.   Previous iterate = 0 at k = 0."""
    if Up is None or Up.shape[1] == 0:
        return float(np.linalg.norm(Sk))
    _, Ra = householder_qr(np.hstack([Uk, Up]))
    _, Rb = householder_qr(np.hstack([Vk, Vp]))
    D = np.concatenate([Sk, -Sp])
    return float(np.linalg.norm((Ra * D[None, :]) @ Rb.T, "fro"))


def eta_of(Uk: np.ndarray, idx: np.ndarray) -> float:
    """eta = || (U_k(idx,:))^+ ||_2 = 1 / sigma_min(U_k(idx,:))  (Alg. 4 line 25, PAPER.md:180;
    reading Q14).  +inf when sigma_min = 0 or the index set is empty."""
    idx = np.asarray(idx, dtype=np.int64)
    if idx.size == 0:
        return math.inf
    sm = sigma_min(Uk[idx, :])
    return math.inf if sm == 0.0 else 1.0 / sm


def indicator(eta1: float, eta2: float, smin_full: float) -> float:
    """min(eta1 (1+eta2), eta2 (1+eta1)) * S_min  (Alg. 4 line 26); 0 * inf := 0."""
    if smin_full == 0.0:
        return 0.0
    return min(eta1 * (1.0 + eta2), eta2 * (1.0 + eta1)) * smin_full


def final_rank(S: np.ndarray, tol: float, max_rank: int, tol_mode: int = 0) -> int:
    """Alg. 4 lines 30-31: smallest r* with sum_{c>r*} S_c^2 < eps^2 (x sum S^2 in
    relative mode, reading Q15);  r = max(min(r*, r_max), 1)."""
    S2 = np.asarray(S, dtype=np.float64) ** 2
    thresh = tol * tol * (S2.sum() if tol_mode == 0 else 1.0)
    rstar = S2.size
    tail = 0.0
    for c in range(S2.size - 1, -1, -1):          # tail sums accumulated from the small end
        tail += S2[c]
        if tail < thresh:
            rstar = c
        else:
            break
    return max(min(rstar, max_rank), 1)


# ----------------------------------------------------------------------------- O5-O12 solve
@dataclass
class SweepRecord:
    I: np.ndarray          # I_k after union/safeguard, before pruning
    J: np.ndarray
    keepI: np.ndarray      # prune masks (True = survives)
    keepJ: np.ndarray
    Istar: np.ndarray      # leverage selections (empty under replay)
    Jstar: np.ndarray
    rank: int
    rho: float
    ind: float
    eta1: float
    eta2: float
    smin_full: float
    snorm: float
    scoresU: np.ndarray = field(default=None, repr=False)
    scoresV: np.ndarray = field(default=None, repr=False)
    rC: np.ndarray = field(default=None, repr=False)
    rR: np.ndarray = field(default=None, repr=False)


@dataclass
class SolveResult:
    UW: np.ndarray         # physical-space factors, W ~= UW diag(SW) VW^T
    SW: np.ndarray
    VW: np.ndarray
    Uhat: np.ndarray       # spectral iterate before the final truncation (all r_k columns)
    Shat: np.ndarray
    Vhat: np.ndarray
    UhF: np.ndarray        # spectral RHS factors
    VhF: np.ndarray
    d: np.ndarray
    rank: int
    sweeps: int
    converged: bool
    trace: list
    rank_capped: bool = False   # r* > r_max (Alg. 4 line 31): the truncated result does not meet the tolerance (reading Q20)


def _union(prev: np.ndarray, star: np.ndarray) -> tuple[np.ndarray, int]:
    """I_k = [survivors of I_{k-1}, in stored order] ++ [members of I* not present, in I*'s order]
    (Alg. 4 line 6; reading Q8)."""
    present = set(int(v) for v in prev)
    out = [int(v) for v in prev]
    added = 0
    for v in star:
        v = int(v)
        if v not in present:
            out.append(v)
            present.add(v)
            added += 1
    return np.asarray(out, dtype=np.int32), added


def _safeguard(cur: np.ndarray, safeguard, scores) -> np.ndarray:
    """Append one index from the complement (Alg. 4 lines 7-12; reading Q9):
    the first entry of the pre-drawn list not in the set; when the list is exhausted, the
    best-scoring index not in the set."""
    present = set(int(v) for v in cur)
    if safeguard is not None:
        for cand in safeguard:
            cand = int(cand)
            if cand not in present:
                return np.append(cur, np.int32(cand)).astype(np.int32)
    order = np.lexsort((np.arange(scores.shape[0]), -scores))
    for cand in order:
        if int(cand) not in present:
            return np.append(cur, np.int32(cand)).astype(np.int32)
    return cur


@dataclass
class CrossDeimResult:
    U: np.ndarray          # last iterate before the final truncation (all r_k columns)
    S: np.ndarray
    V: np.ndarray
    rank: int              # r of Alg. 4 lines 30-32
    sweeps: int
    converged: bool
    trace: list
    rank_capped: bool = False


def cross_deim(n: int, fibers, U0: np.ndarray, V0: np.ndarray, *, tol: float, max_rank: int, oversample: int = 8,
               max_sweeps: int = 20, safeguard=None, tol_mode: int = 0, replay=None,
               selection: str = "topk", ls_seed: int = 0, ls_c: float = 0.0) -> CrossDeimResult:
    """Algorithm 4 for a matrix given as a function handle ("G(i,j) as a function
    handle"): `fibers(I, J)` returns C = G(:, J) (n x |J|) and Rt = G(I, :)^T (n x |I|).  Leverage-score selection
    (Alg. 3), scross (Alg. 1).  U0, V0: initial guess of Alg. 4,
    used for the first selection only.  Steps O5-O11 of SURVEY.md 8(c); square case m = n.

    replay: optional list of dicts {I, J, keepI, keepJ} (one per sweep) + key 'final_rank' on the last one; then
    selection, union, safeguard, prune and stopping decisions are taken from it.
    selection: "topk" = the deterministic top-(cols + p_os) form (reading Q5); "bernoulli" = Alg. 3 lines 4-5 as printed,
    with c = ls_c if ls_c > 0 else cols + p_os (expected sample size <= the deterministic form's count) and uniforms
    from `counter_uniforms(ls_seed, sweep, side, n)` (side 0: rows / U, side 1: columns / V); "qdeim" / "deim" = Alg. 2
    applied to the orthonormal factor of the previous iterate (its thin QR; cols indices, in pivot order).
    """
    K_cap = 2 * (max_rank + oversample)                      # reading Q10
    Uprev_sel = np.asarray(U0)                               # O5 (reading Q7)
    Vprev_sel = np.asarray(V0)
    I_prev = np.zeros(0, dtype=np.int32)
    J_prev = np.zeros(0, dtype=np.int32)
    Up = Sp = Vp = None
    trace: list = []
    converged = False
    res = None
    nsweeps = max_sweeps if replay is None else len(replay)
    for k in range(nsweeps):
        if replay is None:
            # O6: selection. k = 0 (user factors) needs the QR; later iterates are orthonormal
            # up to rounding, for which the QR is the identity (reading Q6) -- the oracle still
            # performs it, as the definition.
            if selection in ("qdeim", "deim"):
                QU, _ = householder_qr(Uprev_sel)            # Alg. 2 line 1: "Input: orthogonal matrix U"
                QV, _ = householder_qr(Vprev_sel)
                scU = np.einsum("ij,ij->i", QU, QU)          # kept for the safeguard fallback and the trace
                scV = np.einsum("ij,ij->i", QV, QV)
                Istar = qdeim_select(QU) if selection == "qdeim" else deim_select(QU)
                Jstar = qdeim_select(QV) if selection == "qdeim" else deim_select(QV)
            elif selection == "bernoulli":
                scU = leverage_scores(Uprev_sel)
                scV = leverage_scores(Vprev_sel)
                cU = ls_c if ls_c > 0 else float(Uprev_sel.shape[1] + oversample)
                cV = ls_c if ls_c > 0 else float(Vprev_sel.shape[1] + oversample)
                Istar = bernoulli_select(scU, Uprev_sel.shape[1], cU, counter_uniforms(ls_seed, k, 0, n), 2 * K_cap)
                Jstar = bernoulli_select(scV, Vprev_sel.shape[1], cV, counter_uniforms(ls_seed, k, 1, n), 2 * K_cap)
            else:
                Istar, scU = leverage_select(Uprev_sel, min(Uprev_sel.shape[1] + oversample, n))
                Jstar, scV = leverage_select(Vprev_sel, min(Vprev_sel.shape[1] + oversample, n))
            I_k, addedI = _union(I_prev, Istar)              # O7
            J_k, addedJ = _union(J_prev, Jstar)
            if addedI == 0 or k == 0:
                I_k = _safeguard(I_k, safeguard, scU)
            if addedJ == 0 or k == 0:
                J_k = _safeguard(J_k, safeguard, scV)
            I_k = I_k[:K_cap]
            J_k = J_k[:K_cap]
        else:
            Istar = Jstar = np.zeros(0, dtype=np.int32)
            scU = scV = None
            I_k = np.asarray(replay[k]["I"], dtype=np.int32)
            J_k = np.asarray(replay[k]["J"], dtype=np.int32)
        C, Rt = fibers(I_k, J_k)                             # O4
        res = scross(C, Rt, I_k, J_k)                        # O8
        if replay is None or replay[k].get("keepI") is None:
            keepI = res.rR >= PRUNE_REL * res.rR.max()       # O9 (rows of R <-> I)
            keepJ = res.rC >= PRUNE_REL * res.rC.max()       #    (columns of C <-> J)
        else:
            keepI = np.asarray(replay[k]["keepI"], dtype=bool)
            keepJ = np.asarray(replay[k]["keepJ"], dtype=bool)
        I_pr = I_k[keepI]
        J_pr = J_k[keepJ]
        rho = rho_factored(res.U, res.S, res.V, Up, Sp, Vp)  # O10
        eta1 = eta_of(res.U, I_pr)
        eta2 = eta_of(res.V, J_pr)
        ind = indicator(eta1, eta2, res.smin_full)
        snorm = float(np.linalg.norm(res.S))
        trace.append(SweepRecord(I=I_k.copy(), J=J_k.copy(), keepI=keepI.copy(), keepJ=keepJ.copy(),
                                 Istar=np.asarray(Istar), Jstar=np.asarray(Jstar), rank=res.rank,
                                 rho=rho, ind=ind, eta1=eta1, eta2=eta2, smin_full=res.smin_full,
                                 snorm=snorm, scoresU=scU, scoresV=scV, rC=res.rC, rR=res.rR))
        Up, Sp, Vp = res.U, res.S, res.V
        Uprev_sel, Vprev_sel = res.U, res.V
        I_prev, J_prev = I_pr, J_pr
        thresh = tol * (snorm if tol_mode == 0 else 1.0)
        if replay is None and max(rho, ind) < thresh:        # Alg. 4 line 26, Q15
            converged = True
            break
    rank_capped = False
    if replay is not None and replay[-1].get("final_rank"):
        r = int(replay[-1]["final_rank"])
        converged = True
    else:
        r = final_rank(res.S, tol, max_rank, tol_mode)       # O11
        rank_capped = final_rank(res.S, tol, res.S.size + 1, tol_mode) > max_rank      # reading Q20: r* > r_max
    r = min(r, res.rank)
    return CrossDeimResult(U=res.U, S=res.S, V=res.V, rank=r, sweeps=len(trace), converged=converged, trace=trace,
                           rank_capped=rank_capped)


def cross_deim_solve(n: int, UF: np.ndarray, SF: np.ndarray, VF: np.ndarray, *, tol: float,
                     max_rank: int, oversample: int = 8, max_sweeps: int = 20,
                     safeguard=None, tol_mode: int = 0, U0=None, V0=None,
                     replay=None, selection: str = "topk", ls_seed: int = 0, ls_c: float = 0.0) -> SolveResult:
    """Low-rank Poisson solve of T W + W T^T = h^2 F, F = UF diag(SF) VF^T  (PAPER.md:194-196,
    222-236): Cross-DEIM (`cross_deim` above) on the spectral solution G(i,j) = (Uh S Vh^T)(i,j)/(d_i + d_j) (eq. (4),
    PAPER.md:213) between two batched DST-I.  Steps O1-O12 of SURVEY.md 8(c).
    """
    scale = orthonormal_scale(n)
    d = eigenvalues_d(n)                                     # O1
    UhF = dst1(UF, scale)                                    # O3
    VhF = dst1(VF, scale)
    SF = np.asarray(SF, dtype=np.float64)
    cd = cross_deim(n, lambda I, J: sample_fibers(UhF, SF, VhF, d, I, J),
                    UhF if U0 is None else np.asarray(U0), VhF if V0 is None else np.asarray(V0),     # O5 (reading Q7)
                    tol=tol, max_rank=max_rank, oversample=oversample, max_sweeps=max_sweeps, safeguard=safeguard,
                    tol_mode=tol_mode, replay=replay, selection=selection, ls_seed=ls_seed, ls_c=ls_c)
    r = cd.rank
    UW = dst1(cd.U[:, :r], scale)                            # O12
    VW = dst1(cd.V[:, :r], scale)
    return SolveResult(UW=UW, SW=cd.S[:r].copy(), VW=VW, Uhat=cd.U, Shat=cd.S, Vhat=cd.V,
                       UhF=UhF, VhF=VhF, d=d, rank=r, sweeps=cd.sweeps, converged=cd.converged,
                       trace=cd.trace, rank_capped=cd.rank_capped)


# ----------------------------------------------------------------------------- test matrices (eq. (6))
def hilbert_entries(rows, cols) -> np.ndarray:
    """H(i,j) = 1 / (1 + i + j), 0-based i, j: the Hilbert matrix of eq. (6), PAPER.md:264-266 (rapid singular value decay)."""
    rows = np.asarray(rows, dtype=np.float64)
    cols = np.asarray(cols, dtype=np.float64)
    return 1.0 / (1.0 + rows + cols)


def kmatrix_entries(n: int, rows, cols) -> np.ndarray:
    """K(i,j) = (|x_i + y_j| / 2)^5 on x_i = -1 + 2 i/(n-1), y_j = -1 + 2 j/(n-1), 0-based (eq. (6), PAPER.md:264-267,
    whose grid is printed 1-based): C^4 with a kink along x + y = 0, slow singular value decay."""
    x = -1.0 + 2.0 * np.asarray(rows, dtype=np.float64) / (n - 1)
    y = -1.0 + 2.0 * np.asarray(cols, dtype=np.float64) / (n - 1)
    return (np.abs(x + y) / 2.0) ** 5


def matrix_fibers(kind: str, n: int):
    """Function handle `fibers(I, J) -> (C, Rt)` of a test matrix of eq. (6) ('hilbert' or 'kmatrix'), square n x n."""
    i = np.arange(n)

    def entries(r, c):
        return hilbert_entries(r, c) if kind == "hilbert" else kmatrix_entries(n, r, c)

    def fibers(I, J):
        I = np.asarray(I, dtype=np.int64)
        J = np.asarray(J, dtype=np.int64)
        C = entries(i[:, None], J[None, :])                  # G(:, J)
        Rt = entries(I[None, :], i[:, None])                 # G(I, :)^T: row c of G(I,:) is column c
        return C, Rt
    return fibers


def trace_to_replay(trace, final_rank_value: int | None = None) -> list:
    rep = [dict(I=np.asarray(t.I), J=np.asarray(t.J), keepI=np.asarray(t.keepI),
                keepJ=np.asarray(t.keepJ)) for t in trace]
    if final_rank_value:
        rep[-1]["final_rank"] = int(final_rank_value)
    return rep


# ----------------------------------------------------------------------------- dense truth (A8)
def dst1_matrix(n: int) -> np.ndarray:
    """The orthonormal Z of PAPER.md:198-200 as a dense n x n matrix (tiny n only)."""
    N = n + 1
    tab = _sin_table(N)
    j = np.arange(1, n + 1, dtype=np.int64)
    return orthonormal_scale(n) * tab[(j[:, None] * j[None, :]) % (2 * N)]


def dense_poisson(n: int, F: np.ndarray) -> np.ndarray:
    """Full-rank DST solver of §3.1: What = Z F Z ./ (d_i + d_j), W = Z What Z
    (eq. (4) with the h^2 folded into d = lambda/h^2).  O(n^3) here; tiny grids only."""
    Z = dst1_matrix(n)
    d = eigenvalues_d(n)
    Fh = Z @ F @ Z
    Wh = Fh / (d[:, None] + d[None, :])
    return Z @ Wh @ Z


def tridiag_T(n: int) -> np.ndarray:
    """T = tridiag(-1, 2, -1) of eq. (3)."""
    return 2.0 * np.eye(n) - np.eye(n, k=1) - np.eye(n, k=-1)
