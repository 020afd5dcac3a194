// core.cu -- the small dense core of scross and of the Cross-DEIM stop test, one CTA per problem:
//   one-sided (Hestenes) Jacobi SVD, SVD pseudo-inverse, the k x l core M of Alg. 1 lines 5-15,
//   eta = 1/sigma_min(U_k(I_k,:)) (Alg. 4 line 25) and rho (Alg. 4 line 24).
// Everything here is K x K (K <= a few hundred): latency-bound, not a roofline item.  Matrices live in the
// caller's workspace (L1/L2 resident for the single CTA that touches them), column-major.
#include "common.cuh"
#include "core.cuh"
#include <math.h>
#include <float.h>

namespace {

constexpr int CORE_NT = 512;
constexpr int JACOBI_MAX_SWEEPS = 60;

// 1/sqrt(x) and 1/x for normal positive x to ~1 ulp, branch free: the hardware seed (MUFU.RSQ64H / RCP64H, ~22 bits)
// plus one cubically / two quadratically convergent correction steps.  The library routines cost ~3x the fp64
// instructions (slow-path checks), and every lane of every warp of the Jacobi sweep executes them.
__device__ __forceinline__ double fast_rsqrt(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double r2 = y * y, e = fma(-x, r2, 1.0), t = fma(e, 0.375, 0.5), u = y * e;
    return fma(t, u, y);
}
__device__ __forceinline__ double fast_rcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    e = fma(e, e, e);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}

// Column access of the small dense kernels.  SH: the pointer is known to lie in shared memory -- explicit ld.shared /
// st.shared through the 32-bit window address (a generic LD / ST would be emitted otherwise: the working set is chosen
// between shared and global memory at run time).
template <bool SH> struct ColPtr {
    double* g; unsigned s;
    __device__ __forceinline__ explicit ColPtr(double* p) : g(p), s(SH ? (unsigned)__cvta_generic_to_shared(p) : 0u) {}
    __device__ __forceinline__ double ld(int t) const {
        if (SH) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(s + 8u * (unsigned)t)); return v; }
        return g[t];
    }
    __device__ __forceinline__ void st(int t, double v) const {
        if (SH) asm volatile("st.shared.f64 [%0], %1;" :: "r"(s + 8u * (unsigned)t), "d"(v) : "memory");
        else g[t] = v;
    }
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

// One round of the tournament with G lanes per column pair (32 / G pairs per warp, JR rows per lane: m <= G JR).  The
// two columns, the two columns of V and the two running norms are all requested up front and stay in registers until
// the rotated stores; the reductions take log2(G) shuffles and one warp instruction serves 32 / G pairs.  A round is the
// dependent chain of one pair (load, dot, reduce, rotation parameters, rotate, store, barrier): measured 1350-1900
// cycles per round at 57 x 56 whatever G (profiles/r02_core_jacobi.md); G = 16 is the fastest by a few per cent.
// SH: A, V and nrm2 are in shared memory -- explicit ld.shared / st.shared (ColPtr) instead of generic accesses.
// Pairs of a round are disjoint: no ordering inside it.
template <int G, int JR, bool SH>
__device__ __forceinline__ void jacobi_round_sub(double* __restrict__ A, int lda, int m, int n, double* __restrict__ V, int ldv,
                                                 double* __restrict__ nrm2, int np, int r, int* s_flag) {
    constexpr int GPW = 32 / G;
    const int tid = threadIdx.x, lane = tid & 31, gl = lane & (G - 1);
    const int ngroups = (blockDim.x >> 5) * GPW;
    const bool hasV = V != nullptr;
    for (int i0 = (tid >> 5) * GPW; i0 < np / 2; i0 += ngroups) {          // warp-uniform bounds
        const int i = i0 + lane / G;
        int p = 0, q = 0;
        bool act = i < np / 2;
        if (act) {
            if (i == 0) { p = np - 1; q = r; }
            else {
                p = r + i; if (p >= np - 1) p -= np - 1;
                q = r - i; if (q < 0) q += np - 1;
            }
            if (p > q) { const int t = p; p = q; q = t; }
            act = q < n;
        }
        if (!act) { p = 0; q = 0; }                                         // inactive groups read column 0, write nothing
        const ColPtr<SH> ap(A + (size_t)p * lda), aq(A + (size_t)q * lda), nr(nrm2);
        const ColPtr<SH> vp(hasV ? V + (size_t)p * ldv : A), vq(hasV ? V + (size_t)q * ldv : A);
        double x[JR], y[JR], xv[JR], yv[JR];
#pragma unroll
        for (int u = 0; u < JR; ++u) {
            const int t = gl + G * u;
            const bool in = t < m;
            x[u] = in ? ap.ld(t) : 0.0; y[u] = in ? aq.ld(t) : 0.0;
        }
        const double al = nr.ld(p), be = nr.ld(q);
        if (hasV) {
#pragma unroll
            for (int u = 0; u < JR; ++u) {
                const int t = gl + G * u;
                const bool in = t < n;
                xv[u] = in ? vp.ld(t) : 0.0; yv[u] = in ? vq.ld(t) : 0.0;
            }
        }
        double ga0 = 0.0, ga1 = 0.0;
#pragma unroll
        for (int u = 0; u < JR; u += 2) { ga0 = fma(x[u], y[u], ga0); if (u + 1 < JR) ga1 = fma(x[u + 1], y[u + 1], ga1); }
        double ga = ga0 + ga1;
#pragma unroll
        for (int d = G / 2; d > 0; d >>= 1) ga += __shfl_xor_sync(0xffffffffu, ga, d);
        const bool rot = act && !(ga == 0.0 || ga * ga <= (DBL_EPSILON * DBL_EPSILON) * (al * be));
        if (!__any_sync(0xffffffffu, rot)) continue;
        // t = sign(d) g2 / (|d| + hypot(d, g2)), d = be - al, g2 = 2 ga;  c = 1/sqrt(1 + t^2), s = c t
        const double dd = be - al, g2 = 2.0 * ga;
        const double q2 = fma(dd, dd, g2 * g2);
        const double hh = q2 * fast_rsqrt(rot ? q2 : 1.0);
        const double tt = copysign(1.0, dd) * g2 * fast_rcp(rot ? fabs(dd) + hh : 1.0);
        const double c = fast_rsqrt(fma(tt, tt, 1.0)), sn = c * tt;
        double aln = fma(-tt, ga, al), ben = fma(tt, ga, be);
        const bool redo = rot && (!(aln > 1e-4 * al) || !(ben > 1e-4 * be));   // cancellation: recompute exactly
#pragma unroll
        for (int u = 0; u < JR; ++u) {
            const double xn = c * x[u] - sn * y[u], yn = sn * x[u] + c * y[u];
            x[u] = xn; y[u] = yn;
        }
        if (__any_sync(0xffffffffu, redo)) {
            double sa = 0.0, sb = 0.0, sa1 = 0.0, sb1 = 0.0;
#pragma unroll
            for (int u = 0; u < JR; u += 2) {
                sa = fma(x[u], x[u], sa); sb = fma(y[u], y[u], sb);
                if (u + 1 < JR) { sa1 = fma(x[u + 1], x[u + 1], sa1); sb1 = fma(y[u + 1], y[u + 1], sb1); }
            }
            sa += sa1; sb += sb1;
#pragma unroll
            for (int d = G / 2; d > 0; d >>= 1) {
                sa += __shfl_xor_sync(0xffffffffu, sa, d);
                sb += __shfl_xor_sync(0xffffffffu, sb, d);
            }
            if (redo) { aln = sa; ben = sb; }
        }
        if (rot) {
#pragma unroll
            for (int u = 0; u < JR; ++u) {
                const int t = gl + G * u;
                if (t < m) { ap.st(t, x[u]); aq.st(t, y[u]); }
            }
            if (hasV) {
#pragma unroll
                for (int u = 0; u < JR; ++u) {
                    const int t = gl + G * u;
                    if (t < n) { vp.st(t, c * xv[u] - sn * yv[u]); vq.st(t, sn * xv[u] + c * yv[u]); }
                }
            }
            if (gl == 0) { nr.st(p, aln); nr.st(q, ben); *s_flag = 1; }
        }
    }
}

// the whole Jacobi iteration for m <= G JR (one compiled body per shape class; see cta_jacobi for the contract)
template <int G, int JR, bool SH>
__device__ __noinline__ void cta_jacobi_sub(double* A, int lda, int m, int n, double* V, int ldv, int* s_flag, double* nrm2) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const int np = (n + 1) & ~1;
    for (int sweep = 0; sweep < JACOBI_MAX_SWEEPS; ++sweep) {
        if (tid == 0) *s_flag = 0;
        for (int c = warp; c < n; c += nwarps) {
            const double* ac = A + (size_t)c * lda;
            double acc = 0.0;
            for (int t = lane; t < m; t += 32) acc = fma(ac[t], ac[t], acc);
            acc = warp_sum(acc);
            if (lane == 0) nrm2[c] = acc;
        }
        __syncthreads();
        for (int r = 0; r < np - 1; ++r) {
            jacobi_round_sub<G, JR, SH>(A, lda, m, n, V, ldv, nrm2, np, r, s_flag);
            __syncthreads();
        }
        const int again = *s_flag;
        __syncthreads();
        if (!again) break;
    }
}

// One-sided Jacobi on A (m x n, m >= n, ld lda), accumulating the rotations into V (n x n, ld ldv, must be I on
// entry; V == nullptr: singular values only).  Round-robin tournament ordering; one warp per column pair.  On exit
// A = U diag(s), columns orthogonal.  nrm2 (n doubles, shared or global): squared column norms, recomputed at the
// start of every sweep and updated by the rotation formulas in between (al' = al - t ga, be' = be + t ga), with an
// explicit recomputation whenever the update cancels (so a pair costs one dot product instead of three).
__device__ __noinline__ void cta_jacobi(double* A, int lda, int m, int n, double* V, int ldv, int* s_flag, double* nrm2, bool sh = false) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const int np = (n + 1) & ~1;                 // players (padded to even)
    if (n < 2) return;
    if (m <= 128) {
        if (sh) {
            if (m <= 32) cta_jacobi_sub<8, 4, true>(A, lda, m, n, V, ldv, s_flag, nrm2);
            else if (m <= 64) cta_jacobi_sub<16, 4, true>(A, lda, m, n, V, ldv, s_flag, nrm2);
            else cta_jacobi_sub<16, 8, true>(A, lda, m, n, V, ldv, s_flag, nrm2);
        } else {
            if (m <= 32) cta_jacobi_sub<8, 4, false>(A, lda, m, n, V, ldv, s_flag, nrm2);
            else if (m <= 64) cta_jacobi_sub<16, 4, false>(A, lda, m, n, V, ldv, s_flag, nrm2);
            else cta_jacobi_sub<16, 8, false>(A, lda, m, n, V, ldv, s_flag, nrm2);
        }
        return;
    }
    for (int sweep = 0; sweep < JACOBI_MAX_SWEEPS; ++sweep) {
        if (tid == 0) *s_flag = 0;
        for (int c = warp; c < n; c += nwarps) {
            const double* ac = A + (size_t)c * lda;
            double acc = 0.0;
            for (int t = lane; t < m; t += 32) acc = fma(ac[t], ac[t], acc);
            acc = warp_sum(acc);
            if (lane == 0) nrm2[c] = acc;
        }
        __syncthreads();
        for (int r = 0; r < np - 1; ++r) {
            for (int i = warp; i < np / 2; i += nwarps) {
                int p, q;
                if (i == 0) { p = np - 1; q = r; }
                else {
                    p = r + i; if (p >= np - 1) p -= np - 1;
                    q = r - i; if (q < 0) q += np - 1;
                }
                if (p > q) { int t = p; p = q; q = t; }
                if (q >= n) continue;
                double* ap = A + (size_t)p * lda;
                double* aq = A + (size_t)q * lda;
                const double al = nrm2[p], be = nrm2[q];
                double ga = 0.0;
                for (int t = lane; t < m; t += 32) ga = fma(ap[t], aq[t], ga);
                ga = warp_sum(ga);
                // converged pair: |ga| <= eps sqrt(al be)
                if (ga == 0.0 || ga * ga <= (DBL_EPSILON * DBL_EPSILON) * (al * be)) continue;
                // t = sign(zeta) / (|zeta| + sqrt(1 + zeta^2)), zeta = (be - al) / (2 ga), without forming zeta:
                // t = sign(d) g2 / (|d| + hypot(d, g2)), d = be - al, g2 = 2 ga;  c = 1/sqrt(1 + t^2), s = c t
                const double dd = be - al, g2 = 2.0 * ga;
                const double q2 = fma(dd, dd, g2 * g2);
                const double hh = q2 * fast_rsqrt(q2);
                const double tt = copysign(1.0, dd) * g2 * fast_rcp(fabs(dd) + hh);
                const double c = fast_rsqrt(fma(tt, tt, 1.0)), s = c * tt;
                double aln = fma(-tt, ga, al), ben = fma(tt, ga, be);
                const bool redo = !(aln > 1e-4 * al) || !(ben > 1e-4 * be);      // cancellation: recompute exactly
                double sa = 0.0, sb = 0.0;
                for (int t = lane; t < m; t += 32) {
                    double x = ap[t], y = aq[t];
                    const double xn = c * x - s * y, yn = s * x + c * y;
                    ap[t] = xn; aq[t] = yn;
                    if (redo) { sa = fma(xn, xn, sa); sb = fma(yn, yn, sb); }
                }
                if (redo) {
#pragma unroll
                    for (int d = 16; d > 0; d >>= 1) {
                        sa += __shfl_xor_sync(0xffffffffu, sa, d);
                        sb += __shfl_xor_sync(0xffffffffu, sb, d);
                    }
                    aln = sa; ben = sb;
                }
                if (V != nullptr) {
                    double* vp = V + (size_t)p * ldv;
                    double* vq = V + (size_t)q * ldv;
                    for (int t = lane; t < n; t += 32) {
                        double x = vp[t], y = vq[t];
                        vp[t] = c * x - s * y; vq[t] = s * x + c * y;
                    }
                }
                if (lane == 0) { nrm2[p] = aln; nrm2[q] = ben; *s_flag = 1; }
            }
            __syncthreads();
        }
        int again = *s_flag;
        __syncthreads();
        if (!again) break;
    }
}

// Thin SVD of M (m x n, ld ldm): U (m x p), s (p, descending), V (n x p), p = min(m, n).
// work: max(m,n)*p + p*p + p doubles, iwork: p ints.  Columns of U for exactly-zero singular values are zero.
__device__ __noinline__ void cta_svd(const double* M, int ldm, int m, int n, double* U, int ldu, double* s, double* V, int ldv,
                        double* work, int* iwork, int* s_flag, double* sm = nullptr, int sm_doubles = 0,
                        bool vectors = true) {
    const int tid = threadIdx.x, nt = blockDim.x;
    const bool tr = m < n;
    const int T = tr ? n : m, p = tr ? m : n;
    // the Jacobi working set (T x p columns + p x p rotations) lives in shared memory when it fits: every round of
    // the sweep is a dependent read-modify-write of two columns per warp, i.e. pure latency
    const bool in_smem = sm != nullptr && (size_t)T * p + (size_t)p * p + (size_t)p <= (size_t)sm_doubles;
    double* A = in_smem ? sm : work;                 // T x p
    double* W = A + (size_t)T * p;                   // p x p
    double* sv = work + (size_t)T * p + (size_t)p * p; // p
    double* nrm2 = in_smem ? W + (size_t)p * p : sv;   // p (running squared column norms of the sweep)
    for (int e = tid; e < T * p; e += nt) {
        int t = e % T, c = e / T;
        A[e] = tr ? M[c + (size_t)t * ldm] : M[t + (size_t)c * ldm];
    }
    if (vectors) for (int e = tid; e < p * p; e += nt) W[e] = (e % p == e / p) ? 1.0 : 0.0;
    __syncthreads();
    cta_jacobi(A, T, T, p, vectors ? W : nullptr, p, s_flag, nrm2, in_smem);
    __syncthreads();
    {   // column norms, one warp per column
        const int lane = tid & 31, warp = tid >> 5, nwarps = nt >> 5;
        for (int c = warp; c < p; c += nwarps) {
            double acc = 0.0;
            for (int t = lane; t < T; t += 32) { double x = A[t + (size_t)c * T]; acc = fma(x, x, acc); }
            acc = warp_sum(acc);
            if (lane == 0) sv[c] = sqrt(acc);
        }
    }
    __syncthreads();
    for (int c = tid; c < p; c += nt) {   // rank by (value desc, index asc)
        int rk = 0; double v = sv[c];
        for (int o = 0; o < p; ++o) rk += (sv[o] > v) || (sv[o] == v && o < c);
        iwork[c] = rk;
    }
    __syncthreads();
    if (!vectors) {                                              // singular values only
        for (int c = tid; c < p; c += nt) s[iwork[c]] = sv[c];
        __syncthreads();
        return;
    }
    double* Ubig = tr ? V : U; int ldbig = tr ? ldv : ldu;       // receives the normalised A columns (T rows)
    double* Usml = tr ? U : V; int ldsml = tr ? ldu : ldv;       // receives the rotation columns (p rows)
    for (int e = tid; e < T * p; e += nt) {
        int t = e % T, c = e / T; double v = sv[c];
        Ubig[t + (size_t)iwork[c] * ldbig] = v > 0.0 ? A[e] / v : 0.0;
    }
    for (int e = tid; e < p * p; e += nt) {
        int t = e % p, c = e / p;
        Usml[t + (size_t)iwork[c] * ldsml] = W[e];
    }
    for (int c = tid; c < p; c += nt) s[iwork[c]] = sv[c];
    __syncthreads();
}

// C (m x n, ldc) = op(A) op(B) with explicit strides: A(i,t) = A[i*sai + t*sat], B(t,j) = B[t*sbt + j*sbj]
__device__ void cta_matmul(double* C, int ldc, int m, int n, int kk, const double* A, int sai, int sat,
                           const double* B, int sbt, int sbj) {
    for (int e = threadIdx.x; e < m * n; e += blockDim.x) {
        int i = e % m, j = e / m;
        double acc = 0.0;
        for (int t = 0; t < kk; ++t) acc = fma(A[(size_t)i * sai + (size_t)t * sat], B[(size_t)t * sbt + (size_t)j * sbj], acc);
        C[i + (size_t)j * ldc] = acc;
    }
    __syncthreads();
}

// Least squares X Y = B by Householder QR of W = [X | B] (rows x (xn + nb), column-major, ld ldw, overwritten):
// Y (xn x nb, ld ldy) = R^-1 (Q^T B)(0:xn, :).  Equals pinv(X) B when X has full column rank, which is how the
// pseudo-inverse of Alg. 1 lines 5-14 is applied when X is well conditioned ("\" in the paper);
// *cond_flag is set to 1 (the caller then takes the SVD pseudo-inverse, whose 1e-13 cut is reading Q4) unless
// kappa_F(R) = ||R||_F ||R^-1||_F <= 1e8, a rigorous bound (kappa_2 <= kappa_F <= n kappa_2): the diagonal of an
// unpivoted R alone can look harmless for a numerically singular X (Kahan's matrices).  R^-1 comes out of the same back
// substitution, from xn identity columns appended behind B: W needs room for xn + nb + xn columns.
template <int G, bool SH>
__device__ __noinline__ void cta_ls_householder_t(double* __restrict__ W, int ldw, int rows, int xn, int nb, double* __restrict__ Y, int ldy,
                                                  double* s_scal, int* cond_flag) {
    constexpr int GPW = 32 / G;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, gl = lane & (G - 1);
    const int ngroups = (blockDim.x >> 5) * GPW;
    const int ncol = xn + nb;
    for (int c = 0; c < xn; ++c) {
        const ColPtr<SH> xc(W + (size_t)c * ldw);
        if (warp == 0) {
            double sig = 0.0;
            for (int r = c + 1 + lane; r < rows; r += 32) { const double v = xc.ld(r); sig = fma(v, v, sig); }
            sig = warp_sum(sig);
            const double alpha = xc.ld(c);
            double beta, tau, inv;
            if (sig == 0.0) { beta = alpha; tau = 0.0; inv = 0.0; }
            else {
                const double nrm2 = fma(alpha, alpha, sig), aa = fabs(alpha);
                const double rs = fast_rsqrt(nrm2), mu = nrm2 * rs;          // |beta|
                beta = -copysign(mu, alpha);
                tau = fma(aa, rs, 1.0);                                      // (beta - alpha) / beta
                inv = copysign(fast_rcp(aa + mu), alpha);                    // 1 / (alpha - beta)
            }
            for (int r = c + 1 + lane; r < rows; r += 32) xc.st(r, xc.ld(r) * inv);   // v (unit diagonal implicit)
            if (lane == 0) { xc.st(c, beta); s_scal[0] = tau; }
        }
        __syncthreads();
        const double tau = s_scal[0];
        // one column per group of G lanes: 32 / G columns per warp instruction
        for (int j0 = c + 1 + warp * GPW; j0 < ncol; j0 += ngroups) {        // warp-uniform bounds
            const int j = j0 + lane / G;
            const bool act = j < ncol;
            const ColPtr<SH> aj(W + (size_t)(act ? j : c + 1) * ldw);
            double acc = 0.0;
            for (int r = c + 1 + gl; r < rows; r += G) acc = fma(xc.ld(r), aj.ld(r), acc);
#pragma unroll
            for (int d = G / 2; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
            if (act) {
                const double w = tau * (aj.ld(c) + acc);
                for (int r = c + 1 + gl; r < rows; r += G) aj.st(r, fma(-xc.ld(r), w, aj.ld(r)));
                if (gl == 0) aj.st(c, aj.ld(c) - w);
            }
        }
        __syncthreads();
    }
    if (tid == 0) {                      // quick reject: kappa_2 >= max|R_cc| / min|R_cc|
        double mx = 0.0, mn = INFINITY;
        for (int c = 0; c < xn; ++c) { double d = fabs(W[c + (size_t)c * ldw]); mx = fmax(mx, d); mn = fmin(mn, d); }
        *cond_flag = !(mn >= 1e-8 * mx && mx > 0.0);
    }
    for (int e = tid; e < xn * xn; e += blockDim.x) {                       // identity behind B
        const int i = e % xn, j = e / xn;
        W[i + (size_t)(xn + nb + j) * ldw] = (i == j) ? 1.0 : 0.0;
    }
    __syncthreads();
    if (*cond_flag) return;
    // back substitution R [Y | R^-1] = [(Q^T B)(0:xn, :) | I], column oriented and in place in W: step i fixes row i for
    // all right-hand sides, then removes its contribution from the rows above (xn steps of i * nbt independent updates)
    const int nbt = nb + xn;
    for (int i = xn - 1; i >= 0; --i) {
        const double rii = W[i + (size_t)i * ldw];
        for (int j = tid; j < nbt; j += blockDim.x) W[i + (size_t)(xn + j) * ldw] /= rii;
        __syncthreads();
        for (int e = tid; e < i * nbt; e += blockDim.x) {
            const int t = e % i, j = e / i;
            double* bj = W + (size_t)(xn + j) * ldw;
            bj[t] = fma(-W[t + (size_t)i * ldw], bj[i], bj[t]);
        }
        __syncthreads();
    }
    if (warp == 0) {                     // kappa_F(R)^2 = sum R^2 * sum (R^-1)^2 over the upper triangles, fixed order
        double r2 = 0.0, i2 = 0.0;
        for (int e = lane; e < xn * xn; e += 32) {
            const int i = e % xn, j = e / xn;
            if (i <= j) {
                const double a = W[i + (size_t)j * ldw], b = W[i + (size_t)(xn + nb + j) * ldw];
                r2 = fma(a, a, r2); i2 = fma(b, b, i2);
            }
        }
        r2 = warp_sum(r2); i2 = warp_sum(i2);
        if (lane == 0) *cond_flag = !(r2 * i2 <= 1e16);
    }
    __syncthreads();
    if (*cond_flag) return;
    for (int e = tid; e < xn * nb; e += blockDim.x) {
        const int i = e % xn, j = e / xn;
        Y[i + (size_t)j * ldy] = W[i + (size_t)(xn + j) * ldw];
    }
    __syncthreads();
}

// sh: W is in shared memory (LDS / STS instead of generic accesses)
__device__ void cta_ls_householder(double* W, int ldw, int rows, int xn, int nb, double* Y, int ldy,
                                   double* s_scal, int* cond_flag, bool sh) {
    if (sh) {
        if (rows <= 64) cta_ls_householder_t<8, true>(W, ldw, rows, xn, nb, Y, ldy, s_scal, cond_flag);
        else if (rows <= 128) cta_ls_householder_t<16, true>(W, ldw, rows, xn, nb, Y, ldy, s_scal, cond_flag);
        else cta_ls_householder_t<32, true>(W, ldw, rows, xn, nb, Y, ldy, s_scal, cond_flag);
    } else {
        if (rows <= 64) cta_ls_householder_t<8, false>(W, ldw, rows, xn, nb, Y, ldy, s_scal, cond_flag);
        else if (rows <= 128) cta_ls_householder_t<16, false>(W, ldw, rows, xn, nb, Y, ldy, s_scal, cond_flag);
        else cta_ls_householder_t<32, false>(W, ldw, rows, xn, nb, Y, ldy, s_scal, cond_flag);
    }
}

// ----------------------------------------------------------------------------------------------------------
// scross core.  QR factors: Qf (n x k) with R_C (k x k), Zf (n x l) with R_R (l x l).
__global__ void __launch_bounds__(CORE_NT)
scross_core_kernel(CoreArgs a) {
    __shared__ int s_flag;
    const int tid = threadIdx.x, nt = blockDim.x;
    const int k = a.k, l = a.l;
    const bool kle = k <= l;
    // X = Q(I,:) (l x k) if k <= l else Z(J,:) (k x l)
    const int xm = kle ? l : k, xn = kle ? k : l;      // xm >= xn
    const double* F = kle ? a.Q : a.Z; const int64_t ldf = kle ? a.ldq : a.ldz;
    const int32_t* idx = kle ? a.I : a.J;
    double* X = a.work;                                 // xm x xn
    double* Ux = X + (size_t)xm * xn;                   // xm x xn
    double* sx = Ux + (size_t)xm * xn;                  // xn
    double* Vx = sx + xn;                               // xn x xn
    double* P = Vx + (size_t)xn * xn;                   // xn x xm   (pseudo-inverse)
    double* Mc = P + (size_t)xn * xm;                   // k x l
    double* svdw = Mc + (size_t)k * l;                  // SVD scratch
    for (int e = tid; e < xm * xn; e += nt) {
        int r = e % xm, c = e / xm;
        X[e] = F[(int64_t)idx[r] + (int64_t)c * ldf];
    }
    for (int c = tid; c < k; c += nt) a.rC[c] = fabs(a.RC[c + (size_t)c * a.ldrc]);
    for (int c = tid; c < l; c += nt) a.rR[c] = fabs(a.RR[c + (size_t)c * a.ldrr]);
    __syncthreads();
    extern __shared__ __align__(16) double dyn_smem[];
    __shared__ double s_scal[2];
    __shared__ int s_cond;
    // Well-conditioned X (the usual case): M = X^+ B as the Householder least-squares solution of X Y = B, with
    // B = R_R^T (k <= l, M = Y) or B = R_C^T (k > l, M = Y^T).  Otherwise the SVD pseudo-inverse below.
    {
        const int ldw = xm | 1;                                       // odd leading dimension: no bank conflicts
        const bool fits = (size_t)ldw * (xn + xm + xn) <= (size_t)a.smem_doubles;
        double* Wls = fits ? dyn_smem : svdw;                         // svdw has room only when core_work is sized for it
        const double* Ro = kle ? a.RR : a.RC; const int64_t ldo = kle ? a.ldrr : a.ldrc;
        if (fits) {
            for (int e = tid; e < xm * xn; e += nt) Wls[(e % xm) + (size_t)(e / xm) * ldw] = X[e];
            for (int e = tid; e < xm * xm; e += nt) {
                int i = e % xm, j = e / xm;                            // B(i,j) = Rother(j,i)
                Wls[i + (size_t)(xn + j) * ldw] = Ro[j + (size_t)i * ldo];
            }
            __syncthreads();
            cta_ls_householder(Wls, ldw, xm, xn, xm, P, xn, s_scal, &s_cond, fits);   // Y (xn x xm) into P's storage
        } else {
            if (tid == 0) s_cond = 1;
            __syncthreads();
        }
    }
    if (!s_cond) {
        // Y = P (xn x xm).  k <= l: M = Y (k x l);  k > l: M = Y^T
        for (int e = tid; e < k * l; e += nt) {
            int i = e % k, j = e / k;
            Mc[e] = kle ? P[i + (size_t)j * xn] : P[j + (size_t)i * xn];
        }
        __syncthreads();
    } else {
    cta_svd(X, xm, xm, xn, Ux, xm, sx, Vx, xn, svdw, a.iwork, &s_flag, dyn_smem, a.smem_doubles);
    // P = Vx diag(1/sx) Ux^T over the kept singular values (relative cut, reading Q4)
    {
        const double cut = a.pinv_rcond * sx[0];
        for (int e = tid; e < xn * xm; e += nt) {
            int i = e % xn, j = e / xn;
            double acc = 0.0;
            for (int t = 0; t < xn; ++t) {
                double sv = sx[t];
                if (sv > cut) acc = fma(Vx[i + (size_t)t * xn] / sv, Ux[j + (size_t)t * xm], acc);
            }
            P[e] = acc;
        }
        __syncthreads();
    }
    if (kle) {
        // M = P (k x l) * R_R^T (l x l):  M(i,j) = sum_t P(i,t) R_R(j,t)
        cta_matmul(Mc, k, k, l, l, P, 1, k, a.RR, (int)a.ldrr, 1);
    } else {
        // M = R_C (k x k) * P^T (k x l): M(i,j) = sum_t R_C(i,t) P(j,t),  P is l x k
        cta_matmul(Mc, k, k, l, k, a.RC, 1, (int)a.ldrc, P, l, 1);
    }
    }
    const int p = k < l ? k : l;
    cta_svd(Mc, k, k, l, a.Uc, k, a.S, a.Vc, l, svdw, a.iwork, &s_flag, dyn_smem, a.smem_doubles);
    if (tid == 0) {
        double s1 = a.S[0];
        int rank = 0;
        for (int c = 0; c < p; ++c) rank += a.S[c] > a.rank_rcond * s1;
        if (rank < 1) rank = 1;
        a.scal_i[0] = rank;
        a.scal_d[0] = a.S[p - 1];                       // smin_full (reading Q11)
    }
}

// eta_side = 1 / sigma_min(F(idx,:)), F tall n x r, idx: nidx indices.  blockIdx.x selects the side (U/I or V/J).
__global__ void __launch_bounds__(CORE_NT)
eta_kernel(EtaArgs a) {
    __shared__ int s_flag;
    const int side = blockIdx.x;
    const int tid = threadIdx.x, nt = blockDim.x;
    const double* F = side == 0 ? a.U : a.V; const int64_t ldf = side == 0 ? a.ldu : a.ldv;
    const int32_t* idx = side == 0 ? a.I : a.J; const int nidx = side == 0 ? a.nI : a.nJ;
    const double* Cf = side == 0 ? a.CU : a.CV; const int kf = side == 0 ? a.kU : a.kV; const int64_t ldcf = side == 0 ? a.ldcu : a.ldcv;
    const int r = a.r;
    double* out = a.eta + side;
    if (nidx == 0 || r == 0) { if (tid == 0) *out = INFINITY; return; }
    double* work = a.work + (size_t)side * a.work_stride;
    int* iwork = a.iwork + (size_t)side * a.iwork_stride;
    const int p = nidx < r ? nidx : r;
    double* X = work;                                    // nidx x r
    double* Ux = X + (size_t)nidx * r;                   // nidx x p
    double* sx = Ux + (size_t)nidx * p;                  // p
    double* Vx = sx + p;                                 // r x p
    double* svdw = Vx + (size_t)r * p;
    for (int e = tid; e < nidx * r; e += nt) {
        int i = e % nidx, c = e / nidx;
        if (Cf == nullptr) X[e] = F[(int64_t)idx[i] + (int64_t)c * ldf];
        else {                                           // row idx[i] of (QF CF)(:, c)
            double acc = 0.0;
            for (int t = 0; t < kf; ++t) acc = fma(F[(int64_t)idx[i] + (int64_t)t * ldf], Cf[t + (int64_t)c * ldcf], acc);
            X[e] = acc;
        }
    }
    __syncthreads();
    extern __shared__ __align__(16) double dyn_smem[];
    cta_svd(X, nidx, nidx, r, Ux, nidx, sx, Vx, r, svdw, iwork, &s_flag, dyn_smem, a.smem_doubles, false);
    if (tid == 0) { double sm = sx[p - 1]; *out = sm == 0.0 ? INFINITY : 1.0 / sm; }
}

// rho^2 = ||S_k - A S' B^T||_F^2 + ||A S' E_V^T||_F^2 + ||E_U S' B^T||_F^2 + ||E_U S' E_V^T||_F^2 with
// U_{k-1} = U_k A + E_U, V_{k-1} = V_k B + E_V (A = U_k^T U_{k-1}, B = V_k^T V_{k-1}, GU = E_U^T E_U, GV = E_V^T E_V).
// All four terms are non-negative (no Gram expansion of the difference; reading Q13).
__global__ void __launch_bounds__(CORE_NT)
rho_kernel(RhoArgs a) {
    __shared__ double red[32];
    __shared__ unsigned s_last;
    // the (independent) output elements of the three sums are spread over the grid; per-CTA partial sums are added by the
    // last CTA to arrive, in block order (deterministic)
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nt = gridDim.x * blockDim.x;
    const int r = a.r, rp = a.rp;
    double acc = 0.0;
    // T1 = A diag(Sp)  (r x rp);  term1: sum_{i,j} (Sk(i) delta_ij - sum_t T1(i,t) B(j,t))^2
    for (int e = tid; e < r * r; e += nt) {
        int i = e % r, j = e / r;
        double v = (i == j) ? a.Sk[i] : 0.0;
#pragma unroll 4
        for (int t = 0; t < rp; ++t) v = fma(-a.A[i + (size_t)t * r] * a.Sp[t], a.B[j + (size_t)t * r], v);
        acc = fma(v, v, acc);
    }
    // term2: ||A S' E_V^T||_F^2 = sum_i sum_{t,u} A(i,t) Sp(t) GV(t,u) Sp(u) A(i,u);  term3 likewise with B, GU.
    // One (side, i, t) per thread step; the total is non-negative up to rounding (clamped with the sum below).
    for (int e = tid; e < 2 * r * rp; e += nt) {
        const int side = e / (r * rp), rem = e % (r * rp), i = rem % r, t = rem / r;
        const double* Mx = side == 0 ? a.A : a.B; const double* G = side == 0 ? a.GV : a.GU;
        double w = 0.0;
#pragma unroll 4
        for (int u = 0; u < rp; ++u) w = fma(G[t + (size_t)u * rp], a.Sp[u] * Mx[i + (size_t)u * r], w);
        acc = fma(Mx[i + (size_t)t * r] * a.Sp[t], w, acc);
    }
    // term4: ||E_U S' E_V^T||_F^2 = sum_{t,u} GU(t,u) Sp(t) Sp(u) GV(t,u)
    for (int e = tid; e < rp * rp; e += nt) {
        int t = e % rp, u = e / rp;
        acc = fma(a.GU[e] * a.Sp[t] * a.Sp[u], a.GV[e], acc);
    }
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < (int)blockDim.x / 32; ++w) t += red[w];
        a.partial[blockIdx.x] = t;
        __threadfence();
        s_last = (atomicAdd(a.ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (!s_last || threadIdx.x != 0) return;
    __threadfence();
    double t = 0.0;
    for (int b = 0; b < (int)gridDim.x; ++b) t += __ldcg(a.partial + b);
    double sn = 0.0;
    for (int c = 0; c < r; ++c) sn = fma(a.Sk[c], a.Sk[c], sn);
    a.out[0] = sqrt(t > 0.0 ? t : 0.0);
    a.out[1] = sqrt(sn);
    *a.ticket = 0u;                                   // ready for the next launch
}

struct RhoNestedArgs { int r, rp, use_smem; RhoNestedSide s0, s1; };

// use_smem: Y, M, A and compact copies of Uc, Ucp live in dynamic shared memory (small cores); otherwise Y, M in the
// global scratch and the factors are read in place.
// dot product with four independent partial sums (the single chain is latency-bound: one DFMA per ~8 cycles)
template <typename FA, typename FB>
__device__ __forceinline__ double dot4(int len, FA fa, FB fb) {
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int c = 0;
    for (; c + 4 <= len; c += 4) {
        a0 = fma(fa(c), fb(c), a0); a1 = fma(fa(c + 1), fb(c + 1), a1);
        a2 = fma(fa(c + 2), fb(c + 2), a2); a3 = fma(fa(c + 3), fb(c + 3), a3);
    }
    for (; c < len; ++c) a0 = fma(fa(c), fb(c), a0);
    return (a0 + a1) + (a2 + a3);
}

template <bool USE_SMEM>
__global__ void __launch_bounds__(CORE_NT)
rho_nested_kernel(RhoNestedArgs a) {
    extern __shared__ __align__(16) double dyn_smem[];
    // field-wise select (a dynamically indexed parameter array would live in local memory)
    const RhoNestedSide s = blockIdx.x == 0 ? a.s0 : a.s1;
    const int tid = threadIdx.x, nt = blockDim.x, r = a.r, rp = a.rp;
    const int nrest = s.kkp - s.k0;
    double* Y = s.scratch; double* M = s.scratch + (size_t)s.kk * rp;
    double* Aw = s.A;
    const double* Uc = s.Uc; int ldc = s.ldc;
    const double* Ucp = s.Ucp; int ldcp = s.ldcp;
    if (USE_SMEM) {
        Y = dyn_smem; M = Y + (size_t)s.kk * rp; Aw = M + (size_t)s.kk * rp;
        double* uc = Aw + (size_t)r * rp; double* ucp = uc + (size_t)s.kk * r;
        for (int e = tid; e < s.kk * r; e += nt) uc[e] = s.Uc[(e % s.kk) + (size_t)(e / s.kk) * s.ldc];
        for (int e = tid; e < s.kkp * rp; e += nt) ucp[e] = s.Ucp[(e % s.kkp) + (size_t)(e / s.kkp) * s.ldcp];
        Uc = uc; ldc = s.kk; Ucp = ucp; ldcp = s.kkp;
        __syncthreads();
    }
    const double* Ucr = Ucp + s.k0;                              // Uc_rest(q, t) = Ucr[q + t * ldcp]
    for (int e = tid; e < s.kk * rp; e += nt) {                  // Y = [Uc_pref; 0] + T Uc_rest
        int c = e % s.kk, t = e / s.kk;
        double acc = c < s.k0 ? Ucp[c + (size_t)t * ldcp] : 0.0;
        for (int q = 0; q < nrest; ++q) acc = fma(s.T[c + (size_t)q * s.kk], Ucr[q + (size_t)t * ldcp], acc);
        Y[e] = acc;
    }
    __syncthreads();
    for (int e = tid; e < r * rp; e += nt) {                     // A = Uc^T Y
        int i = e % r, t = e / r;
        const double* ua = Uc + (size_t)i * ldc; const double* ya = Y + (size_t)t * s.kk;
        Aw[e] = dot4(s.kk, [&](int c) { return ua[c]; }, [&](int c) { return ya[c]; });
    }
    __syncthreads();
    for (int e = tid; e < s.kk * rp; e += nt) {                  // M = Y - Uc A
        int c = e % s.kk, t = e / s.kk;
        const double* ua = Uc + c; const double* aa = Aw + (size_t)t * r;
        M[e] = Y[e] - dot4(r, [&](int i) { return ua[(size_t)i * ldc]; }, [&](int i) { return aa[i]; });
    }
    if (USE_SMEM) for (int e = tid; e < r * rp; e += nt) s.A[e] = Aw[e];
    __syncthreads();
    for (int e = tid; e < rp * rp; e += nt) {                    // G = M^T M + Uc_rest^T (P^T P) Uc_rest
        int t = e % rp, u = e / rp;
        const double* mt = M + (size_t)t * s.kk; const double* mu = M + (size_t)u * s.kk;
        double acc = dot4(s.kk, [&](int c) { return mt[c]; }, [&](int c) { return mu[c]; });
        for (int q = 0; q < nrest; ++q) {
            double w = 0.0;
            for (int q2 = 0; q2 < nrest; ++q2) w = fma(s.Gp[q + (size_t)q2 * nrest], Ucr[q2 + (size_t)u * ldcp], w);
            acc = fma(Ucr[q + (size_t)t * ldcp], w, acc);
        }
        s.G[e] = acc;
    }
}

__global__ void snorm_kernel(int r, const double* S, double* out) {
    if (threadIdx.x == 0) {
        double sn = 0.0;
        for (int c = 0; c < r; ++c) sn = fma(S[c], S[c], sn);
        out[0] = sqrt(sn); out[1] = sqrt(sn);
    }
}

__global__ void colmask_kernel(int k, const double* R, int64_t ldr, double rcond, unsigned char* mask) {
    __shared__ double mx;
    if (threadIdx.x == 0) {
        double m = 0.0;
        for (int c = 0; c < k; ++c) m = fmax(m, fabs(R[c + (size_t)c * ldr]));
        mx = m;
    }
    __syncthreads();
    for (int c = threadIdx.x; c < k; c += blockDim.x) mask[c] = (mx > 0.0 && fabs(R[c + (size_t)c * ldr]) >= rcond * mx) ? 1 : 0;
}

}  // namespace

size_t core_work_doubles(int k, int l) {
    size_t xm = k > l ? k : l, xn = k > l ? l : k;
    size_t d = 0;
    d += xm * xn * 2 + xn + xn * xn + xn * xm + (size_t)k * l;
    d += xm * xn + xn * xn + xn + 64;       // SVD scratch (T*p + p*p + p)
    return d;
}

static size_t jacobi_smem_bytes(const lrp_ctx* ctx, int T, int p) {
    size_t need = ((size_t)T * p + (size_t)p * p + (size_t)p) * sizeof(double);
    size_t cap = (size_t)ctx->smem_optin > 2048 ? (size_t)ctx->smem_optin - 2048 : 0;
    return need <= cap ? need : 0;                 // 0: stay in global memory
}

// Dynamic shared-memory opt-in of the one-CTA kernels: once per context (lrp_create), to everything the device allows.
template <typename F> static int core_optin(lrp_ctx* ctx, F fn) {
    cudaFuncAttributes fa;
    LRP_CUDA(ctx, cudaFuncGetAttributes(&fa, fn));
    const int v = ctx->smem_optin - (int)fa.sharedSizeBytes;
    if (v > 48 * 1024) LRP_CUDA(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, v));
    return LRP_OK;
}
int core_init(lrp_ctx* ctx) {
    LRP_TRY(core_optin(ctx, scross_core_kernel));
    LRP_TRY(core_optin(ctx, eta_kernel));
    LRP_TRY(core_optin(ctx, rho_nested_kernel<true>));
    return LRP_OK;
}

int scross_core(lrp_ctx* ctx, const CoreArgs& a0) {
    CoreArgs a = a0;
    const int T = a.k > a.l ? a.k : a.l, p = a.k > a.l ? a.l : a.k;
    size_t smem = jacobi_smem_bytes(ctx, T, p);
    {
        size_t ls = (size_t)(T | 1) * (size_t)(p + T + p) * sizeof(double);      // [X | B | I] of the least squares
        size_t cap = (size_t)ctx->smem_optin > 2048 ? (size_t)ctx->smem_optin - 2048 : 0;
        if (ls > smem && ls <= cap) smem = ls;
    }
    a.smem_doubles = (int)(smem / sizeof(double));
    LRP_PROF(ctx, K_CORE, 0, 0);
    scross_core_kernel<<<1, CORE_NT, smem, ctx->stream>>>(a);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

size_t eta_work_doubles(int nmax, int r) {
    size_t p = nmax < r ? nmax : r, T = nmax > r ? nmax : r;
    return (size_t)nmax * r + (size_t)nmax * p + p + (size_t)r * p + T * p + p * p + p + 64;
}

int eta_pair(lrp_ctx* ctx, const EtaArgs& a0) {
    EtaArgs a = a0;
    const int nmax = a.nI > a.nJ ? a.nI : a.nJ;
    const int T = nmax > a.r ? nmax : a.r, p = nmax > a.r ? a.r : nmax;
    const size_t smem = jacobi_smem_bytes(ctx, T, p > 0 ? p : 1);
    a.smem_doubles = (int)(smem / sizeof(double));
    LRP_PROF(ctx, K_ETA, 0, 0);
    eta_kernel<<<2, CORE_NT, smem, ctx->stream>>>(a);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

int rho_small(lrp_ctx* ctx, const RhoArgs& a) {
    LRP_PROF(ctx, K_RHO, 0, 0);
    if (a.rp == 0) snorm_kernel<<<1, 32, 0, ctx->stream>>>(a.r, a.Sk, a.out);
    else {
        int work = a.r * a.r + 2 * a.r * a.rp + a.rp * a.rp;
        int grid = (work + 255) / 256; if (grid > RHO_MAX_GRID) grid = RHO_MAX_GRID; if (grid < 1) grid = 1;
        LRP_CUDA(ctx, cudaMemsetAsync(a.ticket, 0, sizeof(unsigned), ctx->stream));
        rho_kernel<<<grid, 256, 0, ctx->stream>>>(a);
    }
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

int rho_nested_prep(lrp_ctx* ctx, int r, int rp, const RhoNestedSide& u, const RhoNestedSide& v) {
    RhoNestedArgs a{};
    a.r = r; a.rp = rp; a.s0 = u; a.s1 = v;
    auto need = [&](const RhoNestedSide& s) { return sizeof(double) * ((size_t)2 * s.kk * rp + (size_t)r * rp + (size_t)s.kk * r + (size_t)s.kkp * rp); };
    size_t smem = need(u) > need(v) ? need(u) : need(v);
    a.use_smem = smem <= (size_t)200 * 1024 ? 1 : 0;
    if (!a.use_smem) smem = 0;
    LRP_PROF(ctx, K_RHO, 0, 0);
    if (a.use_smem) rho_nested_kernel<true><<<2, CORE_NT, smem, ctx->stream>>>(a);
    else rho_nested_kernel<false><<<2, CORE_NT, 0, ctx->stream>>>(a);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

int leverage_colmask(lrp_ctx* ctx, int k, const double* R, int64_t ldr, double rcond, unsigned char* mask) {
    LRP_PROF(ctx, K_COLMASK, 0, 0);
    colmask_kernel<<<1, 128, 0, ctx->stream>>>(k, R, ldr, rcond, mask);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}
