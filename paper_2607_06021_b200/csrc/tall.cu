// tall.cu -- streaming kernels over "tall" (n x small, column-major) fp64 matrices:
//   tall_gemm    : Out(n x m) = epilogue( A(n x k) B(k x m) )     fiber sampling (eq. (4)),
//                  factor rebuild U = Q Uc (Alg. 1 lines 9/14), Gram-Schmidt update P -= Q S
//   tall_gemm_t  : S(k x m) = A(n x k)^T B(n x m)                  projections / Gram blocks (reduction over n)
//   row norms, gathers, low-rank entry evaluation.
// Plain DFMA register tiling: on sm_100a the fp64 tensor pipe (DMMA) has the same peak as the FMA pipe and
// these contractions sit at or below the fp64/HBM balance point.
#include "common.cuh"
#include "tall.cuh"
#include <math.h>

namespace {

constexpr int GT_THREADS = 128, GT_RT = 2, GT_CT = 32;
constexpr int GT_ROWS = GT_THREADS * GT_RT;

// d_i = lambda_{i+1} / h^2 = 4 N^2 sin^2(pi (i+1) / (2N))   (PAPER.md:200 as 4 sin^2(theta/2), reading Q1)
__device__ __forceinline__ double eig_d(int64_t i, double invN, double fourN2) {
    double s = sinpi(0.5 * (double)(i + 1) * invN);
    return fourN2 * s * s;
}

// Out(i, c) for a 256-row slab per CTA; B slice (k x GT_CT) staged in shared memory per column chunk.
__global__ void __launch_bounds__(GT_THREADS)
tall_gemm_kernel(TallGemmArgs p) {
    extern __shared__ __align__(16) double smem[];
    double* Bs = smem;                         // [k][GT_CT]
    double* dcol = smem + (size_t)p.k * GT_CT; // [GT_CT] eigenvalue of the sampled column (sampler epilogue)
    const int tid = threadIdx.x;
    const int64_t row0 = (int64_t)blockIdx.x * GT_ROWS + tid;
    const double invN = 1.0 / (double)(p.n + 1);
    const double fourN2 = 4.0 * (double)(p.n + 1) * (double)(p.n + 1);
    bool valid[GT_RT]; int64_t rows[GT_RT]; double drow[GT_RT]; double nrm[GT_RT];
#pragma unroll
    for (int rr = 0; rr < GT_RT; ++rr) {
        rows[rr] = row0 + (int64_t)rr * GT_THREADS;
        valid[rr] = rows[rr] < p.n;
        drow[rr] = (p.mode == TG_SAMPLE && valid[rr]) ? eig_d(rows[rr], invN, fourN2) : 0.0;
        nrm[rr] = 0.0;
    }
    for (int c0 = 0; c0 < p.m; c0 += GT_CT) {
        const int cw = (p.m - c0) < GT_CT ? (p.m - c0) : GT_CT;
        __syncthreads();
        // stage B(:, c0:c0+cw): B(t, c) = Bsrc[t*ldb_t + c*ldb_c] (* scale_t[t]) ; gathered rows for the sampler
        for (int e = tid; e < p.k * GT_CT; e += GT_THREADS) {
            int t = e / GT_CT, c = e % GT_CT;
            double v = 0.0;
            if (c < cw) {
                if (p.mode == TG_SAMPLE) v = p.B[(int64_t)p.idx[c0 + c] + (int64_t)t * p.ldb] * p.scale_t[t];
                else v = p.B[(int64_t)t + (int64_t)(c0 + c) * p.ldb];
            }
            Bs[t * GT_CT + c] = v;
        }
        if (p.mode == TG_SAMPLE)
            for (int c = tid; c < GT_CT; c += GT_THREADS) dcol[c] = c < cw ? eig_d(p.idx[c0 + c], invN, fourN2) : 1.0;
        __syncthreads();
        double acc[GT_RT][GT_CT];
#pragma unroll
        for (int rr = 0; rr < GT_RT; ++rr)
#pragma unroll
            for (int c = 0; c < GT_CT; ++c) acc[rr][c] = 0.0;
        const double* a0 = p.A + (valid[0] ? rows[0] : 0);
        const double* a1 = p.A + (valid[1] ? rows[1] : 0);
        int t = 0;
        for (; t + 4 <= p.k; t += 4) {
            double av[4][GT_RT];
#pragma unroll
            for (int u = 0; u < 4; ++u) { av[u][0] = a0[(int64_t)(t + u) * p.lda]; av[u][1] = a1[(int64_t)(t + u) * p.lda]; }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const double2* b2 = (const double2*)(Bs + (t + u) * GT_CT);
#pragma unroll
                for (int c = 0; c < GT_CT / 2; ++c) {
                    double2 b = b2[c];
                    acc[0][2 * c] = fma(av[u][0], b.x, acc[0][2 * c]);
                    acc[0][2 * c + 1] = fma(av[u][0], b.y, acc[0][2 * c + 1]);
                    acc[1][2 * c] = fma(av[u][1], b.x, acc[1][2 * c]);
                    acc[1][2 * c + 1] = fma(av[u][1], b.y, acc[1][2 * c + 1]);
                }
            }
        }
        for (; t < p.k; ++t) {
            double x0 = a0[(int64_t)t * p.lda], x1 = a1[(int64_t)t * p.lda];
            const double2* b2 = (const double2*)(Bs + t * GT_CT);
#pragma unroll
            for (int c = 0; c < GT_CT / 2; ++c) {
                double2 b = b2[c];
                acc[0][2 * c] = fma(x0, b.x, acc[0][2 * c]);
                acc[0][2 * c + 1] = fma(x0, b.y, acc[0][2 * c + 1]);
                acc[1][2 * c] = fma(x1, b.x, acc[1][2 * c]);
                acc[1][2 * c + 1] = fma(x1, b.y, acc[1][2 * c + 1]);
            }
        }
        // epilogue
#pragma unroll
        for (int rr = 0; rr < GT_RT; ++rr) {
            if (!valid[rr]) continue;
#pragma unroll
            for (int c = 0; c < GT_CT; ++c) {
                if (c < cw) {
                    double v = acc[rr][c];
                    double* o = p.Out + rows[rr] + (int64_t)(c0 + c) * p.ldo;
                    if (p.mode == TG_SAMPLE) v = v / (drow[rr] + dcol[c]);
                    else if (p.mode == TG_SUBTRACT) v = p.Cin[rows[rr] + (int64_t)(c0 + c) * p.ldc] - v;
                    *o = v;
                    nrm[rr] = fma(v, v, nrm[rr]);
                }
            }
        }
    }
    if (p.rownorm2)
#pragma unroll
        for (int rr = 0; rr < GT_RT; ++rr)
            if (valid[rr]) p.rownorm2[rows[rr]] = nrm[rr];
}

// ---- S = A^T B, reduction over n --------------------------------------------------------------------------
constexpr int TT_THREADS = 256, TT_TA = 8, TT_TB = 4, TT_ROWS = 16;
// one CTA: rows [blockIdx.x * rows_per_cta, ...), output tile (a0..a0+TA*16) x (b0..b0+TB*16): 128 x 64 per CTA
constexpr int TT_KA = 128, TT_MB = 64;

__global__ void __launch_bounds__(TT_THREADS)
tall_gemm_t_kernel(const double* __restrict__ A, int64_t lda, int k, const double* __restrict__ B, int64_t ldb, int m,
                   int64_t n, int64_t rows_per_cta, double* __restrict__ partial) {
    __shared__ double As[TT_KA][TT_ROWS + 1];
    __shared__ double Bsm[TT_MB][TT_ROWS + 1];
    const int tid = threadIdx.x;
    const int ta = tid % 16, tb = tid / 16;                 // thread tile: a = ta + 16*i (i<8), b = tb + 16*j (j<4)
    const int a_base = blockIdx.y * TT_KA, b_base = blockIdx.z * TT_MB;
    const int64_t r_begin = (int64_t)blockIdx.x * rows_per_cta;
    int64_t r_end = r_begin + rows_per_cta; if (r_end > n) r_end = n;
    double acc[TT_TA][TT_TB];
#pragma unroll
    for (int i = 0; i < TT_TA; ++i)
#pragma unroll
        for (int j = 0; j < TT_TB; ++j) acc[i][j] = 0.0;
    const int ka = (k - a_base) < TT_KA ? (k - a_base) : TT_KA;
    const int mb = (m - b_base) < TT_MB ? (m - b_base) : TT_MB;
    for (int64_t r0 = r_begin; r0 < r_end; r0 += TT_ROWS) {
        __syncthreads();
        for (int e = tid; e < TT_KA * TT_ROWS; e += TT_THREADS) {
            int rr = e % TT_ROWS, a = e / TT_ROWS;
            int64_t r = r0 + rr;
            As[a][rr] = (a < ka && r < r_end) ? A[r + (int64_t)(a_base + a) * lda] : 0.0;
        }
        for (int e = tid; e < TT_MB * TT_ROWS; e += TT_THREADS) {
            int rr = e % TT_ROWS, b = e / TT_ROWS;
            int64_t r = r0 + rr;
            Bsm[b][rr] = (b < mb && r < r_end) ? B[r + (int64_t)(b_base + b) * ldb] : 0.0;
        }
        __syncthreads();
#pragma unroll 4
        for (int rr = 0; rr < TT_ROWS; ++rr) {
            double av[TT_TA], bv[TT_TB];
#pragma unroll
            for (int i = 0; i < TT_TA; ++i) av[i] = As[ta + 16 * i][rr];
#pragma unroll
            for (int j = 0; j < TT_TB; ++j) bv[j] = Bsm[tb + 16 * j][rr];
#pragma unroll
            for (int i = 0; i < TT_TA; ++i)
#pragma unroll
                for (int j = 0; j < TT_TB; ++j) acc[i][j] = fma(av[i], bv[j], acc[i][j]);
        }
    }
    double* P = partial + (int64_t)blockIdx.x * k * m;
#pragma unroll
    for (int i = 0; i < TT_TA; ++i)
#pragma unroll
        for (int j = 0; j < TT_TB; ++j) {
            int a = a_base + ta + 16 * i, b = b_base + tb + 16 * j;
            if (a < k && b < m) P[a + (int64_t)b * k] = acc[i][j];
        }
}

// S(a,b) = alpha * sum_blk partial[blk](a,b) (+ S(a,b) if accumulate), fixed summation order (deterministic)
__global__ void reduce_partials_kernel(const double* __restrict__ partial, int nblk, int k, int m,
                                       double* __restrict__ S, int64_t lds, int accumulate) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= k * m) return;
    double s = 0.0;
    for (int b = 0; b < nblk; ++b) s += partial[(int64_t)b * k * m + e];
    int a = e % k, c = e / k;
    double* o = S + a + (int64_t)c * lds;
    *o = accumulate ? (*o + s) : s;
}

__global__ void rownorm2_kernel(int64_t n, int k, const double* __restrict__ A, int64_t lda,
                                const unsigned char* __restrict__ colmask, double* __restrict__ out) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double s = 0.0;
    for (int c = 0; c < k; ++c) {
        if (colmask && !colmask[c]) continue;
        double v = A[i + (int64_t)c * lda];
        s = fma(v, v, s);
    }
    out[i] = s;
}

// Out(r, c) = A(idx[r], c),  r < nidx, c < k   (small dense gather, column-major, ld = ldo)
__global__ void gather_rows_kernel(const double* __restrict__ A, int64_t lda, int k, const int32_t* __restrict__ idx,
                                   int nidx, double* __restrict__ Out, int ldo) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nidx * k) return;
    int r = e % nidx, c = e / nidx;
    Out[r + (int64_t)c * ldo] = A[(int64_t)idx[r] + (int64_t)c * lda];
}

__global__ void lowrank_entries_kernel(int r, const double* __restrict__ U, int64_t ldu, const double* __restrict__ S,
                                       const double* __restrict__ V, int64_t ldv, const int64_t* __restrict__ rows,
                                       const int64_t* __restrict__ cols, int64_t count, double* __restrict__ out) {
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= count) return;
    int64_t i = rows[t], j = cols[t];
    double acc = 0.0;
    for (int c = 0; c < r; ++c) acc = fma(U[i + (int64_t)c * ldu] * S[c], V[j + (int64_t)c * ldv], acc);
    out[t] = acc;
}

__global__ void copy_tall_kernel(int64_t n, int k, const double* __restrict__ A, int64_t lda, double* __restrict__ B, int64_t ldb) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    for (int c = blockIdx.y; c < k; c += gridDim.y) B[i + (int64_t)c * ldb] = A[i + (int64_t)c * lda];
}

}  // namespace

int tall_gemm(lrp_ctx* ctx, const TallGemmArgs& p) {
    if (p.n <= 0 || p.m <= 0) return LRP_OK;
    size_t smem = sizeof(double) * ((size_t)(p.k > 0 ? p.k : 1) * GT_CT + GT_CT);
    if (smem > 48 * 1024) {
        if (smem > (size_t)ctx->smem_optin) return LRP_ERR_BADARG;
        LRP_CUDA(ctx, cudaFuncSetAttribute(tall_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    }
    int64_t grid = (p.n + GT_ROWS - 1) / GT_ROWS;
    LRP_PROF(ctx, p.mode == TG_SAMPLE ? K_GEMM_SAMPLE : (p.mode == TG_SUBTRACT ? K_GEMM_SUBTRACT : K_GEMM_PLAIN),
             8.0 * p.n * (p.k + p.m + (p.mode == TG_SUBTRACT ? p.m : 0)), 2.0 * p.n * p.k * p.m);
    tall_gemm_kernel<<<(unsigned)grid, GT_THREADS, smem, ctx->stream>>>(p);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

int tall_gemm_t_nblk(const lrp_ctx* ctx, int64_t n) {
    (void)ctx;
    int64_t want = 148 * 4;                    // B200: 148 SMs; fixed so that workspace sizes need no device query
    int64_t by_rows = (n + 255) / 256;
    int64_t nb = want < by_rows ? want : by_rows;
    return (int)(nb < 1 ? 1 : nb);
}

size_t tall_gemm_t_ws_doubles(const lrp_ctx* ctx, int64_t n, int k, int m) {
    return (size_t)tall_gemm_t_nblk(ctx, n) * k * m;
}

int tall_gemm_t(lrp_ctx* ctx, int64_t n, const double* A, int64_t lda, int k, const double* B, int64_t ldb, int m,
                double* S, int64_t lds, int accumulate, double* partial_ws) {
    if (k <= 0 || m <= 0) return LRP_OK;
    int nblk = tall_gemm_t_nblk(ctx, n);
    int64_t rows_per = (n + nblk - 1) / nblk;
    rows_per = (rows_per + TT_ROWS - 1) / TT_ROWS * TT_ROWS;
    nblk = (int)((n + rows_per - 1) / rows_per);
    dim3 grid(nblk, (k + TT_KA - 1) / TT_KA, (m + TT_MB - 1) / TT_MB);
    LRP_PROF(ctx, K_GEMM_T, 8.0 * n * (k + m), 2.0 * n * k * m);
    tall_gemm_t_kernel<<<grid, TT_THREADS, 0, ctx->stream>>>(A, lda, k, B, ldb, m, n, rows_per, partial_ws);
    LRP_LAUNCHED(ctx);
    int tot = k * m;
    LRP_PROF(ctx, K_REDUCE, 8.0 * nblk * k * m, 0);
    reduce_partials_kernel<<<(tot + 127) / 128, 128, 0, ctx->stream>>>(partial_ws, nblk, k, m, S, lds, accumulate);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

int tall_rownorm2(lrp_ctx* ctx, int64_t n, int k, const double* A, int64_t lda, const unsigned char* colmask, double* out) {
    LRP_PROF(ctx, K_ROWNORM, 8.0 * n * (k + 1), 2.0 * n * k);
    rownorm2_kernel<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(n, k, A, lda, colmask, out);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

int tall_gather_rows(lrp_ctx* ctx, const double* A, int64_t lda, int k, const int32_t* idx, int nidx, double* Out, int ldo) {
    if (nidx <= 0 || k <= 0) return LRP_OK;
    int tot = nidx * k;
    LRP_PROF(ctx, K_GATHER, 0, 0);
    gather_rows_kernel<<<(tot + 255) / 256, 256, 0, ctx->stream>>>(A, lda, k, idx, nidx, Out, ldo);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

int tall_copy(lrp_ctx* ctx, int64_t n, int k, const double* A, int64_t lda, double* B, int64_t ldb) {
    if (k <= 0) return LRP_OK;
    dim3 grid((unsigned)((n + 255) / 256), k < 64 ? k : 64);
    LRP_PROF(ctx, K_COPY, 16.0 * n * k, 0);
    copy_tall_kernel<<<grid, 256, 0, ctx->stream>>>(n, k, A, lda, B, ldb);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

int tall_lowrank_entries(lrp_ctx* ctx, int r, const double* U, int64_t ldu, const double* S, const double* V, int64_t ldv,
                         const int64_t* rows, const int64_t* cols, int64_t count, double* out) {
    if (count <= 0) return LRP_OK;
    LRP_PROF(ctx, K_ENTRIES, 0, 0);
    lowrank_entries_kernel<<<(unsigned)((count + 255) / 256), 256, 0, ctx->stream>>>(r, U, ldu, S, V, ldv, rows, cols, count, out);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}
