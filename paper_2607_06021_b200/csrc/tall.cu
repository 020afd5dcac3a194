// tall.cu -- streaming kernels over "tall" (n x small, column-major) fp64 matrices:
//   tall_gemm    : Out(n x m) = epilogue( A(n x k) B(k x m) )     fiber sampling (eq. (4)),
//                  factor rebuild U = Q Uc (Alg. 1 lines 9/14), Gram-Schmidt update P -= Q S
//   tall_gemm_t  : S(k x m) = A(n x k)^T B(n x m)                  projections / Gram blocks (reduction over n)
//   row norms, gathers, low-rank entry evaluation.
// The two contractions (tall_gemm, tall_gemm_t) live in tall_mma.cu.
#include "common.cuh"
#include "tall.cuh"
#include <math.h>

namespace {

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

// Fibers of the test matrices of eq. (6), PAPER.md:264-267 (0-based i, j; square n x n):
//   kind 1 (Hilbert):  G(i,j) = 1 / (1 + i + j)
//   kind 2 (K):        G(i,j) = (|x_i + y_j| / 2)^5,  x_i = -1 + 2 i/(n-1),  y_j = -1 + 2 j/(n-1)
// transposed = 0: Out(i, c) = G(i, idx[c]) (columns, C = G(:,J));  transposed = 1: Out(j, c) = G(idx[c], j) (rows, G(I,:)^T)
__device__ __forceinline__ double matrix_entry(int kind, int64_t n, int64_t i, int64_t j) {
    if (kind == 1) return 1.0 / (1.0 + (double)i + (double)j);
    const double x = -1.0 + 2.0 * (double)i / (double)(n - 1), y = -1.0 + 2.0 * (double)j / (double)(n - 1);
    const double t = fabs(x + y) / 2.0, t2 = t * t;
    return t2 * t2 * t;
}
__global__ void matrix_fibers_kernel(int kind, int64_t n, int transposed, const int32_t* __restrict__ idx, int nidx,
                                     double* __restrict__ Out, int64_t ldo) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    for (int c = blockIdx.y; c < nidx; c += gridDim.y) {
        const int64_t f = idx[c];
        Out[i + (int64_t)c * ldo] = transposed ? matrix_entry(kind, n, f, i) : matrix_entry(kind, n, i, f);
    }
}

// B (n x n, ld ldb) = A^T (A n x n, ld lda): 32 x 32 tiles through shared memory (dense full-rank baseline only)
__global__ void transpose_kernel(int64_t n, const double* __restrict__ A, int64_t lda, double* __restrict__ B, int64_t ldb) {
    __shared__ double tile[32][33];
    const int64_t i0 = (int64_t)blockIdx.x * 32, j0 = (int64_t)blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int64_t i = i0 + threadIdx.x, j = j0 + r;
        if (i < n && j < n) tile[r][threadIdx.x] = A[i + j * lda];
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int64_t j = j0 + threadIdx.x, i = i0 + r;
        if (i < n && j < n) B[j + i * ldb] = tile[threadIdx.x][r];
    }
}
// A(i,j) /= d_i + d_j,  d_k = 4 (n+1)^2 sin^2(pi (k+1) / (2(n+1)))     eq. (4)
__global__ void spectral_divide_kernel(int64_t n, double* __restrict__ A, int64_t lda) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double invN = 1.0 / (double)(n + 1), f = 4.0 * (double)(n + 1) * (double)(n + 1);
    const double si = sinpi(0.5 * (double)(i + 1) * invN), di = f * si * si;
    for (int64_t j = blockIdx.y; j < n; j += gridDim.y) {
        const double sj = sinpi(0.5 * (double)(j + 1) * invN);
        A[i + j * lda] /= di + f * sj * sj;
    }
}

}  // namespace

int tall_transpose(lrp_ctx* ctx, int64_t n, const double* A, int64_t lda, double* B, int64_t ldb) {
    dim3 grid((unsigned)((n + 31) / 32), (unsigned)((n + 31) / 32));
    LRP_PROF(ctx, K_COPY, 16.0 * n * n, 0);
    transpose_kernel<<<grid, dim3(32, 8), 0, ctx->stream>>>(n, A, lda, B, ldb);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}
int tall_spectral_divide(lrp_ctx* ctx, int64_t n, double* A, int64_t lda) {
    dim3 grid((unsigned)((n + 255) / 256), (unsigned)(n < 1024 ? n : 1024));
    LRP_PROF(ctx, K_COPY, 16.0 * n * n, 0);
    spectral_divide_kernel<<<grid, 256, 0, ctx->stream>>>(n, A, lda);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

int tall_matrix_fibers(lrp_ctx* ctx, int kind, int64_t n, int transposed, const int32_t* idx, int nidx, double* Out, int64_t ldo) {
    if (nidx <= 0) return LRP_OK;
    dim3 grid((unsigned)((n + 255) / 256), nidx < 64 ? nidx : 64);
    LRP_PROF(ctx, K_GEMM_SAMPLE, 8.0 * n * nidx, 6.0 * n * nidx);
    matrix_fibers_kernel<<<grid, 256, 0, ctx->stream>>>(kind, n, transposed, idx, nidx, Out, ldo);
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
