// tall.cuh -- host-side entry points of the tall-matrix streaming kernels (tall.cu).
#pragma once
#include "common.cuh"

enum { TG_PLAIN = 0, TG_SAMPLE = 1, TG_SUBTRACT = 2 };

// Out(n x m, ld ldo) = epilogue( A(n x k, ld lda) * B(k x m) )
//   TG_PLAIN    : B column-major k x m with ld ldb;                 Out = A B
//   TG_SUBTRACT : same B;                                          Out = Cin - A B   (Cin may alias Out)
//   TG_SAMPLE   : B(t,c) = scale_t[t] * Bsrc[idx[c] + t*ldb] (gathered rows of a tall factor);
//                 Out(i,c) = (A B)(i,c) / (d_i + d_idx[c])         eq. (4)
//   rownorm2 (may be NULL): rownorm2[i] = sum_c Out(i,c)^2          (next sweep's leverage scores, Alg. 3 line 3)
struct TallGemmArgs {
    int64_t n; int k; int m; int mode;
    const double* A; int64_t lda;
    const double* B; int64_t ldb;
    const int32_t* idx; const double* scale_t;
    const double* Cin; int64_t ldc;
    double* Out; int64_t ldo;
    double* rownorm2;
    const int* cond;            // optional device flag: the launch does nothing when *cond == 0 (decided on the device)
};

int tall_gemm(lrp_ctx* ctx, const TallGemmArgs& p);
// S(k x m, ld lds) (+)= A(n x k)^T B(n x m); partial_ws: tall_gemm_t_ws_doubles(ctx, n, k, m) doubles of scratch.
// Sadd (optional, ld ldadd) += the same product (the accumulated Gram-Schmidt coefficients).  One launch: the
// reduction over row slabs happens inside the kernel.
size_t tall_gemm_t_ws_doubles(const lrp_ctx* ctx, int64_t n, int k, int m);
int tall_gemm_t(lrp_ctx* ctx, int64_t n, const double* A, int64_t lda, int k, const double* B, int64_t ldb, int m,
                double* S, int64_t lds, int accumulate, double* partial_ws, double* Sadd = nullptr, int64_t ldadd = 0,
                const int* cond = nullptr);
int tall_rownorm2(lrp_ctx* ctx, int64_t n, int k, const double* A, int64_t lda, const unsigned char* colmask, double* out);
int tall_gather_rows(lrp_ctx* ctx, const double* A, int64_t lda, int k, const int32_t* idx, int nidx, double* Out, int ldo);
// fibers of the closed-form test matrices (eq. (6)): kind 1 Hilbert, kind 2 K; see tall.cu
int tall_matrix_fibers(lrp_ctx* ctx, int kind, int64_t n, int transposed, const int32_t* idx, int nidx, double* Out, int64_t ldo);
int tall_transpose(lrp_ctx* ctx, int64_t n, const double* A, int64_t lda, double* B, int64_t ldb);
int tall_spectral_divide(lrp_ctx* ctx, int64_t n, double* A, int64_t lda);
int tall_copy(lrp_ctx* ctx, int64_t n, int k, const double* A, int64_t lda, double* B, int64_t ldb);
int tall_lowrank_entries(lrp_ctx* ctx, int r, const double* U, int64_t ldu, const double* S, const double* V, int64_t ldv,
                         const int64_t* rows, const int64_t* cols, int64_t count, double* out);

// G (m x m) = E^T E with E = Cin - A B formed on the fly (never written).  Returns 1 (nothing launched) when the shape
// is outside the fused kernel's range; partial_ws as for tall_gemm_t(n, m, m).
int tall_mma_init(lrp_ctx* ctx);                 // one-time kernel attributes (lrp_create)
int tall_resid_gram(lrp_ctx* ctx, int64_t n, const double* A, int64_t lda, int k, const double* B, int64_t ldb,
                    const double* Cin, int64_t ldc, int m, double* G, int64_t ldg, double* partial_ws);
