// qr.cuh -- thin QR of tall matrices (qr.cu)
#pragma once
#include "common.cuh"
// In place: A (n x K, ld lda) <- Q;  R (K x K, ld ldr, device) <- upper-triangular factor.  Requires n >= K.
// ws: tall_qr_ws_doubles(ctx, n, K) doubles of scratch.
size_t tall_qr_ws_doubles(const lrp_ctx* ctx, int64_t n, int K);
int tall_qr_init(lrp_ctx* ctx);                  // one-time kernel attributes (lrp_create)
int tall_qr(lrp_ctx* ctx, int64_t n, int K, double* A, int64_t lda, double* R, int64_t ldr, double* ws);
// Two independent factorizations advanced panel by panel on ctx->stream and ctx->aux (joined on return into ctx->stream).
int tall_qr_pair(lrp_ctx* ctx, int64_t n, int K1, double* A1, int64_t lda1, double* R1, int64_t ldr1, double* ws1,
                 int K2, double* A2, int64_t lda2, double* R2, int64_t ldr2, double* ws2);

// Same, extending existing factorizations: the leading k01 (k02) columns of A1 (A2) already hold orthonormal Q columns
// and the leading k0 x k0 block of R their triangular factor (QR of a column prefix is the prefix of the QR); only
// the columns from k0 on are projected and factored.  k0 = 0: the whole block.
int tall_qr_pair_from(lrp_ctx* ctx, int64_t n, int K1, int k01, double* A1, int64_t lda1, double* R1, int64_t ldr1, double* ws1,
                      int K2, int k02, double* A2, int64_t lda2, double* R2, int64_t ldr2, double* ws2);

struct QrJob {
    int k0;                                       // leading columns already factored (0: none)
    int64_t n; int K; double* A; int64_t lda; double* R; int64_t ldr; double* ws; cudaStream_t stream;
    double *stack, *partial, *Stmp, *d_small;     // carved from ws by tall_qr_begin
};
