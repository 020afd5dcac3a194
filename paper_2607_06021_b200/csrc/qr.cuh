// qr.cuh -- thin QR of tall matrices (qr.cu)
#pragma once
#include "common.cuh"
// In place: A (n x K, ld lda) <- Q;  R (K x K, ld ldr, device) <- upper-triangular factor.  Requires n >= K.
// ws: tall_qr_ws_doubles(ctx, n, K) doubles of scratch.
size_t tall_qr_ws_doubles(const lrp_ctx* ctx, int64_t n, int K);
int tall_qr(lrp_ctx* ctx, int64_t n, int K, double* A, int64_t lda, double* R, int64_t ldr, double* ws);
