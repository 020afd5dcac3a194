// deim.cu -- index selection by the discrete empirical interpolation methods of Alg. 2:
//   QDEIM (lines 7-10): column-pivoted QR of U^T -- here as row-pivoted Gram-Schmidt on the n x r matrix U itself (equal in
//          exact arithmetic): at every step the row with the largest residual 2-norm is the pivot, its normalised
//          residual q is projected out of every row and the residual norms are recomputed exactly;
//   DEIM  (lines 3-6): LU with partial pivoting of U: at step c the unchosen row with the largest |entry| of column c is the
//          pivot and column c is eliminated from the other unchosen rows.
// Both return r indices in pivot order and cost O(n r^2) ("scale quadratically with the size of the index
// set"): one launch per step; a thread owns a row, every CTA reports its best (value, index), the last CTA to arrive
// reduces the partials in a fixed order (lowest index wins ties: deterministic), records the pivot and stages the pivot
// row for the next step.  These are the pivoted factorizations the paper could not get natively on the GPU
// (PAPER.md:246, 256).  The working matrix is destroyed.
#include "common.cuh"
#include "core.cuh"
#include <limits.h>

namespace {

constexpr int DM_NT = 256;

struct DeimArgs {
    int64_t n; int r; int step; int qdeim;
    double* A; int64_t lda;
    int32_t* idx_out;                 // [r] device
    double* blk_val; int32_t* blk_idx; int G;
    double* piv;                      // [r + 2]: pivot row (DEIM) / unit residual q (QDEIM); [r] = pivot index as double
    unsigned* counter; unsigned char* taken;
};

__device__ __forceinline__ bool dm_better(double v, int i, double bv, int bi) { return v > bv || (v == bv && i < bi); }

// step < 0: initial scan (no update).  step = c >= 0: project out / eliminate with pivot c, then find pivot c + 1.
__global__ void __launch_bounds__(DM_NT)
deim_step_kernel(DeimArgs a) {
    extern __shared__ double pv[];                 // [r + 1]
    __shared__ double sv[DM_NT / 32]; __shared__ int si[DM_NT / 32];
    __shared__ int s_last;
    const int tid = threadIdx.x, r = a.r, c = a.step;
    const int64_t i = (int64_t)blockIdx.x * DM_NT + tid;
    if (c >= 0) { for (int t = tid; t <= r; t += DM_NT) pv[t] = __ldcg(a.piv + t); }
    __syncthreads();
    double val = -1.0;
    if (i < a.n) {
        double* row = a.A + i;
        const bool was_taken = a.taken[i] != 0;
        if (c >= 0 && (int64_t)pv[r] == i) {       // the pivot row of this step: out of the game
            a.taken[i] = 1;
            for (int t = (a.qdeim ? 0 : c + 1); t < r; ++t) row[(int64_t)t * a.lda] = 0.0;
        } else if (!was_taken) {
            if (a.qdeim) {
                double nrm = 0.0;
                if (c >= 0) {
                    double w = 0.0;
                    for (int t = 0; t < r; ++t) w = fma(row[(int64_t)t * a.lda], pv[t], w);
                    for (int t = 0; t < r; ++t) {
                        const double x = fma(-w, pv[t], row[(int64_t)t * a.lda]);
                        row[(int64_t)t * a.lda] = x; nrm = fma(x, x, nrm);
                    }
                } else {
                    for (int t = 0; t < r; ++t) { const double x = row[(int64_t)t * a.lda]; nrm = fma(x, x, nrm); }
                }
                val = nrm;
            } else {
                if (c >= 0) {
                    const double m = pv[c] != 0.0 ? row[(int64_t)c * a.lda] / pv[c] : 0.0;
                    for (int t = c + 1; t < r; ++t) row[(int64_t)t * a.lda] = fma(-m, pv[t], row[(int64_t)t * a.lda]);
                }
                if (c + 1 < r) val = fabs(row[(int64_t)(c + 1) * a.lda]);
            }
        }
    }
    // block best (value desc, index asc)
    int bi = (i < a.n) ? (int)i : INT_MAX;
    double bv = val;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, bv, d); const int oi = __shfl_xor_sync(0xffffffffu, bi, d);
        if (dm_better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
    }
    if ((tid & 31) == 0) { sv[tid >> 5] = bv; si[tid >> 5] = bi; }
    __syncthreads();
    if (tid == 0) {
        for (int w = 1; w < DM_NT / 32; ++w) if (dm_better(sv[w], si[w], bv, bi)) { bv = sv[w]; bi = si[w]; }
        a.blk_val[blockIdx.x] = bv; a.blk_idx[blockIdx.x] = bi;
        __threadfence();
        s_last = (atomicAdd(a.counter, 1u) == (unsigned)a.G - 1u) ? 1 : 0;
    }
    __threadfence();
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // last CTA: global best over the G partials, fixed order
    bv = -2.0; bi = INT_MAX;
    for (int g = tid; g < a.G; g += DM_NT) {
        const double v = __ldcg(a.blk_val + g); const int ix = __ldcg(a.blk_idx + g);
        if (dm_better(v, ix, bv, bi)) { bv = v; bi = ix; }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, bv, d); const int oi = __shfl_xor_sync(0xffffffffu, bi, d);
        if (dm_better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
    }
    __syncthreads();
    if ((tid & 31) == 0) { sv[tid >> 5] = bv; si[tid >> 5] = bi; }
    __syncthreads();
    if (tid == 0) {
        for (int w = 1; w < DM_NT / 32; ++w) if (dm_better(sv[w], si[w], bv, bi)) { bv = sv[w]; bi = si[w]; }
        sv[0] = bv; si[0] = bi;
        a.idx_out[c + 1] = bi;
        *a.counter = 0u;
    }
    __syncthreads();
    const int p = si[0];
    const double pvnorm = sv[0];
    if (p == INT_MAX) return;
    // stage the pivot row for the next step (QDEIM: the unit residual; DEIM: the row itself)
    const double sc = a.qdeim ? (pvnorm > 0.0 ? rsqrt(pvnorm) : 0.0) : 1.0;
    for (int t = tid; t < r; t += DM_NT) a.piv[t] = __ldcg(a.A + p + (int64_t)t * a.lda) * sc;
    if (tid == 0) a.piv[r] = (double)p;
}

}  // namespace

size_t deim_ws_bytes(int64_t n, int r) {
    const int64_t G = (n + DM_NT - 1) / DM_NT;
    return lrp_align_up((size_t)G * sizeof(double)) + lrp_align_up((size_t)G * sizeof(int32_t)) + lrp_align_up((size_t)(r + 2) * sizeof(double)) +
           lrp_align_up(256) + lrp_align_up((size_t)n);
}

// r indices of the n x r matrix A (orthonormal columns expected; destroyed) by QDEIM (qdeim = 1) or DEIM (0) -> idx_out[0..r)
int deim_select(lrp_ctx* ctx, int qdeim, int64_t n, int r, double* A, int64_t lda, int32_t* idx_out, void* ws) {
    if (r <= 0) return LRP_OK;
    if (r > n) return LRP_ERR_BADARG;
    DeimArgs a{};
    a.n = n; a.r = r; a.qdeim = qdeim; a.A = A; a.lda = lda; a.idx_out = idx_out;
    a.G = (int)((n + DM_NT - 1) / DM_NT);
    char* base = (char*)ws;
    a.blk_val = (double*)base; base += lrp_align_up((size_t)a.G * sizeof(double));
    a.blk_idx = (int32_t*)base; base += lrp_align_up((size_t)a.G * sizeof(int32_t));
    a.piv = (double*)base; base += lrp_align_up((size_t)(r + 2) * sizeof(double));
    a.counter = (unsigned*)base; base += lrp_align_up(256);
    a.taken = (unsigned char*)base;
    LRP_CUDA(ctx, cudaMemsetAsync(a.counter, 0, 256, ctx->stream));
    LRP_CUDA(ctx, cudaMemsetAsync(a.taken, 0, (size_t)n, ctx->stream));
    const size_t smem = (size_t)(r + 1) * sizeof(double);
    for (int c = -1; c < r - 1; ++c) {            // launch c finds pivot c + 1
        a.step = c;
        const double cols = qdeim ? (double)r : (double)(r - c - 1);
        LRP_PROF(ctx, K_DEIM, 8.0 * n * cols * (c < 0 ? 1.0 : (qdeim ? 3.0 : 2.0)), 2.0 * n * cols * (c < 0 ? 1.0 : 2.0));
        deim_step_kernel<<<a.G, DM_NT, smem, ctx->stream>>>(a);
        LRP_LAUNCHED(ctx);
    }
    return LRP_OK;
}
