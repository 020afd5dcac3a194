// select.cu -- deterministic top-k of the leverage scores (Alg. 3 lines 4-6, in the top-k form of
// DESIGN.md reading Q5): the `num` largest scores ordered by (score descending, index ascending).
// Two levels: every CTA extracts the sorted top-`num` of its contiguous chunk by repeated block arg-max (each
// thread caches the best of its <= 64 strided elements and only the winner rescans), then one CTA merges the
// sorted candidate lists.
#include "common.cuh"
#include "core.cuh"
#include <limits.h>

namespace {

constexpr int SEL_NT = 256;
constexpr int SEL_MAX_PER_THREAD = 64;
constexpr int SEL_MAX_CHUNK = SEL_NT * SEL_MAX_PER_THREAD;   // 16384

struct KV { double s; int i; };
__device__ __forceinline__ bool better(const KV& a, const KV& b) { return a.s > b.s || (a.s == b.s && a.i < b.i); }
__device__ __forceinline__ KV warp_best(KV v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        KV o; o.s = __shfl_xor_sync(0xffffffffu, v.s, d); o.i = __shfl_xor_sync(0xffffffffu, v.i, d);
        if (better(o, v)) v = o;
    }
    return v;
}
// block-wide best; every thread returns the winner.  wb: >= 33 KV of shared memory.
__device__ __forceinline__ KV block_best(KV v, KV* wb) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    v = warp_best(v);
    if (lane == 0) wb[warp] = v;
    __syncthreads();
    if (warp == 0) {
        KV t; t.s = -1.0; t.i = INT_MAX;
        if (lane < nw) t = wb[lane];
        t = warp_best(t);
        if (lane == 0) wb[32] = t;
    }
    __syncthreads();
    KV r = wb[32];
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(SEL_NT)
topk_chunk_kernel(int64_t n, int64_t chunk, const double* __restrict__ scores, int num,
                  double* __restrict__ cand_s, int32_t* __restrict__ cand_i) {
    __shared__ KV wb[33];
    const int tid = threadIdx.x;
    const int64_t b0 = (int64_t)blockIdx.x * chunk;
    int64_t b1 = b0 + chunk; if (b1 > n) b1 = n;
    const int cnt = (int)(b1 - b0);
    unsigned long long taken = 0ull;
    auto rescan = [&]() {
        KV best; best.s = -1.0; best.i = INT_MAX;
        int slot = 0;
        for (int e = tid; e < cnt; e += SEL_NT, ++slot) {
            if ((taken >> slot) & 1ull) continue;
            KV c; c.s = scores[b0 + e]; c.i = (int)(b0 + e);
            if (better(c, best)) best = c;
        }
        return best;
    };
    KV mine = rescan();
    for (int r = 0; r < num; ++r) {
        KV w = block_best(mine, wb);
        if (tid == 0) {
            cand_s[(int64_t)blockIdx.x * num + r] = w.s;
            cand_i[(int64_t)blockIdx.x * num + r] = (w.i == INT_MAX) ? -1 : w.i;
        }
        if (w.i != INT_MAX && (int)((w.i - b0) % SEL_NT) == tid) {
            int slot = (int)((w.i - b0) / SEL_NT);
            taken |= 1ull << slot;
            mine = rescan();
        }
    }
}

// merge G descending lists of length num (entries with index -1 are exhausted) into idx_out[0..num)
__global__ void __launch_bounds__(1024)
topk_merge_kernel(int G, int num, const double* __restrict__ cand_s, const int32_t* __restrict__ cand_i,
                  int32_t* __restrict__ idx_out) {
    __shared__ KV wb[33];
    extern __shared__ int heads[];            // G list heads
    const int tid = threadIdx.x;
    for (int g = tid; g < G; g += blockDim.x) heads[g] = 0;
    __syncthreads();
    for (int r = 0; r < num; ++r) {
        KV best; best.s = -1.0; best.i = INT_MAX;
        for (int g = tid; g < G; g += blockDim.x) {
            int h = heads[g];
            if (h < num) {
                int32_t ci = cand_i[(int64_t)g * num + h];
                if (ci >= 0) { KV c; c.s = cand_s[(int64_t)g * num + h]; c.i = ci; if (better(c, best)) best = c; }
            }
        }
        KV w = block_best(best, wb);
        if (tid == 0) idx_out[r] = (w.i == INT_MAX) ? -1 : w.i;
        if (w.i != INT_MAX) {
            for (int g = tid; g < G; g += blockDim.x) {
                int h = heads[g];
                if (h < num && cand_i[(int64_t)g * num + h] == w.i) heads[g] = h + 1;
            }
        }
        __syncthreads();
    }
}

void sel_geometry(const lrp_ctx* ctx, int64_t n, int* G, int64_t* chunk) {
    int64_t g = (n + SEL_MAX_CHUNK - 1) / SEL_MAX_CHUNK;
    int64_t want = (int64_t)lrp_sm_count(ctx) * 4;      // without a ctx (workspace sizing): the upper bound of the SM count
    int64_t by_rows = (n + 1023) / 1024;
    int64_t g2 = want < by_rows ? want : by_rows;
    if (g2 > g) g = g2;
    if (g < 1) g = 1;
    int64_t c = (n + g - 1) / g;
    g = (n + c - 1) / c;
    *G = (int)g; *chunk = c;
}

}  // namespace

size_t select_ws_bytes(const lrp_ctx* ctx, int64_t n, int num) {
    int G; int64_t chunk; sel_geometry(ctx, n, &G, &chunk);
    return lrp_align_up((size_t)G * num * sizeof(double)) + lrp_align_up((size_t)G * num * sizeof(int32_t));
}

int select_topk(lrp_ctx* ctx, int64_t n, const double* scores, int num, int32_t* idx_out, void* ws) {
    if (num <= 0) return LRP_OK;
    int G; int64_t chunk; sel_geometry(ctx, n, &G, &chunk);
    double* cand_s = (double*)ws;
    int32_t* cand_i = (int32_t*)((char*)ws + lrp_align_up((size_t)G * num * sizeof(double)));
    LRP_PROF(ctx, K_TOPK_CHUNK, 8.0 * n, 0);
    topk_chunk_kernel<<<G, SEL_NT, 0, ctx->stream>>>(n, chunk, scores, num, cand_s, G == 1 ? idx_out : cand_i);
    LRP_LAUNCHED(ctx);
    if (G > 1) {
        LRP_PROF(ctx, K_TOPK_MERGE, 0, 0);
        topk_merge_kernel<<<1, 1024, G * sizeof(int), ctx->stream>>>(G, num, cand_s, cand_i, idx_out);
        LRP_LAUNCHED(ctx);
    }
    return LRP_OK;
}
