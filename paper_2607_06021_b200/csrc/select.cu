// select.cu -- index selection from the leverage scores (Alg. 3 lines 4-6):
//   * deterministic top-k (reading Q5): the `num` largest scores ordered by (score descending, index ascending);
//   * the randomized form as printed (reading Q23): keep index i with probability min{1, c pi_i}, pi_i = score_i / cols,
//     with uniforms from a counter-based generator (a pure function of seed, sweep, side and i -- the oracle implements
//     the same integer recipe, so both sides draw the same numbers without sharing code); the kept indices come back
//     in the same (score desc, index asc) order.
// One mechanism serves both: every CTA sorts a chunk of 8192 (key, index) pairs in shared memory (bitonic network on a
// 64-bit order-preserving image of the score, ties by index) and keeps its first `num`; the survivors of all chunks are
// sorted again, level by level, until one CTA holds the answer.  Masked-out entries (not kept by the Bernoulli draw)
// and padding carry the largest key and sort last.  Bit-exact order, no floating-point comparison anywhere.
#include "common.cuh"
#include "core.cuh"
#include <limits.h>

namespace {

constexpr int SEL_NT = 1024;
constexpr int SEL_CHUNK = 8192;
constexpr size_t SEL_SMEM = (size_t)SEL_CHUNK * (sizeof(unsigned long long) + sizeof(int));
constexpr unsigned long long KEY_LAST = ~0ull;

// ascending key <=> descending score: order-preserving map of an IEEE double to uint64, complemented
__device__ __forceinline__ unsigned long long desc_key(double s) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(s);
    const unsigned long long asc = (b >> 63) ? ~b : (b | 0x8000000000000000ull);
    return ~asc;
}

// u in [0,1): SplitMix64 finaliser of a key built from (seed, sweep, side, i) -- oracle/lrp_oracle.py counter_uniforms
__device__ __forceinline__ double counter_uniform(unsigned long long x, long long i) {
    unsigned long long z = x + 0xD1B54A32D192ED03ull * (unsigned long long)(i + 1);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z = z ^ (z >> 31);
    return (double)(z >> 11) * 0x1.0p-53;
}

struct SelIn {
    const double* scores; int64_t n;                             // level 1: raw scores
    const unsigned long long* ckey; const int32_t* cidx; int64_t m;     // levels >= 2: candidate pairs
    int bernoulli; double c_over_cols_c, cols; unsigned long long x;     // Bernoulli mask (level 1 only)
    int* count;                                                  // kept-element counter (Bernoulli)
};

// sort the CTA's chunk and emit its first `num` pairs (final = 1: indices only, -1 where exhausted)
__global__ void __launch_bounds__(SEL_NT)
select_sort_kernel(SelIn in, int num, unsigned long long* __restrict__ okey, int32_t* __restrict__ oidx, int final_level) {
    extern __shared__ __align__(16) unsigned char sel_raw[];
    unsigned long long* key = (unsigned long long*)sel_raw;
    int* idx = (int*)(key + SEL_CHUNK);
    __shared__ int s_cnt;
    const int tid = threadIdx.x;
    const int64_t total = in.scores ? in.n : in.m;
    const int64_t b0 = (int64_t)blockIdx.x * SEL_CHUNK;
    int64_t left = total - b0; if (left > SEL_CHUNK) left = SEL_CHUNK;
    const int cnt = (int)left;
    int N = 32; while (N < cnt) N <<= 1;                         // sorted length: next power of two (>= 32)
    if (tid == 0) s_cnt = 0;
    __syncthreads();
    int kept = 0;
    for (int e = tid; e < N; e += SEL_NT) {
        unsigned long long k = KEY_LAST; int ix = INT_MAX;
        if (e < cnt) {
            if (in.scores) {
                const double s = in.scores[b0 + e];
                bool keep = true;
                if (in.bernoulli) {                              // p = min(1, c * (score / cols)); kept iff u < p
                    const double p = fmin(1.0, in.c_over_cols_c * (s / in.cols));
                    keep = counter_uniform(in.x, b0 + e) < p;
                    kept += keep ? 1 : 0;
                }
                if (keep) { k = desc_key(s); ix = (int)(b0 + e); }
            } else { k = in.ckey[b0 + e]; ix = in.cidx[b0 + e]; }
        }
        key[e] = k; idx[e] = ix;
    }
    if (in.bernoulli && in.scores && in.count) {
        for (int d = 16; d > 0; d >>= 1) kept += __shfl_xor_sync(0xffffffffu, kept, d);
        if ((tid & 31) == 0 && kept) atomicAdd(&s_cnt, kept);
    }
    __syncthreads();
    if (in.bernoulli && in.scores && in.count && tid == 0 && s_cnt) atomicAdd(in.count, s_cnt);
    for (int k2 = 2; k2 <= N; k2 <<= 1) {
        for (int j = k2 >> 1; j > 0; j >>= 1) {
            for (int p = tid; p < N / 2; p += SEL_NT) {
                const int i = ((p & ~(j - 1)) << 1) | (p & (j - 1)), l = i | j;
                const unsigned long long ka = key[i], kb = key[l];
                const int ia = idx[i], ib = idx[l];
                const bool a_gt_b = ka > kb || (ka == kb && ia > ib);
                const bool up = (i & k2) == 0;
                if (a_gt_b == up) { key[i] = kb; key[l] = ka; idx[i] = ib; idx[l] = ia; }
            }
            __syncthreads();
        }
    }
    for (int r = tid; r < num; r += SEL_NT) {
        const bool have = r < N;
        const unsigned long long k = have ? key[r] : KEY_LAST;
        const int ix = have ? idx[r] : INT_MAX;
        if (final_level) oidx[r] = (ix == INT_MAX) ? -1 : ix;
        else { okey[(int64_t)blockIdx.x * num + r] = k; oidx[(int64_t)blockIdx.x * num + r] = ix; }
    }
}

int64_t sel_chunks(int64_t m) { return (m + SEL_CHUNK - 1) / SEL_CHUNK; }

}  // namespace

int select_init(lrp_ctx* ctx) {
    LRP_CUDA(ctx, cudaFuncSetAttribute(select_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SEL_SMEM));
    return LRP_OK;
}

// two candidate buffers (levels ping-pong): G1 * num and G2 * num pairs, + the Bernoulli counter
size_t select_ws_bytes(const lrp_ctx* ctx, int64_t n, int num) {
    (void)ctx;
    if (num < 1) num = 1;
    const int64_t g1 = sel_chunks(n), g2 = sel_chunks(g1 * num);
    return lrp_align_up((size_t)g1 * num * 8) + lrp_align_up((size_t)g1 * num * 4) + lrp_align_up((size_t)g2 * num * 8) +
           lrp_align_up((size_t)g2 * num * 4) + 256;
}

int select_topk(lrp_ctx* ctx, int64_t n, const double* scores, int num, int32_t* idx_out, void* ws, const SelectBernoulli* bern,
                int* d_count) {
    if (num <= 0) return LRP_OK;
    if (num > SEL_CHUNK / 2) return LRP_ERR_BADARG;
    const int64_t g1 = sel_chunks(n), g2 = sel_chunks(g1 * num);
    char* base = (char*)ws;
    unsigned long long* keyA = (unsigned long long*)base; base += lrp_align_up((size_t)g1 * num * 8);
    int32_t* idxA = (int32_t*)base; base += lrp_align_up((size_t)g1 * num * 4);
    unsigned long long* keyB = (unsigned long long*)base; base += lrp_align_up((size_t)g2 * num * 8);
    int32_t* idxB = (int32_t*)base;
    SelIn in{};
    in.scores = scores; in.n = n;
    if (bern) {
        in.bernoulli = 1; in.c_over_cols_c = bern->c; in.cols = (double)bern->cols; in.count = d_count;
        in.x = bern->seed + 0x9E3779B97F4A7C15ull * (unsigned long long)(1 + 2 * bern->sweep + bern->side);
        if (d_count) LRP_CUDA(ctx, cudaMemsetAsync(d_count, 0, sizeof(int), ctx->stream));
    }
    int64_t G = g1;
    bool toA = true;
    for (int level = 0;; ++level) {
        const bool fin = G == 1;
        LRP_PROF(ctx, K_TOPK, level == 0 ? 8.0 * n : 0.0, 0);
        select_sort_kernel<<<(unsigned)G, SEL_NT, SEL_SMEM, ctx->stream>>>(in, num, toA ? keyA : keyB, fin ? idx_out : (toA ? idxA : idxB), fin ? 1 : 0);
        LRP_LAUNCHED(ctx);
        if (fin) break;
        in = SelIn{};
        in.ckey = toA ? keyA : keyB; in.cidx = toA ? idxA : idxB; in.m = G * num;
        G = sel_chunks(in.m);
        toA = !toA;
    }
    return LRP_OK;
}
