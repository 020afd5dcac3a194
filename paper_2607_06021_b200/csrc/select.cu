// select.cu -- index selection from the leverage scores (Alg. 3 lines 4-6):
//   * deterministic top-k (reading Q5): the `num` largest scores ordered by (score descending, index ascending);
//   * the randomized form as printed (reading Q23): keep index i with probability min{1, c pi_i}, pi_i = score_i / cols,
//     with uniforms from a counter-based generator (a pure function of seed, sweep, side and i -- the oracle implements
//     the same integer recipe, so both sides draw the same numbers without sharing code); the kept indices come back
//     in the same (score desc, index asc) order.
// Every comparison is on a 64-bit order-preserving image of the score (ties by index): bit-exact order, no floating-point
// comparison anywhere.  Two launches in the common case (num << n):
//   select_hist_kernel    : histogram of the keys' leading 13 bits (shared-memory histogram per CTA, merged into one global
//                           one); the last CTA to arrive scans it for the threshold bin T that holds the num-th key;
//   select_collect_kernel : every key with bin <= T (a few hundred at most for a decaying score distribution) is appended
//                           to a candidate list; the last CTA to arrive sorts the list (bitonic network in shared memory)
//                           and writes the first `num` indices.
// When more than SEL_CAND keys share the threshold bin's prefix (flat score distributions, massive ties) the state's
// `fallback` flag is set and the multi-level sort takes over: every CTA sorts a chunk of 8192 (key, index) pairs and keeps
// its first `num`; the survivors are sorted again, level by level, until one CTA holds the answer.  Those launches are
// always enqueued and return at once when the flag is clear (no host round trip).  Masked-out entries (not kept by the
// Bernoulli draw) and padding carry the largest key and sort last.
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

// ------------------------------------------------------------------------------------------------ histogram path
constexpr int SEL_BINS = 8192;                 // leading 13 bits of a non-negative score's key: exponent + 2 mantissa bits
constexpr int SEL_HNT = 512;
constexpr int SEL_CAND = 4096;                 // candidate list capacity (>= the largest num)
constexpr size_t SEL_CSMEM = (size_t)SEL_CAND * (sizeof(unsigned long long) + sizeof(int));

// monotone non-decreasing in the key; negative scores (impossible for sums of squares) and NaN patterns share the last bin
__device__ __forceinline__ int key_bin(unsigned long long key) { return (key >> 63) ? SEL_BINS - 1 : (int)(key >> 50); }

struct SelState {                               // zeroed by a memset node at the start of every call
    unsigned int ticketA, ticketB, nwritten;
    unsigned int T, ncand, total;
    int fallback;
    int pad;
};

struct SelMask { int bernoulli; double c; double cols; unsigned long long x; };

__device__ __forceinline__ bool sel_keep(const SelMask& mk, double s, int64_t i) {   // p = min(1, c * (score / cols)); kept iff u < p
    if (!mk.bernoulli) return true;
    const double p = fmin(1.0, mk.c * (s / mk.cols));
    return counter_uniform(mk.x, i) < p;
}

__global__ void __launch_bounds__(SEL_HNT)
select_hist_kernel(const double* __restrict__ scores, int64_t n, SelMask mk, int num, unsigned int* __restrict__ ghist,
                   SelState* __restrict__ st, int* __restrict__ count) {
    __shared__ unsigned int sh[SEL_BINS];
    __shared__ unsigned int s_warp[SEL_HNT / 32];
    __shared__ unsigned int s_misc[2];
    const int tid = threadIdx.x;
    for (int b = tid; b < SEL_BINS; b += SEL_HNT) sh[b] = 0u;
    __syncthreads();
    const int64_t stride = (int64_t)gridDim.x * SEL_HNT;
    for (int64_t i = (int64_t)blockIdx.x * SEL_HNT + tid; i < n; i += stride) {
        const double s = __ldg(scores + i);
        if (sel_keep(mk, s, i)) atomicAdd(&sh[key_bin(desc_key(s))], 1u);
    }
    __syncthreads();
    for (int b = tid; b < SEL_BINS; b += SEL_HNT) { const unsigned int v = sh[b]; if (v) atomicAdd(ghist + b, v); }
    __threadfence();
    __syncthreads();
    if (tid == 0) s_misc[0] = (atomicAdd(&st->ticketA, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!s_misc[0]) return;
    __threadfence();
    // last CTA: the threshold bin T = the first bin at which the running count reaches want = min(num, total)
    constexpr int PER = SEL_BINS / SEL_HNT;
    unsigned int h[PER], loc = 0;
#pragma unroll
    for (int q = 0; q < PER; ++q) { h[q] = __ldcg(ghist + tid * PER + q); loc += h[q]; }
    unsigned int inc = loc;                                           // inclusive scan over the CTA's threads
    for (int d = 1; d < 32; d <<= 1) { const unsigned int t = __shfl_up_sync(0xffffffffu, inc, d); if ((tid & 31) >= d) inc += t; }
    if ((tid & 31) == 31) s_warp[tid >> 5] = inc;
    __syncthreads();
    unsigned int base = 0, total = 0;
    for (int w = 0; w < SEL_HNT / 32; ++w) { const unsigned int v = s_warp[w]; if (w < (tid >> 5)) base += v; total += v; }
    unsigned int run = base + inc - loc;                              // keys in the bins before this thread's
    const unsigned int want = min((unsigned int)num, total);
    if (tid == 0) { st->total = total; st->ncand = 0u; st->T = 0u; st->fallback = 0; if (count) *count = (int)total; }
    __syncthreads();
    if (want > 0) {
#pragma unroll
        for (int q = 0; q < PER; ++q) {
            if (run < want && run + h[q] >= want) { st->T = (unsigned int)(tid * PER + q); st->ncand = run + h[q]; st->fallback = (run + h[q] > (unsigned int)SEL_CAND) ? 1 : 0; }
            run += h[q];
        }
    }
}

// candidates (bin <= T) -> list; the last CTA sorts the list and writes idx_out[0..num) (-1 where the list is exhausted)
__global__ void __launch_bounds__(SEL_HNT)
select_collect_kernel(const double* __restrict__ scores, int64_t n, SelMask mk, int num, SelState* __restrict__ st,
                      unsigned long long* __restrict__ ckey, int32_t* __restrict__ cidx, int32_t* __restrict__ idx_out) {
    extern __shared__ __align__(16) unsigned char selc_raw[];
    __shared__ unsigned int s_last;
    const int tid = threadIdx.x;
    if (*(volatile int*)&st->fallback) return;
    const unsigned int ncand = *(volatile unsigned int*)&st->ncand;
    const int T = (int)*(volatile unsigned int*)&st->T;
    if (ncand > 0) {
        const int64_t stride = (int64_t)gridDim.x * SEL_HNT;
        for (int64_t i = (int64_t)blockIdx.x * SEL_HNT + tid; i < n; i += stride) {
            const double s = __ldg(scores + i);
            const unsigned long long k = desc_key(s);
            if (key_bin(k) <= T && sel_keep(mk, s, i)) {
                const unsigned int p = atomicAdd(&st->nwritten, 1u);
                if (p < (unsigned int)SEL_CAND) { ckey[p] = k; cidx[p] = (int32_t)i; }
            }
        }
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = (atomicAdd(&st->ticketB, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    unsigned long long* key = (unsigned long long*)selc_raw;
    int* idx = (int*)(key + SEL_CAND);
    const int cnt = (int)ncand;
    int N = 32; while (N < cnt) N <<= 1;
    for (int e = tid; e < N; e += SEL_HNT) {
        const bool have = e < cnt;
        key[e] = have ? __ldcg(ckey + e) : KEY_LAST;
        idx[e] = have ? __ldcg(cidx + e) : INT_MAX;
    }
    __syncthreads();
    for (int k2 = 2; k2 <= N; k2 <<= 1) {
        for (int j = k2 >> 1; j > 0; j >>= 1) {
            for (int p = tid; p < N / 2; p += SEL_HNT) {
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
    for (int r = tid; r < num; r += SEL_HNT) idx_out[r] = (r < N && idx[r] != INT_MAX) ? idx[r] : -1;
}

// ------------------------------------------------------------------------------------------------ multi-level sort (fallback)
struct SelIn {
    const double* scores; int64_t n;                             // level 1: raw scores
    const unsigned long long* ckey; const int32_t* cidx; int64_t m;     // levels >= 2: candidate pairs
    int bernoulli; double c_over_cols_c, cols; unsigned long long x;     // Bernoulli mask (level 1 only)
    int* count;                                                  // kept-element counter (Bernoulli)
};

// sort the CTA's chunk and emit its first `num` pairs (final = 1: indices only, -1 where exhausted)
__global__ void __launch_bounds__(SEL_NT)
select_sort_kernel(SelIn in, int num, unsigned long long* __restrict__ okey, int32_t* __restrict__ oidx, int final_level,
                   const int* __restrict__ cond) {
    extern __shared__ __align__(16) unsigned char sel_raw[];
    if (cond && *(volatile const int*)cond == 0) return;            // the histogram path already produced the answer
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
    LRP_CUDA(ctx, cudaFuncSetAttribute(select_collect_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SEL_CSMEM));
    return LRP_OK;
}

// histogram + state + candidate list, then the two candidate buffers of the fallback (levels ping-pong): G1 * num and G2 * num pairs
size_t select_ws_bytes(const lrp_ctx* ctx, int64_t n, int num) {
    (void)ctx;
    if (num < 1) num = 1;
    const int64_t g1 = sel_chunks(n), g2 = sel_chunks(g1 * num);
    return lrp_align_up(sizeof(unsigned int) * SEL_BINS + sizeof(SelState)) + lrp_align_up((size_t)SEL_CAND * 8) +
           lrp_align_up((size_t)SEL_CAND * 4) + lrp_align_up((size_t)g1 * num * 8) + lrp_align_up((size_t)g1 * num * 4) +
           lrp_align_up((size_t)g2 * num * 8) + lrp_align_up((size_t)g2 * num * 4) + 256;
}

int select_topk(lrp_ctx* ctx, int64_t n, const double* scores, int num, int32_t* idx_out, void* ws, const SelectBernoulli* bern,
                int* d_count) {
    if (num <= 0) return LRP_OK;
    if (num > SEL_CAND) return LRP_ERR_BADARG;
    const int64_t g1 = sel_chunks(n), g2 = sel_chunks(g1 * num);
    char* base = (char*)ws;
    unsigned int* ghist = (unsigned int*)base;
    SelState* st = (SelState*)(ghist + SEL_BINS); base += lrp_align_up(sizeof(unsigned int) * SEL_BINS + sizeof(SelState));
    unsigned long long* ckey = (unsigned long long*)base; base += lrp_align_up((size_t)SEL_CAND * 8);
    int32_t* cidx = (int32_t*)base; base += lrp_align_up((size_t)SEL_CAND * 4);
    unsigned long long* keyA = (unsigned long long*)base; base += lrp_align_up((size_t)g1 * num * 8);
    int32_t* idxA = (int32_t*)base; base += lrp_align_up((size_t)g1 * num * 4);
    unsigned long long* keyB = (unsigned long long*)base; base += lrp_align_up((size_t)g2 * num * 8);
    int32_t* idxB = (int32_t*)base;
    SelMask mk{};
    if (bern) {
        mk.bernoulli = 1; mk.c = bern->c; mk.cols = (double)bern->cols;
        mk.x = bern->seed + 0x9E3779B97F4A7C15ull * (unsigned long long)(1 + 2 * bern->sweep + bern->side);
    }
    LRP_CUDA(ctx, cudaMemsetAsync(ghist, 0, sizeof(unsigned int) * SEL_BINS + sizeof(SelState), ctx->stream));
    int64_t gh = (n + (int64_t)SEL_HNT * 4 - 1) / ((int64_t)SEL_HNT * 4);
    const int64_t gmax = 2 * (int64_t)lrp_sm_count(ctx);
    if (gh > gmax) gh = gmax;
    if (gh < 1) gh = 1;
    LRP_PROF(ctx, K_TOPK, 8.0 * n, 0);
    select_hist_kernel<<<(unsigned)gh, SEL_HNT, 0, ctx->stream>>>(scores, n, mk, num, ghist, st, bern ? d_count : nullptr);
    LRP_LAUNCHED(ctx);
    LRP_PROF(ctx, K_TOPK, 8.0 * n, 0);
    select_collect_kernel<<<(unsigned)gh, SEL_HNT, SEL_CSMEM, ctx->stream>>>(scores, n, mk, num, st, ckey, cidx, idx_out);
    LRP_LAUNCHED(ctx);
    // fallback levels: enqueued always, a no-op unless st->fallback was set
    SelIn in{};
    in.scores = scores; in.n = n;
    if (bern) { in.bernoulli = 1; in.c_over_cols_c = bern->c; in.cols = (double)bern->cols; in.count = nullptr; in.x = mk.x; }
    int64_t G = g1;
    bool toA = true;
    for (int level = 0;; ++level) {
        const bool fin = G == 1;
        LRP_PROF(ctx, K_COND, 0.0, 0);
        select_sort_kernel<<<(unsigned)G, SEL_NT, SEL_SMEM, ctx->stream>>>(in, num, toA ? keyA : keyB, fin ? idx_out : (toA ? idxA : idxB), fin ? 1 : 0,
                                                                          &st->fallback);
        LRP_LAUNCHED(ctx);
        if (fin) break;
        in = SelIn{};
        in.ckey = toA ? keyA : keyB; in.cidx = toA ? idxA : idxB; in.m = G * num;
        G = sel_chunks(in.m);
        toA = !toA;
    }
    return LRP_OK;
}
