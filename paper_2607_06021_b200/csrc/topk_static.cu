// topk_static.cu -- lrp_topk_static: the deterministic top-k of select.cu (Alg. 3 line 6, reading Q5:
// the `num` largest scores ordered by (score descending, index ascending)) for callers that cannot allocate or hand over a
// workspace: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The candidate buffers
// that the multi-level sort of select.cu takes from the ctx workspace live here in ONE file-scope device array of fixed
// size, topk_scratch (TOPK_SCRATCH_BYTES = 1.6 MB), which every GPU that loads the library holds until the process exits.
//
//   * no cudaMalloc / cudaFree / allocating library call anywhere on this path; no ctx, no workspace;
//   * limits: n <= LRP_TOPK_STATIC_MAX_N (2^22), num <= LRP_TOPK_STATIC_MAX_NUM (256); beyond them LRP_ERR_STATIC_LIMIT;
//   * `topk_scratch` in HOST code is only a stand-in for the symbol: the device address comes from cudaGetSymbolAddress,
//     looked up once per device (with that device current) the first time the entry point runs there, and that pointer is
//     what the kernels get;
//   * every call shares the array and finds the previous call's contents in it.  Nothing has to start at zero: level l
//     writes all G_l * num candidate slots that level l + 1 reads, so stale pairs are never consumed (the test makes two
//     calls of different shape in a row).  Calls that overlap on the GPU (two streams, or two host threads) RACE on it:
//     serialise them.
// Same bitonic network on the same order-preserving 64-bit keys as select.cu, so the result is bit-identical to the
// workspace path (tests/test_zz_no_alloc.py).
#include "../../include/lrp.h"
#include <cuda_runtime.h>
#include <limits.h>
#include <mutex>

namespace {

constexpr int TS_NT = 1024;
constexpr int TS_CHUNK = 8192;
constexpr size_t TS_SMEM = (size_t)TS_CHUNK * (sizeof(unsigned long long) + sizeof(int));
constexpr unsigned long long TS_KEY_LAST = ~0ull;
constexpr int TS_MAX_DEV = 64;

constexpr int64_t ts_chunks(int64_t m) { return (m + TS_CHUNK - 1) / TS_CHUNK; }
// level-1 candidates: G1 * num pairs with G1 = MAX_N / CHUNK = 512; level-2: G2 * num with G2 = ceil(G1 * MAX_NUM / CHUNK) = 16
constexpr int64_t TS_CAP_A = ts_chunks(LRP_TOPK_STATIC_MAX_N) * LRP_TOPK_STATIC_MAX_NUM;
constexpr int64_t TS_CAP_B = ts_chunks(TS_CAP_A) * LRP_TOPK_STATIC_MAX_NUM;
constexpr size_t TS_OFF_KEY_A = 0;
constexpr size_t TS_OFF_KEY_B = TS_OFF_KEY_A + (size_t)TS_CAP_A * 8;
constexpr size_t TS_OFF_IDX_A = TS_OFF_KEY_B + (size_t)TS_CAP_B * 8;
constexpr size_t TS_OFF_IDX_B = TS_OFF_IDX_A + (size_t)TS_CAP_A * 4;
constexpr size_t TOPK_SCRATCH_BYTES = TS_OFF_IDX_B + (size_t)TS_CAP_B * 4;      // 1,622,016 bytes
static_assert(TS_OFF_KEY_B % 256 == 0 && TS_OFF_IDX_A % 256 == 0 && TS_OFF_IDX_B % 256 == 0, "sub-buffers stay aligned");

static __device__ __align__(256) unsigned char topk_scratch[TOPK_SCRATCH_BYTES];

__device__ __forceinline__ unsigned long long ts_desc_key(double s) {      // ascending key <=> descending score
    const unsigned long long b = (unsigned long long)__double_as_longlong(s);
    const unsigned long long asc = (b >> 63) ? ~b : (b | 0x8000000000000000ull);
    return ~asc;
}

// The CTA sorts its chunk of <= 8192 (key, index) pairs and emits the first `num`.  scores != nullptr: level 1 (raw scores,
// n of them); otherwise the candidate pairs of the previous level (m of them).  final_level: indices only, -1 if exhausted.
__global__ void __launch_bounds__(TS_NT)
topk_static_kernel(const double* __restrict__ scores, int64_t n, const unsigned long long* __restrict__ ckey,
                   const int32_t* __restrict__ cidx, int64_t m, int num, unsigned long long* __restrict__ okey,
                   int32_t* __restrict__ oidx, int final_level) {
    extern __shared__ __align__(16) unsigned char ts_raw[];
    unsigned long long* key = (unsigned long long*)ts_raw;
    int* idx = (int*)(key + TS_CHUNK);
    const int tid = threadIdx.x;
    const int64_t total = scores ? n : m;
    const int64_t b0 = (int64_t)blockIdx.x * TS_CHUNK;
    int64_t left = total - b0; if (left > TS_CHUNK) left = TS_CHUNK;
    const int cnt = (int)left;
    int N = 32; while (N < cnt) N <<= 1;
    for (int e = tid; e < N; e += TS_NT) {
        unsigned long long k = TS_KEY_LAST; int ix = INT_MAX;
        if (e < cnt) {
            if (scores) { k = ts_desc_key(scores[b0 + e]); ix = (int)(b0 + e); }
            else { k = ckey[b0 + e]; ix = cidx[b0 + e]; }
        }
        key[e] = k; idx[e] = ix;
    }
    __syncthreads();
    for (int k2 = 2; k2 <= N; k2 <<= 1) {
        for (int j = k2 >> 1; j > 0; j >>= 1) {
            for (int p = tid; p < N / 2; p += TS_NT) {
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
    for (int r = tid; r < num; r += TS_NT) {
        const bool have = r < N;
        const unsigned long long k = have ? key[r] : TS_KEY_LAST;
        const int ix = have ? idx[r] : INT_MAX;
        if (final_level) oidx[r] = (ix == INT_MAX) ? -1 : ix;
        else { okey[(int64_t)blockIdx.x * num + r] = k; oidx[(int64_t)blockIdx.x * num + r] = ix; }
    }
}

// per-device set-up: the device address of topk_scratch and the kernel's shared-memory opt-in
struct TsDevice { bool ready = false; unsigned char* base = nullptr; };
TsDevice g_dev[TS_MAX_DEV];
std::mutex g_mu;

int ts_setup(int dev, unsigned char** base) {
    std::lock_guard<std::mutex> lock(g_mu);
    TsDevice& d = g_dev[dev];
    if (!d.ready) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, topk_scratch) != cudaSuccess || !p) return LRP_ERR_CUDA;
        if (cudaFuncSetAttribute(topk_static_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TS_SMEM) != cudaSuccess)
            return LRP_ERR_CUDA;
        d.base = (unsigned char*)p;
        d.ready = true;
    }
    *base = d.base;
    return LRP_OK;
}

}  // namespace

extern "C" int lrp_topk_static(void* cuda_stream, int64_t n, const double* d_scores, int32_t num_select, int32_t* d_idx_out) {
    if (n < 1 || num_select < 0 || num_select > n || !d_scores || !d_idx_out || ((uintptr_t)d_scores & 7) ||
        ((uintptr_t)d_idx_out & 3))
        return LRP_ERR_BADARG;
    if (n > LRP_TOPK_STATIC_MAX_N || num_select > LRP_TOPK_STATIC_MAX_NUM) return LRP_ERR_STATIC_LIMIT;
    if (num_select == 0) return LRP_OK;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= TS_MAX_DEV) return LRP_ERR_CUDA;
    unsigned char* base = nullptr;
    const int rc = ts_setup(dev, &base);
    if (rc != LRP_OK) return rc;
    unsigned long long* keyA = (unsigned long long*)(base + TS_OFF_KEY_A);
    unsigned long long* keyB = (unsigned long long*)(base + TS_OFF_KEY_B);
    int32_t* idxA = (int32_t*)(base + TS_OFF_IDX_A);
    int32_t* idxB = (int32_t*)(base + TS_OFF_IDX_B);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const int num = num_select;
    // level 1 writes G1 * num <= CAP_A pairs into A; the levels after it ping-pong B, A, B, ... with at most CAP_B pairs
    int64_t G = ts_chunks(n);
    if (G * num > TS_CAP_A) return LRP_ERR_STATIC_LIMIT;                      // cannot happen within the limits above
    const double* sc = d_scores;
    const unsigned long long* ckey = nullptr; const int32_t* cidx = nullptr; int64_t m = 0;
    bool toA = true;
    for (;;) {
        const bool fin = G == 1;
        topk_static_kernel<<<(unsigned)G, TS_NT, TS_SMEM, stream>>>(sc, n, ckey, cidx, m, num, toA ? keyA : keyB,
                                                                   fin ? d_idx_out : (toA ? idxA : idxB), fin ? 1 : 0);
        if (cudaPeekAtLastError() != cudaSuccess) return LRP_ERR_CUDA;
        if (fin) break;
        sc = nullptr;
        ckey = toA ? keyA : keyB; cidx = toA ? idxA : idxB; m = G * num;
        G = ts_chunks(m);
        if (G * num > (toA ? TS_CAP_B : TS_CAP_A) && G != 1) return LRP_ERR_STATIC_LIMIT;
        toA = !toA;
    }
    return LRP_OK;
}
