// common.cuh -- context, error plumbing and launch accounting shared by the liblrp translation units.
// (CUDA path only; shares nothing with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/lrp.h"

#include <vector>

// kernel classes for the per-kernel profile (lrp_profile_*): launch counts, CUDA-event time on the ctx's stream,
// and the ALGORITHMIC bytes / flops of the launches (what the step must move / compute).
enum LrpKernelId {
    K_DST_SMALL, K_DST_NAIVE, K_DST_FUSED, K_DST_BLUESTEIN,
    K_GEMM_SAMPLE, K_GEMM_PLAIN, K_GEMM_SUBTRACT, K_GEMM_T, K_REDUCE, K_ROWNORM, K_GATHER, K_COPY, K_ENTRIES,
    K_PANEL_QR, K_PANEL_APPLY, K_ADD_BLOCK, K_CORE, K_ETA, K_RHO, K_COLMASK, K_TOPK, K_RESID_GRAM, K_COND, K_DEIM, K_NUM
};
static const char* const LRP_KERNEL_NAMES[K_NUM] = {
    "dst1_small", "dst1_naive", "dst1_fused", "dst1_bluestein",
    "tall_gemm_sample", "tall_gemm_plain", "tall_gemm_subtract", "tall_gemm_t", "reduce_partials", "rownorm2", "gather_rows",
    "copy_tall", "lowrank_entries", "panel_qr", "panel_apply", "add_block", "scross_core", "eta", "rho", "colmask",
    "topk", "tall_resid_gram", "conditional_refactor", "deim_step"
};
struct lrp_prof { int64_t count; double ms, bytes, flops; };

constexpr size_t LRP_PINNED_BYTES = 65536;

struct lrp_ctx {
    int device;
    cudaStream_t stream;
    void* ws;
    size_t ws_bytes;
    int last_cuda;
    int64_t launches;
    int sm_count;
    int smem_optin;
    int flags;                            // lrp_solve_opts.flags of the solve in progress (LRP_FLAG_*), 0 otherwise
    int prof_on;
    int prof_pending;                     // kernel id whose start event is recorded, -1 if none
    lrp_prof prof[K_NUM];
    cudaStream_t aux;                     // library-owned second stream: independent sub-steps of a sweep overlap on it
    cudaStream_t aux2;                    // third stream: the one-CTA eta SVDs beside the two rho contractions
    cudaEvent_t ev_fork, ev_join, ev_join2;
    cudaStream_t hi[2];                   // high-priority streams (one per QR job): the small tree levels of the TSQR run here, so
    cudaEvent_t ev_hi[2][2];              // that they do not queue behind the other job's leaf CTAs; [job][to hi / back]
    unsigned* d_counters;                 // 3 x 65 arrival counters (one set per stream) of the in-kernel reductions; zero between launches
    double* pinned;                       // LRP_PINNED_BYTES of pinned host memory: target of the small read-backs of a sweep
    std::vector<cudaEvent_t>* ev;         // event pool: pairs (start, end)
    std::vector<int>* ev_id;
    size_t ev_used;
    std::vector<cudaEvent_t>* solve_ev;   // timing events of lrp_cross_deim_solve (created once, reused by every solve)
    int host_pipeline;                    // 1 while lrp_cross_deim_solve_host runs its solves: small copies avoid the copy engines
    lrp_ctx* lane2;                       // second solver lane of lrp_cross_deim_solve_host: library-owned context + its stream
    cudaStream_t lane2_stream;
    cudaStream_t cp_in, cp_out;           // copy streams of lrp_cross_deim_solve_host (created on its first call)
    cudaEvent_t ev_cp[2][2];              // [inputs arrived / outputs copied][staging slot]
};

// call right before a kernel launch: accounts the launch and, when profiling is on, records its start event
static inline void lrp_prof_begin(lrp_ctx* ctx, int id, double bytes, double flops) {
    ctx->prof[id].count++; ctx->prof[id].bytes += bytes; ctx->prof[id].flops += flops;
    if (!ctx->prof_on) return;
    if (ctx->ev_used + 2 > ctx->ev->size()) {
        cudaEvent_t a, b;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
        ctx->ev->push_back(a); ctx->ev->push_back(b);
    }
    cudaEventRecord((*ctx->ev)[ctx->ev_used], ctx->stream);
    ctx->ev_id->push_back(id);
    ctx->prof_pending = id;
}
static inline void lrp_prof_end(lrp_ctx* ctx) {
    if (ctx->prof_pending < 0) return;
    cudaEventRecord((*ctx->ev)[ctx->ev_used + 1], ctx->stream);
    ctx->ev_used += 2;
    ctx->prof_pending = -1;
}
#define LRP_PROF(ctx, id, bytes, flops) lrp_prof_begin((ctx), (id), (double)(bytes), (double)(flops))

#define LRP_CUDA(ctx, call)                                                      \
    do {                                                                         \
        cudaError_t e_ = (call);                                                 \
        if (e_ != cudaSuccess) { (ctx)->last_cuda = (int)e_; return LRP_ERR_CUDA; } \
    } while (0)

// after every kernel launch: count it and surface launch-configuration errors
#define LRP_LAUNCHED(ctx)                                                        \
    do {                                                                         \
        (ctx)->launches++;                                                       \
        lrp_prof_end(ctx);                                                       \
        cudaError_t e_ = cudaGetLastError();                                     \
        if (e_ != cudaSuccess) { (ctx)->last_cuda = (int)e_; return LRP_ERR_CUDA; } \
    } while (0)

#define LRP_TRY(expr)                                                            \
    do { int rc_ = (expr); if (rc_ < 0) return rc_; } while (0)

// SM count for grid sizing; without a ctx (host-side workspace sizing, no device query) an upper bound
constexpr int LRP_SM_UPPER = 192;
static inline int lrp_sm_count(const lrp_ctx* ctx) { return (ctx && ctx->sm_count > 0 && ctx->sm_count <= LRP_SM_UPPER) ? ctx->sm_count : LRP_SM_UPPER; }

static inline size_t lrp_align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

static inline int lrp_ilog2(int64_t x) { int p = 0; while ((int64_t(1) << p) < x) ++p; return p; }
static inline bool lrp_is_pow2(int64_t x) { return x > 0 && (x & (x - 1)) == 0; }

// bump allocator over the caller's workspace
struct lrp_arena {
    char* base; size_t cap; size_t off;
    lrp_arena(void* b, size_t c) : base((char*)b), cap(c), off(0) {}
    template <typename T> T* take(size_t count) {
        size_t bytes = lrp_align_up(count * sizeof(T));
        if (base == nullptr || off + bytes > cap) { off = cap + 1; return nullptr; }
        T* p = (T*)(base + off); off += bytes; return p;
    }
    bool ok() const { return off <= cap; }
};

// ---- internal entry points (defined across the .cu files) -------------------------------------------------
int lrp_dst1_impl(lrp_ctx* ctx, int64_t n, int32_t batch, const double* d_in, int64_t ld_in,
                  double* d_out, int64_t ld_out, double scale, void* ws, size_t ws_bytes);
size_t lrp_dst1_ws_impl(int64_t n, int32_t batch);
int lrp_dst1_init(lrp_ctx* ctx);      // one-time kernel attributes (lrp_create)
// four-step regime (dst1_large.cu), N = n + 1 > 16384
size_t dst1_large_ws(int64_t N, int32_t batch);
int dst1_large_init(lrp_ctx* ctx);
// general n (n + 1 not a power of two): Bluestein (dst1_bluestein.cu)
int dst1_bluestein_init(lrp_ctx* ctx);
bool dst1_bluestein_supported(int64_t n);
size_t dst1_bluestein_ws(int64_t n, int32_t batch);
int dst1_bluestein(lrp_ctx* ctx, int64_t n, int32_t batch, const double* d_in, int64_t ld_in, double* d_out, int64_t ld_out,
                   double scale, void* ws, size_t ws_bytes);
int dst1_large(lrp_ctx* ctx, int log2N, int32_t batch, const double* d_in, int64_t ld_in,
               double* d_out, int64_t ld_out, double scale, void* ws, size_t ws_bytes);
