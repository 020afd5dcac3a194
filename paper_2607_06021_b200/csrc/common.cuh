// common.cuh -- context, error plumbing and launch accounting shared by the liblrp translation units.
// (CUDA path only; shares nothing with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/lrp.h"

struct lrp_ctx {
    int device;
    cudaStream_t stream;
    void* ws;
    size_t ws_bytes;
    int last_cuda;
    int64_t launches;
    int sm_count;
    int smem_optin;
};

#define LRP_CUDA(ctx, call)                                                      \
    do {                                                                         \
        cudaError_t e_ = (call);                                                 \
        if (e_ != cudaSuccess) { (ctx)->last_cuda = (int)e_; return LRP_ERR_CUDA; } \
    } while (0)

// after every kernel launch: count it and surface launch-configuration errors
#define LRP_LAUNCHED(ctx)                                                        \
    do {                                                                         \
        (ctx)->launches++;                                                       \
        cudaError_t e_ = cudaGetLastError();                                     \
        if (e_ != cudaSuccess) { (ctx)->last_cuda = (int)e_; return LRP_ERR_CUDA; } \
    } while (0)

#define LRP_TRY(expr)                                                            \
    do { int rc_ = (expr); if (rc_ < 0) return rc_; } while (0)

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
