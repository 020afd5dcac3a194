// api.cu -- the C ABI of include/lrp.h and the Cross-DEIM sweep driver (Alg. 4).
// Host control flow only decides sets of a few hundred integers and a handful of scalars per sweep
// (union / safeguard / prune / stop test); every step that touches an n-long axis is a kernel.
#include "common.cuh"
#include <cstdio>
#include "tall.cuh"
#include "qr.cuh"
#include "core.cuh"
#include <math.h>
#include <string.h>
#include <vector>
#include <algorithm>
#include <new>
#include <thread>

namespace {

// constants the paper is silent on (readings Q4, Q6, Q12)
constexpr double PINV_RCOND = 1e-13, RANK_RCOND = 1e-14, LEV_COL_RCOND = 1e-13, PRUNE_REL = 1e-12;

bool aligned8(const void* p) { return ((uintptr_t)p & 7u) == 0; }

// leading dimension of the library's own tall buffers: even (16-byte aligned columns -> 128-bit loads) and not a
// multiple of a large power of two (n + 1 is one: columns would alias in the memory-channel hash)
int64_t internal_ld(int64_t n) { return n + 74 + (n & 1); }

int check_n(int64_t n) {
    if (n < 1) return LRP_ERR_UNSUPPORTED_N;
    int64_t N = n + 1;
    if (lrp_is_pow2(N)) return N > ((int64_t)1 << 25) ? LRP_ERR_UNSUPPORTED_N : LRP_OK;
    return dst1_bluestein_supported(n) ? LRP_OK : LRP_ERR_UNSUPPORTED_N;      // general n: Bluestein, n + 1 <= 2^23
}

// ------------------------------------------------------------------------------------------------ small copies of a sweep
// The read-backs (a few KB into ctx->pinned) and uploads (index lists, 32 x 32 factors) of a sweep normally go through
// cudaMemcpyAsync.  Inside lrp_cross_deim_solve_host the copy engines are busy with the neighbouring problems' factors
// (hundreds of MB, submitted earlier, served first), so there (ctx->host_pipeline) a read-back is a one-CTA kernel that
// writes through the device alias of the pinned buffer and an upload travels as kernel parameters.
constexpr int SMALL_UP_WORDS = 960;                                  // 3840 bytes of payload per launch (parameter space: 4 KB)
struct SmallPayload { uint32_t w[SMALL_UP_WORDS]; };
__global__ void __launch_bounds__(256) small_upload_kernel(uint32_t* __restrict__ dst, int nwords, const SmallPayload pl) {
    for (int i = threadIdx.x; i < nwords; i += blockDim.x) dst[i] = pl.w[i];
}
__global__ void __launch_bounds__(256) small_readback_kernel(uint32_t* __restrict__ host_alias, const uint32_t* __restrict__ src, int nwords) {
    for (int i = threadIdx.x; i < nwords; i += blockDim.x) host_alias[i] = src[i];
}
cudaError_t d2h_small(lrp_ctx* ctx, void* h, const void* d, size_t bytes, cudaStream_t s) {
    const char* pb = (const char*)ctx->pinned;
    if (ctx->host_pipeline && (bytes & 3) == 0 && bytes <= LRP_PINNED_BYTES && (const char*)h >= pb && (const char*)h + bytes <= pb + LRP_PINNED_BYTES) {
        small_readback_kernel<<<1, 256, 0, s>>>((uint32_t*)h, (const uint32_t*)d, (int)(bytes / 4));   // cudaHostAlloc memory: same address on the device (UVA)
        ctx->launches++;
        return cudaGetLastError();
    }
    return cudaMemcpyAsync(h, d, bytes, cudaMemcpyDeviceToHost, s);
}
cudaError_t h2d_small(lrp_ctx* ctx, void* d, const void* h, size_t bytes, cudaStream_t s) {
    if (ctx->host_pipeline && (bytes & 3) == 0 && bytes <= 65536) {
        for (size_t o = 0; o < bytes; o += sizeof(SmallPayload)) {
            const size_t len = bytes - o < sizeof(SmallPayload) ? bytes - o : sizeof(SmallPayload);
            SmallPayload pl;
            memcpy(pl.w, (const char*)h + o, len);
            small_upload_kernel<<<1, 256, 0, s>>>((uint32_t*)((char*)d + o), (int)(len / 4), pl);
            ctx->launches++;
        }
        return cudaGetLastError();
    }
    return cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, s);
}

// ------------------------------------------------------------------------------------------------ scross on owned buffers
struct ScrossWs {
    double *RC, *RR, *Uc, *S, *Vc, *rC, *rR, *scal_d, *core_work, *qr_ws, *qr_ws2;
    int32_t *scal_i, *iwork;
    int ldrc, ldrr;               // leading dimensions of RC / RR: fixed (kmax / lmax), so that a factor survives a change of k
    int Kblk;
    bool carve(lrp_arena& ar, const lrp_ctx* ctx, int64_t n, int kmax, int lmax) {
        int K = kmax > lmax ? kmax : lmax;
        ldrc = kmax; ldrr = lmax;
        RC = ar.take<double>((size_t)kmax * kmax); RR = ar.take<double>((size_t)lmax * lmax);
        Uc = ar.take<double>((size_t)K * K); Vc = ar.take<double>((size_t)K * K);
        // what the host reads after the core, in one block (one copy into pinned memory): S | rC | rR | scal_d | scal_i
        Kblk = K;
        double* rb = ar.take<double>(3 * (size_t)K + 8);
        S = rb; rC = rb + K; rR = rb + 2 * (size_t)K; scal_d = rb + 3 * (size_t)K; scal_i = (int32_t*)(scal_d + 4);
        iwork = ar.take<int32_t>(K);
        core_work = ar.take<double>(core_work_doubles(K, K));
        qr_ws = ar.take<double>(tall_qr_ws_doubles(ctx, n, K));
        qr_ws2 = ar.take<double>(tall_qr_ws_doubles(ctx, n, K));
        return ar.ok();
    }
};

// QR of both fiber blocks (in place), the small core, and the host copies the driver needs.
// On return (stream synchronised): Qb = Q, Zb = Z, ws.Uc/S/Vc hold the core SVD, h_S (p), h_rC (k), h_rR (l) filled.
// k0 / l0: leading columns of Qb / Zb that already hold the Q factor of the same fibers (with their block of RC / RR
// in place) from the previous call: the fibers of surviving indices do not change between sweeps.
int scross_factor(lrp_ctx* ctx, int64_t n, double* Qb, int64_t ldq, int k, int k0, double* Zb, int64_t ldz, int l, int l0,
                  const int32_t* dI, const int32_t* dJ, ScrossWs& w,
                  double* h_S, double* h_rC, double* h_rR, int* h_rank, double* h_smin,
                  cudaEvent_t ev_qr_done) {
    LRP_TRY(tall_qr_pair_from(ctx, n, k, k0, Qb, ldq, w.RC, w.ldrc, w.qr_ws, l, l0, Zb, ldz, w.RR, w.ldrr, w.qr_ws2));
    if (ev_qr_done) LRP_CUDA(ctx, cudaEventRecord(ev_qr_done, ctx->stream));
    CoreArgs a{};
    a.k = k; a.l = l; a.Q = Qb; a.ldq = ldq; a.Z = Zb; a.ldz = ldz; a.RC = w.RC; a.ldrc = w.ldrc; a.RR = w.RR; a.ldrr = w.ldrr;
    a.I = dI; a.J = dJ; a.pinv_rcond = PINV_RCOND; a.rank_rcond = RANK_RCOND;
    a.Uc = w.Uc; a.S = w.S; a.Vc = w.Vc; a.rC = w.rC; a.rR = w.rR; a.scal_i = w.scal_i; a.scal_d = w.scal_d;
    a.work = w.core_work; a.iwork = w.iwork;
    LRP_TRY(scross_core(ctx, a));
    const int p = k < l ? k : l;
    const size_t blk = (3 * (size_t)w.Kblk + 8) * sizeof(double);
    std::vector<double> pageable;
    double* hb = ctx->pinned;
    if (blk > LRP_PINNED_BYTES) { pageable.resize(blk / sizeof(double)); hb = pageable.data(); }
    LRP_CUDA(ctx, d2h_small(ctx, hb, w.S, blk, ctx->stream));
    LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    memcpy(h_S, hb, sizeof(double) * p);
    memcpy(h_rC, hb + w.Kblk, sizeof(double) * k);
    memcpy(h_rR, hb + 2 * (size_t)w.Kblk, sizeof(double) * l);
    *h_smin = hb[3 * (size_t)w.Kblk];
    int32_t hi; memcpy(&hi, hb + 3 * (size_t)w.Kblk + 4, sizeof(int32_t));
    *h_rank = hi;
    return LRP_OK;
}

// U = Q Uc(:, 0:rank) (n x rank) with optional squared row norms (the next sweep's leverage scores)
int rebuild(lrp_ctx* ctx, int64_t n, const double* Qf, int64_t ldq, int kk, const double* Uc, int ldc, int rank,
            double* U, int64_t ldu, double* rownorm2) {
    TallGemmArgs g{};
    g.n = n; g.k = kk; g.m = rank; g.mode = TG_PLAIN; g.A = Qf; g.lda = ldq; g.B = Uc; g.ldb = ldc;
    g.Out = U; g.ldo = ldu; g.rownorm2 = rownorm2;
    return tall_gemm(ctx, g);
}

int sample_side(lrp_ctx* ctx, int64_t n, int r, const double* A, int64_t lda, const double* S, const double* Bt, int64_t ldb,
                const int32_t* idx, int nidx, double* Out, int64_t ldo) {
    TallGemmArgs g{};
    g.n = n; g.k = r; g.m = nidx; g.mode = TG_SAMPLE; g.A = A; g.lda = lda; g.B = Bt; g.ldb = ldb; g.idx = idx; g.scale_t = S;
    g.Out = Out; g.ldo = ldo;
    return tall_gemm(ctx, g);
}

// leverage scores of a tall block through a scratch copy (QR in place on the copy)
int leverage_scores_qr(lrp_ctx* ctx, int64_t n, int k, const double* A, int64_t lda, double* scratch, int64_t lds,
                       double* R, unsigned char* mask, double* qr_ws, double* scores) {
    LRP_TRY(tall_copy(ctx, n, k, A, lda, scratch, lds));
    LRP_TRY(tall_qr(ctx, n, k, scratch, lds, R, k, qr_ws));
    LRP_TRY(leverage_colmask(ctx, k, R, k, LEV_COL_RCOND, mask));
    return tall_rownorm2(ctx, n, k, scratch, lds, mask, scores);
}

int validate_indices(const int32_t* h, int cnt, int64_t n) {
    std::vector<int32_t> v(h, h + cnt);
    std::sort(v.begin(), v.end());
    for (int i = 0; i < cnt; ++i) {
        if (v[i] < 0 || v[i] >= n) return LRP_ERR_BADARG;
        if (i > 0 && v[i] == v[i - 1]) return LRP_ERR_BADARG;
    }
    return LRP_OK;
}

// ------------------------------------------------------------------------------------------------ solve workspace
constexpr int NREST_MAX = 16;      // dropped trailing Q columns of the previous fiber block kept aside for the nested stop test
struct SolveWs {
    double *UhF, *VhF, *Cb, *Rb, *Ua, *Va, *Ub, *Vb, *scoresU, *scoresV;
    double *UcPrev, *VcPrev, *nestU, *nestV;      // previous core factors and scratch of the nested stop test
    double *QrestU, *QrestV, *TU, *TV, *GpU, *GpV;   // dropped trailing Q columns (n x NREST_MAX), T = Q^T Q_rest, P^T P
    double *Sprev, *Amat, *Bmat, *GU, *GV, *rho_out, *eta, *eta_work, *gemmt_ws, *gemmt_ws2, *Rlev, *Rlev2;
    int32_t *dI, *dJ, *dIpr, *dJpr, *dIstar, *dJstar, *eta_iwork;
    unsigned char *mask, *mask2;
    void *sel_ws, *dst_ws, *dst_ws2, *deim_ws;
    size_t eta_stride, dst_ws_bytes;
    ScrossWs sc;
    bool carve(lrp_arena& ar, const lrp_ctx* ctx, int64_t n, int rF, int Kc, int max_rank, bool poisson = true) {
        const size_t ld = (size_t)internal_ld(n);
        UhF = ar.take<double>(poisson ? ld * rF : 1); VhF = ar.take<double>(poisson ? ld * rF : 1);
        Cb = ar.take<double>(ld * Kc); Rb = ar.take<double>(ld * Kc);
        Ua = ar.take<double>(ld * Kc); Va = ar.take<double>(ld * Kc);
        Ub = ar.take<double>(ld * Kc); Vb = ar.take<double>(ld * Kc);
        scoresU = ar.take<double>(ld); scoresV = ar.take<double>(ld);
        Sprev = ar.take<double>(Kc);
        Amat = ar.take<double>((size_t)Kc * Kc); Bmat = ar.take<double>((size_t)Kc * Kc);
        GU = ar.take<double>((size_t)Kc * Kc); GV = ar.take<double>((size_t)Kc * Kc);
        Rlev = ar.take<double>((size_t)Kc * Kc); Rlev2 = ar.take<double>((size_t)Kc * Kc);
        UcPrev = ar.take<double>((size_t)Kc * Kc); VcPrev = ar.take<double>((size_t)Kc * Kc);
        nestU = ar.take<double>(2 * (size_t)Kc * Kc); nestV = ar.take<double>(2 * (size_t)Kc * Kc);
        QrestU = ar.take<double>(ld * NREST_MAX); QrestV = ar.take<double>(ld * NREST_MAX);
        TU = ar.take<double>((size_t)Kc * NREST_MAX); TV = ar.take<double>((size_t)Kc * NREST_MAX);
        GpU = ar.take<double>(NREST_MAX * NREST_MAX); GpV = ar.take<double>(NREST_MAX * NREST_MAX);
        rho_out = ar.take<double>(16 + RHO_MAX_GRID + 2); eta = rho_out + 8;      // [rho, snorm | eta1, eta2] read back together; partial sums and ticket of rho_kernel behind them
        eta_stride = lrp_align_up(eta_work_doubles(Kc, Kc) * sizeof(double)) / sizeof(double);
        eta_work = ar.take<double>(2 * eta_stride);
        eta_iwork = ar.take<int32_t>(2 * (size_t)Kc);
        gemmt_ws = ar.take<double>(tall_gemm_t_ws_doubles(ctx, n, Kc, Kc));
        gemmt_ws2 = ar.take<double>(tall_gemm_t_ws_doubles(ctx, n, Kc, Kc));
        dI = ar.take<int32_t>(Kc); dJ = ar.take<int32_t>(Kc); dIpr = ar.take<int32_t>(Kc); dJpr = ar.take<int32_t>(Kc);
        dIstar = ar.take<int32_t>(2 * (size_t)Kc + 8); dJstar = ar.take<int32_t>(2 * (size_t)Kc + 8);
        mask = ar.take<unsigned char>(Kc); mask2 = ar.take<unsigned char>(Kc);
        sel_ws = ar.take<char>(select_ws_bytes(ctx, n, 2 * Kc + 1));
        deim_ws = ar.take<char>(deim_ws_bytes(n, Kc));
        int dcols = rF > max_rank ? rF : max_rank;
        dst_ws_bytes = poisson ? lrp_dst1_ws_impl(n, dcols) : 0;
        dst_ws = ar.take<char>(dst_ws_bytes ? dst_ws_bytes : 1);
        dst_ws2 = ar.take<char>(dst_ws_bytes ? dst_ws_bytes : 1);
        bool ok = sc.carve(ar, ctx, n, Kc, Kc);
        return ok && ar.ok();
    }
};

// timing events of a solve: owned by the ctx and created once (the first solves grow the pool, later ones reuse it)
struct EventPool {
    lrp_ctx* ctx; size_t used;
    explicit EventPool(lrp_ctx* c) : ctx(c), used(0) {}
    cudaEvent_t take() {
        if (used == ctx->solve_ev->size()) {
            cudaEvent_t e; if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
            ctx->solve_ev->push_back(e);
        }
        return (*ctx->solve_ev)[used++];
    }
    cudaEvent_t rec(lrp_ctx* c) { cudaEvent_t e = take(); if (e) cudaEventRecord(e, c->stream); return e; }
    static float ms(cudaEvent_t a, cudaEvent_t b) { float t = 0.f; if (a && b) cudaEventElapsedTime(&t, a, b); return t; }
};

struct FlagsGuard {                   // lrp_solve_opts.flags are visible to the kernels' host wrappers during one solve
    lrp_ctx* ctx;
    FlagsGuard(lrp_ctx* c, int f) : ctx(c) { c->flags = f; }
    ~FlagsGuard() { ctx->flags = 0; }
};

// Run `expr` (helpers launch on ctx->stream) on another stream.
#define LRP_ON_STREAM(ctx, strm, expr)                                          \
    do { cudaStream_t m_ = (ctx)->stream; (ctx)->stream = (strm); int rc2_ = (expr); (ctx)->stream = m_; if (rc2_ < 0) return rc2_; } while (0)

// Upper-triangular Cholesky factor of the c x c Gram matrix G (column-major, G = R^T R) and its inverse, on the host.
// false when a pivot loses more than 10 digits (kappa(A) beyond ~1e5: the caller takes the Householder QR instead).
static bool host_chol_inverse(const std::vector<double>& G, int c, std::vector<double>& Rinv) {
    std::vector<double> R((size_t)c * c, 0.0);
    for (int j = 0; j < c; ++j) {
        for (int i = 0; i <= j; ++i) {
            double acc = G[i + (size_t)j * c];
            for (int t = 0; t < i; ++t) acc -= R[t + (size_t)i * c] * R[t + (size_t)j * c];
            if (i < j) R[i + (size_t)j * c] = acc / R[i + (size_t)i * c];
            else {
                if (!(acc > 1e-10 * G[j + (size_t)j * c]) || !(G[j + (size_t)j * c] > 0.0)) return false;
                R[j + (size_t)j * c] = std::sqrt(acc);
            }
        }
    }
    Rinv.assign((size_t)c * c, 0.0);
    for (int j = 0; j < c; ++j) {                       // R X = I, column by column (X upper triangular)
        Rinv[j + (size_t)j * c] = 1.0 / R[j + (size_t)j * c];
        for (int i = j - 1; i >= 0; --i) {
            double acc = 0.0;
            for (int t = i + 1; t <= j; ++t) acc -= R[i + (size_t)t * c] * Rinv[t + (size_t)j * c];
            Rinv[i + (size_t)j * c] = acc / R[i + (size_t)i * c];
        }
    }
    return true;
}

void host_union(std::vector<int32_t>& cur, const int32_t* star, int nstar, int* added) {
    *added = 0;
    for (int i = 0; i < nstar; ++i) {
        int32_t v = star[i];
        if (v < 0) continue;
        if (std::find(cur.begin(), cur.end(), v) == cur.end()) { cur.push_back(v); ++*added; }
    }
}

// Alg. 4 lines 30-31: r* = smallest r with sum_{c>r} S_c^2 < eps^2 (x sum S^2, reading Q15); returns
// r = max(min(r*, r_max), 1) and r* itself through rstar_out (r* > r_max: the tolerance is not met, reading Q20).
int final_rank_host(const double* S, int cnt, double tol, int max_rank, int tol_mode, int* rstar_out) {
    double tot = 0.0;
    for (int c = 0; c < cnt; ++c) tot += S[c] * S[c];
    const double thresh = tol * tol * (tol_mode == 0 ? tot : 1.0);
    int rstar = cnt; double tail = 0.0;
    for (int c = cnt - 1; c >= 0; --c) { tail += S[c] * S[c]; if (tail < thresh) rstar = c; else break; }
    *rstar_out = rstar;
    int r = rstar < max_rank ? rstar : max_rank;
    return r < 1 ? 1 : r;
}

}  // namespace

// ================================================================================================ C ABI
extern "C" {

int lrp_create(lrp_ctx** out, int device, void* cuda_stream) {
    if (!out) return LRP_ERR_BADARG;
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || device < 0 || device >= count) return LRP_ERR_CUDA;
    if (cudaSetDevice(device) != cudaSuccess) return LRP_ERR_CUDA;
    lrp_ctx* c = new (std::nothrow) lrp_ctx();
    if (!c) return LRP_ERR_BADARG;
    c->device = device; c->stream = (cudaStream_t)cuda_stream; c->ws = nullptr; c->ws_bytes = 0; c->last_cuda = 0; c->launches = 0;
    c->prof_on = 0; c->prof_pending = -1; memset(c->prof, 0, sizeof(c->prof));
    c->ev = new std::vector<cudaEvent_t>(); c->ev_id = new std::vector<int>(); c->ev_used = 0;
    c->flags = 0; c->solve_ev = new std::vector<cudaEvent_t>();
    for (int q = 0; q < 2; ++q) { c->hi[q] = nullptr; c->ev_hi[q][0] = nullptr; c->ev_hi[q][1] = nullptr; }
    c->cp_in = nullptr; c->cp_out = nullptr; c->host_pipeline = 0; c->lane2 = nullptr; c->lane2_stream = nullptr;
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) c->ev_cp[a][b] = nullptr;
    c->aux = nullptr; c->aux2 = nullptr; c->ev_fork = nullptr; c->ev_join = nullptr; c->ev_join2 = nullptr; c->pinned = nullptr; c->d_counters = nullptr;
    if (cudaStreamCreateWithFlags(&c->aux, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&c->aux2, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join2, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess ||
        cudaHostAlloc((void**)&c->pinned, LRP_PINNED_BYTES, cudaHostAllocDefault) != cudaSuccess ||
        cudaMalloc((void**)&c->d_counters, 3 * 65 * sizeof(unsigned)) != cudaSuccess ||
        cudaMemset(c->d_counters, 0, 3 * 65 * sizeof(unsigned)) != cudaSuccess) { lrp_destroy(c); return LRP_ERR_CUDA; }
    {
        int lo = 0, hiprio = 0;
        cudaDeviceGetStreamPriorityRange(&lo, &hiprio);
        for (int q = 0; q < 2; ++q)
            if (cudaStreamCreateWithPriority(&c->hi[q], cudaStreamNonBlocking, hiprio) != cudaSuccess ||
                cudaEventCreateWithFlags(&c->ev_hi[q][0], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&c->ev_hi[q][1], cudaEventDisableTiming) != cudaSuccess) { lrp_destroy(c); return LRP_ERR_CUDA; }
    }
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
    cudaDeviceGetAttribute(&c->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    // one-time kernel attributes (dynamic shared memory opt-in): not on the per-call path
    if (tall_qr_init(c) != LRP_OK || lrp_dst1_init(c) != LRP_OK || select_init(c) != LRP_OK || core_init(c) != LRP_OK || tall_mma_init(c) != LRP_OK) { lrp_destroy(c); return LRP_ERR_CUDA; }
    *out = c;
    return LRP_OK;
}

int lrp_destroy(lrp_ctx* ctx) {
    if (!ctx) return LRP_OK;
    if (ctx->ev) { for (auto e : *ctx->ev) cudaEventDestroy(e); delete ctx->ev; }
    if (ctx->solve_ev) { for (auto e : *ctx->solve_ev) cudaEventDestroy(e); delete ctx->solve_ev; }
    if (ctx->d_counters) cudaFree(ctx->d_counters);
    for (int q = 0; q < 2; ++q) {
        if (ctx->hi[q]) cudaStreamDestroy(ctx->hi[q]);
        if (ctx->ev_hi[q][0]) cudaEventDestroy(ctx->ev_hi[q][0]);
        if (ctx->ev_hi[q][1]) cudaEventDestroy(ctx->ev_hi[q][1]);
    }
    if (ctx->lane2) { lrp_destroy(ctx->lane2); ctx->lane2 = nullptr; }
    if (ctx->lane2_stream) cudaStreamDestroy(ctx->lane2_stream);
    if (ctx->cp_in) cudaStreamDestroy(ctx->cp_in);
    if (ctx->cp_out) cudaStreamDestroy(ctx->cp_out);
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) if (ctx->ev_cp[a][b]) cudaEventDestroy(ctx->ev_cp[a][b]);
    if (ctx->aux) cudaStreamDestroy(ctx->aux);
    if (ctx->aux2) cudaStreamDestroy(ctx->aux2);
    if (ctx->ev_join2) cudaEventDestroy(ctx->ev_join2);
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    if (ctx->pinned) cudaFreeHost(ctx->pinned);
    delete ctx->ev_id;
    delete ctx;
    return LRP_OK;
}

int lrp_profile_enable(lrp_ctx* ctx, int on) {
    if (!ctx) return LRP_ERR_BADARG;
    ctx->prof_on = on == 2 ? 2 : (on ? 1 : 0);           // 1: serial streams, clean per-kernel times; 2: timeline of the real run
    return LRP_OK;
}

int lrp_profile_timeline(lrp_ctx* ctx, const char* path) {
    if (!ctx || !path) return LRP_ERR_BADARG;
    LRP_CUDA(ctx, cudaDeviceSynchronize());
    FILE* f = fopen(path, "w");
    if (!f) return LRP_ERR_BADARG;
    fprintf(f, "kernel,start_ms,end_ms\n");
    for (size_t i = 0; i + 1 < ctx->ev_used; i += 2) {
        float t0 = 0.f, t1 = 0.f;
        if (cudaEventElapsedTime(&t0, (*ctx->ev)[0], (*ctx->ev)[i]) == cudaSuccess &&
            cudaEventElapsedTime(&t1, (*ctx->ev)[0], (*ctx->ev)[i + 1]) == cudaSuccess)
            fprintf(f, "%s,%.4f,%.4f\n", LRP_KERNEL_NAMES[(*ctx->ev_id)[i / 2]], t0, t1);
    }
    fclose(f);
    return LRP_OK;
}

static int profile_collect(lrp_ctx* ctx) {
    LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (size_t i = 0; i + 1 < ctx->ev_used; i += 2) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, (*ctx->ev)[i], (*ctx->ev)[i + 1]) == cudaSuccess) ctx->prof[(*ctx->ev_id)[i / 2]].ms += t;
    }
    ctx->ev_used = 0; ctx->ev_id->clear();
    return LRP_OK;
}

int lrp_profile_reset(lrp_ctx* ctx) {
    if (!ctx) return LRP_ERR_BADARG;
    LRP_TRY(profile_collect(ctx));
    memset(ctx->prof, 0, sizeof(ctx->prof));
    return LRP_OK;
}

int lrp_profile_count(void) { return (int)K_NUM; }

int lrp_profile_get(lrp_ctx* ctx, int i, const char** name, int64_t* count, double* ms, double* bytes, double* flops) {
    if (!ctx || i < 0 || i >= (int)K_NUM) return LRP_ERR_BADARG;
    LRP_TRY(profile_collect(ctx));
    if (name) *name = LRP_KERNEL_NAMES[i];
    if (count) *count = ctx->prof[i].count;
    if (ms) *ms = ctx->prof[i].ms;
    if (bytes) *bytes = ctx->prof[i].bytes;
    if (flops) *flops = ctx->prof[i].flops;
    return LRP_OK;
}

const char* lrp_strerror(int code) {
    switch (code) {
        case LRP_OK: return "ok";
        case LRP_ERR_BADARG: return "bad argument";
        case LRP_ERR_UNSUPPORTED_N: return "n out of range: n + 1 a power of two <= 2^25, or any n + 1 <= 2^23";
        case LRP_ERR_WORKSPACE: return "workspace missing or too small";
        case LRP_ERR_CUDA: return "CUDA error (see lrp_last_cuda_error)";
        case LRP_ERR_STATIC_LIMIT: return "size beyond the fixed capacity of the built-in scratch (n <= 4194304, num_select <= 256)";
        case LRP_WARN_NOCONV: return "warning: stop test not passed within max_sweeps";
        default: return "unknown code";
    }
}

int lrp_last_cuda_error(const lrp_ctx* ctx) { return ctx ? ctx->last_cuda : 0; }
int64_t lrp_launch_count(const lrp_ctx* ctx) { return ctx ? ctx->launches : 0; }

int lrp_set_workspace(lrp_ctx* ctx, void* d_ws, size_t bytes) {
    if (!ctx) return LRP_ERR_BADARG;
    if (d_ws && ((uintptr_t)d_ws & 255u)) return LRP_ERR_BADARG;
    ctx->ws = d_ws; ctx->ws_bytes = d_ws ? bytes : 0;
    return LRP_OK;
}

size_t lrp_dst1_workspace_bytes(int64_t n, int32_t batch) {
    if (check_n(n) != LRP_OK || batch < 0) return 0;
    return lrp_dst1_ws_impl(n, batch);
}

size_t lrp_workspace_bytes(int64_t n, int32_t rF, int32_t max_rank, int32_t oversample) {
    if (check_n(n) != LRP_OK || rF < 1 || max_rank < 1 || oversample < 0) return 0;
    const int Kc = 2 * (max_rank + oversample);       // reading Q10; the first sweep needs rF + oversample + 1 <= K_cap
    if (Kc < rF + oversample + 1) return 0;
    lrp_arena ar((void*)256, (size_t)-1 / 2);
    SolveWs w;
    w.carve(ar, nullptr, n, rF, Kc, max_rank);
    return ar.off + 256;
}

size_t lrp_matrix_workspace_bytes(int64_t n, int32_t r0, int32_t max_rank, int32_t oversample) {
    if (n < 2 || r0 < 1 || max_rank < 1 || oversample < 0) return 0;
    const int Kc = 2 * (max_rank + oversample);
    if (Kc < r0 + oversample + 1) return 0;
    lrp_arena ar((void*)256, (size_t)-1 / 2);
    SolveWs w;
    w.carve(ar, nullptr, n, r0, Kc, max_rank, false);
    return ar.off + 256;
}

size_t lrp_leverage_workspace_bytes(int64_t n, int32_t k) {
    if (n < 1 || k < 1) return 0;
    lrp_arena ar((void*)256, (size_t)-1 / 2);
    ar.take<double>((size_t)n * k); ar.take<double>((size_t)k * k); ar.take<double>((size_t)n);
    ar.take<unsigned char>(k); ar.take<double>(tall_qr_ws_doubles(nullptr, n, k));
    ar.take<char>(select_ws_bytes(nullptr, n, 4096));
    return ar.off + 256;
}

size_t lrp_scross_workspace_bytes(int64_t n, int32_t k, int32_t l) {
    if (n < 1 || k < 1 || l < 1) return 0;
    lrp_arena ar((void*)256, (size_t)-1 / 2);
    ar.take<double>((size_t)n * k); ar.take<double>((size_t)n * l);
    ScrossWs w; w.carve(ar, nullptr, n, k, l);
    return ar.off + 256;
}

int lrp_dst1_batched(lrp_ctx* ctx, int64_t n, int32_t batch, const double* d_in, int64_t ld_in,
                     double* d_out, int64_t ld_out, double scale) {
    if (!ctx) return LRP_ERR_BADARG;
    LRP_TRY(check_n(n));
    if (batch < 0) return LRP_ERR_BADARG;
    if (batch == 0) return LRP_OK;
    if (!d_in || !d_out || !aligned8(d_in) || !aligned8(d_out) || ld_in < n || ld_out < n) return LRP_ERR_BADARG;
    if (d_in == d_out && ld_in != ld_out) return LRP_ERR_BADARG;
    return lrp_dst1_impl(ctx, n, batch, d_in, ld_in, d_out, ld_out, scale, ctx->ws, ctx->ws_bytes);
}

int lrp_sample_fibers(lrp_ctx* ctx, int64_t n, int32_t r, const double* d_Uh, int64_t ldu, const double* d_S,
                      const double* d_Vh, int64_t ldv, const int32_t* d_I, int32_t nI, const int32_t* d_J, int32_t nJ,
                      double* d_C, int64_t ldc, double* d_Rt, int64_t ldr) {
    if (!ctx || n < 1 || r < 1 || r > 1024 || !d_Uh || !d_S || !d_Vh || ldu < n || ldv < n) return LRP_ERR_BADARG;
    if (nI < 0 || nJ < 0) return LRP_ERR_BADARG;
    if (d_C && nJ > 0) {
        if (!d_J || ldc < n) return LRP_ERR_BADARG;
        LRP_TRY(sample_side(ctx, n, r, d_Uh, ldu, d_S, d_Vh, ldv, d_J, nJ, d_C, ldc));
    }
    if (d_Rt && nI > 0) {
        if (!d_I || ldr < n) return LRP_ERR_BADARG;
        LRP_TRY(sample_side(ctx, n, r, d_Vh, ldv, d_S, d_Uh, ldu, d_I, nI, d_Rt, ldr));
    }
    return LRP_OK;
}

int lrp_leverage_select(lrp_ctx* ctx, int64_t n, int32_t k, const double* d_A, int64_t lda,
                        int32_t num_select, int assume_orthonormal, int32_t* d_idx_out, double* d_scores) {
    if (!ctx || n < 1 || k < 1 || k > 1024 || !d_A || lda < n || !d_idx_out) return LRP_ERR_BADARG;
    if (num_select < 0 || num_select > n || num_select > 4096 || (!assume_orthonormal && k > n)) return LRP_ERR_BADARG;
    if (ctx->ws_bytes < lrp_leverage_workspace_bytes(n, k)) return LRP_ERR_WORKSPACE;
    lrp_arena ar(ctx->ws, ctx->ws_bytes);
    double* scratch = ar.take<double>((size_t)n * k);
    double* R = ar.take<double>((size_t)k * k);
    double* scores = ar.take<double>((size_t)n);
    unsigned char* mask = ar.take<unsigned char>(k);
    double* qr_ws = ar.take<double>(tall_qr_ws_doubles(ctx, n, k));
    void* sel_ws = ar.take<char>(select_ws_bytes(ctx, n, 4096));
    if (!ar.ok()) return LRP_ERR_WORKSPACE;
    double* sc = d_scores ? d_scores : scores;
    if (assume_orthonormal) LRP_TRY(tall_rownorm2(ctx, n, k, d_A, lda, nullptr, sc));
    else LRP_TRY(leverage_scores_qr(ctx, n, k, d_A, lda, scratch, n, R, mask, qr_ws, sc));
    LRP_TRY(select_topk(ctx, n, sc, num_select, d_idx_out, sel_ws));
    LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return LRP_OK;
}

int lrp_scross(lrp_ctx* ctx, int64_t n, const double* d_C, int64_t ldc, int32_t k, const double* d_Rt, int64_t ldr, int32_t l,
               const int32_t* d_I, const int32_t* d_J, double* d_U, int64_t ldu, double* d_S, double* d_V, int64_t ldv,
               double* d_rC, double* d_rR, int32_t* h_rank_out, double* h_smin_full_out) {
    if (!ctx || n < 1 || k < 1 || l < 1 || k > 1024 || l > 1024 || k > n || l > n) return LRP_ERR_BADARG;
    if (!d_C || !d_Rt || !d_I || !d_J || !d_U || !d_S || !d_V || ldc < n || ldr < n || ldu < n || ldv < n) return LRP_ERR_BADARG;
    if (ctx->ws_bytes < lrp_scross_workspace_bytes(n, k, l)) return LRP_ERR_WORKSPACE;
    {   // index validation (host copy)
        std::vector<int32_t> hI(l), hJ(k);
        LRP_CUDA(ctx, cudaMemcpyAsync(hI.data(), d_I, sizeof(int32_t) * l, cudaMemcpyDeviceToHost, ctx->stream));
        LRP_CUDA(ctx, cudaMemcpyAsync(hJ.data(), d_J, sizeof(int32_t) * k, cudaMemcpyDeviceToHost, ctx->stream));
        LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        LRP_TRY(validate_indices(hI.data(), l, n));
        LRP_TRY(validate_indices(hJ.data(), k, n));
    }
    lrp_arena ar(ctx->ws, ctx->ws_bytes);
    double* Qb = ar.take<double>((size_t)n * k);
    double* Zb = ar.take<double>((size_t)n * l);
    ScrossWs w;
    if (!w.carve(ar, ctx, n, k, l)) return LRP_ERR_WORKSPACE;
    LRP_TRY(tall_copy(ctx, n, k, d_C, ldc, Qb, n));
    LRP_TRY(tall_copy(ctx, n, l, d_Rt, ldr, Zb, n));
    const int p = k < l ? k : l;
    std::vector<double> hS(p), hrC(k), hrR(l);
    int rank = 0; double smin = 0.0;
    LRP_TRY(scross_factor(ctx, n, Qb, n, k, 0, Zb, n, l, 0, d_I, d_J, w, hS.data(), hrC.data(), hrR.data(), &rank, &smin, nullptr));
    LRP_TRY(rebuild(ctx, n, Qb, n, k, w.Uc, k, rank, d_U, ldu, nullptr));
    LRP_TRY(rebuild(ctx, n, Zb, n, l, w.Vc, l, rank, d_V, ldv, nullptr));
    LRP_CUDA(ctx, cudaMemcpyAsync(d_S, w.S, sizeof(double) * p, cudaMemcpyDeviceToDevice, ctx->stream));
    if (d_rC) LRP_CUDA(ctx, cudaMemcpyAsync(d_rC, w.rC, sizeof(double) * k, cudaMemcpyDeviceToDevice, ctx->stream));
    if (d_rR) LRP_CUDA(ctx, cudaMemcpyAsync(d_rR, w.rR, sizeof(double) * l, cudaMemcpyDeviceToDevice, ctx->stream));
    LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (h_rank_out) *h_rank_out = rank;
    if (h_smin_full_out) *h_smin_full_out = smin;
    return LRP_OK;
}

int lrp_lowrank_entries(lrp_ctx* ctx, int64_t n, int32_t r, const double* d_U, int64_t ldu, const double* d_S,
                        const double* d_V, int64_t ldv, const int64_t* d_rows, const int64_t* d_cols,
                        int64_t count, double* d_out) {
    if (!ctx || n < 1 || r < 0 || !d_U || !d_S || !d_V || !d_rows || !d_cols || !d_out || ldu < n || ldv < n || count < 0)
        return LRP_ERR_BADARG;
    return tall_lowrank_entries(ctx, r, d_U, ldu, d_S, d_V, ldv, d_rows, d_cols, count, d_out);
}

// Leverage scores of the initial guess (Alg. 3 lines 1-3) for BOTH sides through CholeskyQR2 instead of
// the Householder TSQR: the scores are the diagonal of the projector onto span(A) and do not depend on which orthonormal
// basis is used, and a well-conditioned A (the transformed right-hand-side factors, an orthonormal initial guess) does not
// need Householder's robustness.  Per side: G = A^T A (one DMMA sweep), R = chol(G) on the host (c <= 64), Q1 = A R^-1,
// G2 = Q1^T Q1, Q = Q1 R2^-1 with the squared row norms fused into that last sweep: five passes over c columns instead of
// a panel-by-panel BCGS2 + TSQR (2.0 -> 0.4 ms at C4).  Q ends up in Cb / Rb (DEIM / QDEIM read it there), the scores in
// scoresU / scoresV.  Returns 1 without side effects on the outputs when a Cholesky pivot loses more than 10 digits
// (kappa(A) beyond ~1e5): the caller then runs the Householder path, which is what defines Q for dependent columns.
static int leverage_cholqr2_pair(lrp_ctx* ctx, int64_t n, int c, const double* AU, const double* AV, int64_t lda, SolveWs& w, int64_t ld) {
    cudaStream_t side = ctx->prof_on == 1 ? ctx->stream : ctx->aux;
    std::vector<double> gU((size_t)c * c), gV((size_t)c * c), iU, iV;
    const size_t gb = sizeof(double) * (size_t)c * c;
    auto fork = [&]() -> int {
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_fork, ctx->stream));
        LRP_CUDA(ctx, cudaStreamWaitEvent(side, ctx->ev_fork, 0));
        return LRP_OK;
    };
    auto join_sync = [&]() -> int {
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_join, side));
        LRP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
        LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        return LRP_OK;
    };
    const double* srcU = AU; const double* srcV = AV; int64_t lsrc = lda;
    for (int pass = 0; pass < 2; ++pass) {
        LRP_TRY(fork());
        const bool pin = 2 * gb <= LRP_PINNED_BYTES;          // pageable targets would block the host between the launches
        double* hU = pin ? ctx->pinned : gU.data();
        double* hV = pin ? ctx->pinned + (size_t)c * c : gV.data();
        LRP_TRY(tall_gemm_t(ctx, n, srcU, lsrc, c, srcU, lsrc, c, w.GU, c, 0, w.gemmt_ws));
        LRP_ON_STREAM(ctx, side, tall_gemm_t(ctx, n, srcV, lsrc, c, srcV, lsrc, c, w.GV, c, 0, w.gemmt_ws2));
        LRP_CUDA(ctx, d2h_small(ctx, hU, w.GU, gb, ctx->stream));
        LRP_CUDA(ctx, d2h_small(ctx, hV, w.GV, gb, side));
        LRP_TRY(join_sync());
        if (pin) { memcpy(gU.data(), hU, gb); memcpy(gV.data(), hV, gb); }
        if (!host_chol_inverse(gU, c, iU) || !host_chol_inverse(gV, c, iV)) return 1;
        LRP_CUDA(ctx, h2d_small(ctx, w.Amat, iU.data(), gb, ctx->stream));
        LRP_CUDA(ctx, h2d_small(ctx, w.Bmat, iV.data(), gb, ctx->stream));
        LRP_TRY(fork());
        if (pass == 0) {
            LRP_TRY(rebuild(ctx, n, srcU, lsrc, c, w.Amat, c, c, w.Ua, ld, nullptr));
            LRP_ON_STREAM(ctx, side, rebuild(ctx, n, srcV, lsrc, c, w.Bmat, c, c, w.Va, ld, nullptr));
            srcU = w.Ua; srcV = w.Va; lsrc = ld;
        } else {
            LRP_TRY(rebuild(ctx, n, srcU, lsrc, c, w.Amat, c, c, w.Cb, ld, w.scoresU));
            LRP_ON_STREAM(ctx, side, rebuild(ctx, n, srcV, lsrc, c, w.Bmat, c, c, w.Rb, ld, w.scoresV));
        }
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_join, side));
        LRP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
    }
    return LRP_OK;
}

// The Cross-DEIM driver (Alg. 4) for a matrix given by its fiber sampler ("G(i,j) as a function handle",
// PAPER.md:20, 68).  kind = LRP_G_POISSON: the spectral Poisson solution of eq. (4) between the two batched DST-I
// (rF, d_UF, d_SF, d_VF = right-hand side in physical space); kind = LRP_G_HILBERT / LRP_G_KMATRIX: the closed-form test
// matrices of eq. (6), no transforms (rF = columns of the required initial guess opts->d_U0 / d_V0; d_UF/d_SF/d_VF unused).
static int solve_impl(lrp_ctx* ctx, int kind, int64_t n, int32_t rF, const double* d_UF, int64_t ldu, const double* d_SF,
                      const double* d_VF, int64_t ldv, const lrp_solve_opts* opts,
                      double* d_UW, int64_t lduw, double* d_SW, double* d_VW, int64_t ldvw, lrp_solve_info* info,
                      int32_t* h_trace_I, int32_t* h_trace_J, uint8_t* h_trace_keepI, uint8_t* h_trace_keepJ,
                      double* d_Uhat, double* d_Shat, double* d_Vhat, int64_t ld_hat) {
    if (!ctx || !opts || !info) return LRP_ERR_BADARG;
    const bool poisson = kind == LRP_G_POISSON;
    if (poisson) LRP_TRY(check_n(n));
    else if (kind != LRP_G_HILBERT && kind != LRP_G_KMATRIX) return LRP_ERR_BADARG;
    else if (n < 2 || n > ((int64_t)1 << 30) || !opts->d_U0 || !opts->d_V0) return LRP_ERR_BADARG;
    if (rF < 1 || !d_UW || !d_SW || !d_VW || lduw < n || ldvw < n) return LRP_ERR_BADARG;
    if (poisson && (!d_UF || !d_SF || !d_VF || ldu < n || ldv < n)) return LRP_ERR_BADARG;
    if (opts->max_rank < 1 || opts->oversample < 0 || opts->max_sweeps < 1 || !(opts->tol > 0.0)) return LRP_ERR_BADARG;
    if (opts->selection < LRP_SELECT_TOPK || opts->selection > LRP_SELECT_DEIM) return LRP_ERR_BADARG;
    const int max_rank = opts->max_rank, p_os = opts->oversample;
    const int Kc = 2 * (max_rank + p_os);             // reading Q10 (the oracle's K_cap): index lists are cut there
    if (Kc < rF + p_os + 1) return LRP_ERR_BADARG;    // the first sweep's selection (rF + p_os indices + safeguard) must fit
    if (Kc > n || rF > n) return LRP_ERR_BADARG;
    const bool replay = opts->replay_sweeps > 0;
    const int max_sweeps = replay ? opts->replay_sweeps : opts->max_sweeps;
    if (max_sweeps > LRP_MAX_SWEEPS_INFO) return LRP_ERR_BADARG;
    const double* U0 = opts->d_U0; const double* V0 = opts->d_V0; int r0 = opts->r0; int64_t ld0 = opts->ld0;
    if ((U0 == nullptr) != (V0 == nullptr)) return LRP_ERR_BADARG;
    if (U0 && (r0 < 1 || r0 + p_os + 1 > Kc || ld0 < n)) return LRP_ERR_BADARG;
    if (ctx->ws_bytes < (poisson ? lrp_workspace_bytes(n, rF, max_rank, p_os) : lrp_matrix_workspace_bytes(n, rF, max_rank, p_os))) return LRP_ERR_WORKSPACE;
    lrp_arena ar(ctx->ws, ctx->ws_bytes);
    SolveWs w;
    if (!w.carve(ar, ctx, n, rF, Kc, max_rank, poisson)) return LRP_ERR_WORKSPACE;
    memset(info, 0, sizeof(*info));
    const int64_t launches0 = ctx->launches;
    const int64_t ld = internal_ld(n);
    const double scale = sqrt(2.0 / (double)(n + 1));
    EventPool ep(ctx);
    FlagsGuard fguard(ctx, opts->flags);
    cudaEvent_t e_start = ep.rec(ctx);

    // O3: spectral RHS factors
    if (poisson) {   // the two batched transforms are independent: main and auxiliary stream
        cudaStream_t dside = ctx->prof_on == 1 ? ctx->stream : ctx->aux;
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_fork, ctx->stream));
        LRP_CUDA(ctx, cudaStreamWaitEvent(dside, ctx->ev_fork, 0));
        LRP_TRY(lrp_dst1_impl(ctx, n, rF, d_UF, ldu, w.UhF, ld, scale, w.dst_ws, w.dst_ws_bytes));
        LRP_ON_STREAM(ctx, dside, lrp_dst1_impl(ctx, n, rF, d_VF, ldv, w.VhF, ld, scale, w.dst_ws2, w.dst_ws_bytes));
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_join, dside));
        LRP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
    }
    cudaEvent_t e_dst = ep.rec(ctx);
    info->ms_dst_fwd = 0.f;

    double* Uk = w.Ua; double* Vk = w.Va; double* Up = w.Ub; double* Vp = w.Vb;
    int r_prev = 0;                       // rank of the previous iterate (0 at k = 0: previous iterate = 0, reading Q13)
    const double* selU = U0 ? U0 : w.UhF; const double* selV = U0 ? V0 : w.VhF;
    int64_t sel_ld = U0 ? ld0 : ld; int sel_cols = U0 ? r0 : rF;
    std::vector<int32_t> I_prev, J_prev, I_k, J_k, hstar(2 * (size_t)Kc + 8);
    // Fibers of an index are the same in every sweep, and the QR of a column prefix is the prefix of the QR: the leading
    // columns of this sweep's fiber block that repeat last sweep's block in the same order keep their Q columns (still in
    // Cb / Rb) and their block of R; only the columns after the common prefix are sampled and factored.
    std::vector<int32_t> I_fact, J_fact;          // index lists whose Q factors Rb / Cb hold (empty: none)
    const bool reuse_qr = !(opts->flags & LRP_FLAG_NO_QR_REUSE);
    const bool nested_rho = reuse_qr && !(opts->flags & LRP_FLAG_NO_NESTED_RHO);
    int kk_prev = 0, l_prev = 0;                  // sizes of the previous sweep's index lists (rows of UcPrev / VcPrev)
    std::vector<double> hS(Kc), hrC(Kc), hrR(Kc), hS_last;
    std::vector<uint8_t> keepI, keepJ;
    int rank = 0; double smin = 0.0;
    bool converged = false;
    size_t rep_offI = 0, rep_offJ = 0, tr_offI = 0, tr_offJ = 0;
    int sweeps = 0;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> t_sel, t_sample, t_qr, t_core, t_rebuild, t_stop;

    for (int k = 0; k < max_sweeps; ++k) {
        cudaEvent_t e0 = ep.rec(ctx);
        // ---- O6/O7: selection, union, safeguard
        if (!replay) {
            if (k == 0) {
                // well-conditioned initial guess: CholeskyQR2 (five passes); otherwise Householder, below
                int rc_lev = 1;
                if (sel_cols <= 64 && !(opts->flags & LRP_FLAG_NO_CHOLQR_LEVERAGE))
                    rc_lev = leverage_cholqr2_pair(ctx, n, sel_cols, selU, selV, sel_ld, w, ld);
                if (rc_lev < 0) return rc_lev;
                if (rc_lev == 1) {
                // the two leverage QRs of the initial guess are independent: factored as a pair on the two streams
                LRP_TRY(tall_copy(ctx, n, sel_cols, selU, sel_ld, w.Cb, ld));
                LRP_TRY(tall_copy(ctx, n, sel_cols, selV, sel_ld, w.Rb, ld));
                LRP_TRY(tall_qr_pair(ctx, n, sel_cols, w.Cb, ld, w.Rlev, sel_cols, w.sc.qr_ws, sel_cols, w.Rb, ld, w.Rlev2, sel_cols, w.sc.qr_ws2));
                LRP_TRY(leverage_colmask(ctx, sel_cols, w.Rlev, sel_cols, LEV_COL_RCOND, w.mask));
                LRP_TRY(tall_rownorm2(ctx, n, sel_cols, w.Cb, ld, w.mask, w.scoresU));
                LRP_TRY(leverage_colmask(ctx, sel_cols, w.Rlev2, sel_cols, LEV_COL_RCOND, w.mask2));
                LRP_TRY(tall_rownorm2(ctx, n, sel_cols, w.Rb, ld, w.mask2, w.scoresV));
                }
            }
            int64_t numsel64 = (int64_t)sel_cols + p_os; if (numsel64 > n) numsel64 = n;
            if (numsel64 > 2 * (int64_t)Kc) numsel64 = 2 * (int64_t)Kc;
            const int numsel = (int)numsel64;
            // deterministic top-k: both sides are enqueued before the one host synchronisation that reads them
            const bool topk_pair = opts->selection == LRP_SELECT_TOPK && 2 * sizeof(int32_t) * (size_t)numsel <= LRP_PINNED_BYTES;
            if (topk_pair) {
                int32_t* hp = reinterpret_cast<int32_t*>(ctx->pinned);
                LRP_TRY(select_topk(ctx, n, w.scoresU, numsel, w.dIstar, w.sel_ws));
                LRP_CUDA(ctx, d2h_small(ctx, hp, w.dIstar, sizeof(int32_t) * numsel, ctx->stream));
                LRP_TRY(select_topk(ctx, n, w.scoresV, numsel, w.dJstar, w.sel_ws));
                LRP_CUDA(ctx, d2h_small(ctx, hp + numsel, w.dJstar, sizeof(int32_t) * numsel, ctx->stream));
                LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
            }
            for (int side = 0; side < 2; ++side) {
                std::vector<int32_t>& cur = side == 0 ? I_k : J_k;
                const std::vector<int32_t>& prev = side == 0 ? I_prev : J_prev;
                double* sc = side == 0 ? w.scoresU : w.scoresV;
                int32_t* dstar = side == 0 ? w.dIstar : w.dJstar;
                int nstar = numsel;
                if (opts->selection == LRP_SELECT_QDEIM || opts->selection == LRP_SELECT_DEIM) {
                    // Alg. 2 on the orthonormal factor of the previous iterate: at k = 0 the Q of the
                    // initial guess (left in Cb / Rb by the leverage QR above), later the iterate itself; the target
                    // buffer of this sweep's rebuild is free and serves as the (destroyed) working copy
                    const double* src = k == 0 ? (side == 0 ? w.Cb : w.Rb) : (side == 0 ? Up : Vp);
                    double* work = side == 0 ? Uk : Vk;
                    nstar = sel_cols;
                    LRP_TRY(tall_copy(ctx, n, sel_cols, src, ld, work, ld));
                    LRP_TRY(deim_select(ctx, opts->selection == LRP_SELECT_QDEIM ? 1 : 0, n, sel_cols, work, ld, dstar, w.deim_ws));
                    LRP_CUDA(ctx, cudaMemcpyAsync(hstar.data(), dstar, sizeof(int32_t) * nstar, cudaMemcpyDeviceToHost, ctx->stream));
                    LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
                } else if (opts->selection == LRP_SELECT_BERNOULLI) {   // Alg. 3 lines 4-5 as printed, reading Q23
                    SelectBernoulli b{};
                    b.cols = sel_cols; b.c = opts->ls_c > 0.0 ? opts->ls_c : (double)(sel_cols + p_os);
                    b.seed = opts->ls_seed; b.sweep = k; b.side = side;
                    int64_t cap64 = 2 * (int64_t)Kc; if (cap64 > n) cap64 = n;
                    const int cap = (int)cap64;
                    int32_t* d_count = dstar + 2 * (size_t)Kc + 4;
                    int32_t h_count = 0;
                    LRP_TRY(select_topk(ctx, n, sc, cap, dstar, w.sel_ws, &b, d_count));
                    LRP_CUDA(ctx, cudaMemcpyAsync(hstar.data(), dstar, sizeof(int32_t) * cap, cudaMemcpyDeviceToHost, ctx->stream));
                    LRP_CUDA(ctx, cudaMemcpyAsync(&h_count, d_count, sizeof(int32_t), cudaMemcpyDeviceToHost, ctx->stream));
                    LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
                    nstar = h_count < cap ? h_count : cap;
                } else if (topk_pair) {
                    memcpy(hstar.data(), reinterpret_cast<int32_t*>(ctx->pinned) + (size_t)side * numsel, sizeof(int32_t) * numsel);
                } else {
                    LRP_TRY(select_topk(ctx, n, sc, numsel, dstar, w.sel_ws));
                    const bool pin = sizeof(int32_t) * (size_t)numsel <= LRP_PINNED_BYTES;
                    LRP_CUDA(ctx, d2h_small(ctx, pin ? (void*)ctx->pinned : (void*)hstar.data(), dstar, sizeof(int32_t) * numsel, ctx->stream));
                    LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
                    if (pin) memcpy(hstar.data(), ctx->pinned, sizeof(int32_t) * numsel);
                }
                cur = prev;
                int added = 0;
                host_union(cur, hstar.data(), nstar, &added);
                if (added == 0 || k == 0) {       // Alg. 4 lines 7-12, reading Q9
                    bool done = false;
                    for (int s = 0; s < opts->n_safeguard && opts->h_safeguard; ++s) {
                        int32_t cand = opts->h_safeguard[s];
                        if (cand < 0 || cand >= n) continue;
                        if (std::find(cur.begin(), cur.end(), cand) == cur.end()) { cur.push_back(cand); done = true; break; }
                    }
                    if (!done && (int64_t)cur.size() < n) {   // list exhausted: best-scoring index not in the set
                        int want = (int)cur.size() + 1; if (want > Kc + 1) want = Kc + 1;
                        std::vector<int32_t> more(want);
                        LRP_TRY(select_topk(ctx, n, sc, want, dstar, w.sel_ws));
                        LRP_CUDA(ctx, cudaMemcpyAsync(more.data(), dstar, sizeof(int32_t) * want, cudaMemcpyDeviceToHost, ctx->stream));
                        LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
                        for (int32_t cand : more)
                            if (cand >= 0 && std::find(cur.begin(), cur.end(), cand) == cur.end()) { cur.push_back(cand); break; }
                    }
                }
                if ((int)cur.size() > Kc) cur.resize(Kc);       // reading Q10
            }
        } else {
            const int nI = opts->h_replay_nI[k], nJ = opts->h_replay_nJ[k];
            if (nI < 1 || nJ < 1 || nI > Kc || nJ > Kc) return LRP_ERR_BADARG;
            I_k.assign(opts->h_replay_I + rep_offI, opts->h_replay_I + rep_offI + nI);
            J_k.assign(opts->h_replay_J + rep_offJ, opts->h_replay_J + rep_offJ + nJ);
            LRP_TRY(validate_indices(I_k.data(), nI, n));
            LRP_TRY(validate_indices(J_k.data(), nJ, n));
        }
        const int l = (int)I_k.size(), kk = (int)J_k.size();
        LRP_CUDA(ctx, h2d_small(ctx, w.dI, I_k.data(), sizeof(int32_t) * l, ctx->stream));
        LRP_CUDA(ctx, h2d_small(ctx, w.dJ, J_k.data(), sizeof(int32_t) * kk, ctx->stream));
        cudaEvent_t e1 = ep.rec(ctx);
        // ---- O4: fibers  C = G(:,J) (n x kk), Rt = G(I,:)^T (n x l)
        // the two sides of a sweep are independent until the small core: they run on the main and the auxiliary stream
        // (every tall kernel here is latency-bound well below the HBM peak, so two in flight overlap usefully)
        cudaStream_t side = ctx->prof_on == 1 ? ctx->stream : ctx->aux;      // profiling: serial, clean per-kernel event times
        int k0 = 0, l0 = 0;
        if (reuse_qr) {
            while (k0 < kk && k0 < (int)J_fact.size() && J_fact[k0] == J_k[k0]) ++k0;
            while (l0 < l && l0 < (int)I_fact.size() && I_fact[l0] == I_k[l0]) ++l0;
        }
        // nested stop test (reading R5): the previous block's Q columns after the common prefix are about to be
        // overwritten; up to NREST_MAX of them are set aside (they carry part of U_{k-1})
        const int nrJ = (int)J_fact.size() - k0, nrI = (int)I_fact.size() - l0;
        const bool nested = nested_rho && r_prev > 0 && k0 > 0 && l0 > 0 && (int)J_fact.size() == kk_prev &&
                            (int)I_fact.size() == l_prev && nrJ <= NREST_MAX && nrI <= NREST_MAX;
        if (nested && nrJ > 0) LRP_TRY(tall_copy(ctx, n, nrJ, w.Cb + (int64_t)k0 * ld, ld, w.QrestU, ld));
        if (nested && nrI > 0) LRP_TRY(tall_copy(ctx, n, nrI, w.Rb + (int64_t)l0 * ld, ld, w.QrestV, ld));
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_fork, ctx->stream));
        LRP_CUDA(ctx, cudaStreamWaitEvent(side, ctx->ev_fork, 0));
        if (poisson) {
            if (kk > k0) LRP_TRY(sample_side(ctx, n, rF, w.UhF, ld, d_SF, w.VhF, ld, w.dJ + k0, kk - k0, w.Cb + (int64_t)k0 * ld, ld));
            if (l > l0) LRP_ON_STREAM(ctx, side, sample_side(ctx, n, rF, w.VhF, ld, d_SF, w.UhF, ld, w.dI + l0, l - l0, w.Rb + (int64_t)l0 * ld, ld));
        } else {
            if (kk > k0) LRP_TRY(tall_matrix_fibers(ctx, kind, n, 0, w.dJ + k0, kk - k0, w.Cb + (int64_t)k0 * ld, ld));
            if (l > l0) LRP_ON_STREAM(ctx, side, tall_matrix_fibers(ctx, kind, n, 1, w.dI + l0, l - l0, w.Rb + (int64_t)l0 * ld, ld));
        }
        cudaEvent_t e2 = ep.rec(ctx);
        // ---- O8: scross
        cudaEvent_t e3 = ep.take();
        LRP_TRY(scross_factor(ctx, n, w.Cb, ld, kk, k0, w.Rb, ld, l, l0, w.dI, w.dJ, w.sc, hS.data(), hrC.data(), hrR.data(), &rank, &smin, e3));
        J_fact = J_k; I_fact = I_k;
        cudaEvent_t e4 = ep.rec(ctx);
        const int p = kk < l ? kk : l;
        // ---- O9: prune (Alg. 4 lines 14-23; reading Q12)
        keepI.assign(l, 1); keepJ.assign(kk, 1);
        if (replay && opts->h_replay_keepI && opts->h_replay_keepJ) {
            for (int c = 0; c < l; ++c) keepI[c] = opts->h_replay_keepI[rep_offI + c] ? 1 : 0;
            for (int c = 0; c < kk; ++c) keepJ[c] = opts->h_replay_keepJ[rep_offJ + c] ? 1 : 0;
        } else {
            double mR = 0.0, mC = 0.0;
            for (int c = 0; c < l; ++c) mR = std::max(mR, hrR[c]);
            for (int c = 0; c < kk; ++c) mC = std::max(mC, hrC[c]);
            for (int c = 0; c < l; ++c) keepI[c] = hrR[c] >= PRUNE_REL * mR;
            for (int c = 0; c < kk; ++c) keepJ[c] = hrC[c] >= PRUNE_REL * mC;
        }
        std::vector<int32_t> I_pr, J_pr;
        for (int c = 0; c < l; ++c) if (keepI[c]) I_pr.push_back(I_k[c]);
        for (int c = 0; c < kk; ++c) if (keepJ[c]) J_pr.push_back(J_k[c]);
        if (h_trace_I) memcpy(h_trace_I + tr_offI, I_k.data(), sizeof(int32_t) * l);
        if (h_trace_J) memcpy(h_trace_J + tr_offJ, J_k.data(), sizeof(int32_t) * kk);
        if (h_trace_keepI) memcpy(h_trace_keepI + tr_offI, keepI.data(), l);
        if (h_trace_keepJ) memcpy(h_trace_keepJ + tr_offJ, keepJ.data(), kk);
        tr_offI += l; tr_offJ += kk; rep_offI += l; rep_offJ += kk;
        // ---- eta (reading Q14) from the factored form U(I,:) = Q(I,:) Uc: two one-CTA Jacobi SVDs on the third stream,
        // started before the rebuild so that they hide behind it (and behind the rho contractions of later sweeps)
        cudaStream_t side2 = ctx->prof_on == 1 ? ctx->stream : ctx->aux2;
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_fork, ctx->stream));
        LRP_CUDA(ctx, cudaStreamWaitEvent(side, ctx->ev_fork, 0));
        LRP_CUDA(ctx, cudaStreamWaitEvent(side2, ctx->ev_fork, 0));
        {
            cudaStream_t main_stream = ctx->stream;
            ctx->stream = side2;
            int rc_eta = LRP_OK;
            cudaError_t e1 = h2d_small(ctx, w.dIpr, I_pr.data(), sizeof(int32_t) * I_pr.size(), ctx->stream);
            cudaError_t e2 = h2d_small(ctx, w.dJpr, J_pr.data(), sizeof(int32_t) * J_pr.size(), ctx->stream);
            if (e1 != cudaSuccess || e2 != cudaSuccess) { ctx->last_cuda = (int)(e1 != cudaSuccess ? e1 : e2); rc_eta = LRP_ERR_CUDA; }
            if (rc_eta == LRP_OK) {
                EtaArgs ea{};
                ea.r = rank; ea.U = w.Cb; ea.ldu = ld; ea.I = w.dIpr; ea.nI = (int)I_pr.size(); ea.V = w.Rb; ea.ldv = ld; ea.J = w.dJpr; ea.nJ = (int)J_pr.size();
                ea.CU = w.sc.Uc; ea.kU = kk; ea.ldcu = kk; ea.CV = w.sc.Vc; ea.kV = l; ea.ldcv = l;
                ea.eta = w.eta; ea.work = w.eta_work; ea.work_stride = w.eta_stride; ea.iwork = w.eta_iwork; ea.iwork_stride = Kc;
                rc_eta = eta_pair(ctx, ea);
            }
            cudaError_t e4 = cudaEventRecord(ctx->ev_join2, ctx->stream);
            ctx->stream = main_stream;
            if (rc_eta < 0) return rc_eta;
            if (e4 != cudaSuccess) { ctx->last_cuda = (int)e4; return LRP_ERR_CUDA; }
        }
        LRP_TRY(rebuild(ctx, n, w.Cb, ld, kk, w.sc.Uc, kk, rank, Uk, ld, w.scoresU));
        LRP_ON_STREAM(ctx, side, rebuild(ctx, n, w.Rb, ld, l, w.sc.Vc, l, rank, Vk, ld, w.scoresV));
        cudaEvent_t e5 = ep.rec(ctx);
        // ---- O10: rho (factored, reading Q13), indicator.
        // Nested case: last sweep's lists are (up to a few dropped trailing entries) prefixes of this sweep's and the Q
        // columns of the common prefix were kept: rho needs the small core factors and, for the dropped columns, three
        // narrow passes (T = Q_k^T Q_rest, P = Q_rest - Q_k T, P^T P) instead of the contractions over the tall iterates.
        if (nested) {
            if (nrI > 0) {
                cudaStream_t main_stream = ctx->stream;
                ctx->stream = side;
                // Q_rest was orthonormal to the common prefix in last sweep's Q: only the rows of T that belong to this
                // sweep's new columns are non-zero (the others are rounding, 1e-14), and only those columns are read
                int rc_v = cudaMemsetAsync(w.TV, 0, sizeof(double) * (size_t)l * nrI, ctx->stream) == cudaSuccess ? LRP_OK : LRP_ERR_CUDA;
                if (rc_v >= 0 && l > l0) rc_v = tall_gemm_t(ctx, n, w.Rb + (int64_t)l0 * ld, ld, l - l0, w.QrestV, ld, nrI, w.TV + l0, l, 0, w.gemmt_ws2);
                if (rc_v >= 0 && l > l0) {
                    TallGemmArgs g{};
                    g.n = n; g.k = l - l0; g.m = nrI; g.mode = TG_SUBTRACT; g.A = w.Rb + (int64_t)l0 * ld; g.lda = ld; g.B = w.TV + l0; g.ldb = l;
                    g.Cin = w.QrestV; g.ldc = ld; g.Out = w.QrestV; g.ldo = ld;
                    rc_v = tall_gemm(ctx, g);
                }
                if (rc_v >= 0) rc_v = tall_gemm_t(ctx, n, w.QrestV, ld, nrI, w.QrestV, ld, nrI, w.GpV, nrI, 0, w.gemmt_ws2);
                ctx->stream = main_stream;
                if (rc_v < 0) return rc_v;
            }
            LRP_CUDA(ctx, cudaEventRecord(ctx->ev_join, side));
            if (nrJ > 0) {
                LRP_CUDA(ctx, cudaMemsetAsync(w.TU, 0, sizeof(double) * (size_t)kk * nrJ, ctx->stream));
                if (kk > k0) {
                    LRP_TRY(tall_gemm_t(ctx, n, w.Cb + (int64_t)k0 * ld, ld, kk - k0, w.QrestU, ld, nrJ, w.TU + k0, kk, 0, w.gemmt_ws));
                    TallGemmArgs g{};
                    g.n = n; g.k = kk - k0; g.m = nrJ; g.mode = TG_SUBTRACT; g.A = w.Cb + (int64_t)k0 * ld; g.lda = ld; g.B = w.TU + k0; g.ldb = kk;
                    g.Cin = w.QrestU; g.ldc = ld; g.Out = w.QrestU; g.ldo = ld;
                    LRP_TRY(tall_gemm(ctx, g));
                }
                LRP_TRY(tall_gemm_t(ctx, n, w.QrestU, ld, nrJ, w.QrestU, ld, nrJ, w.GpU, nrJ, 0, w.gemmt_ws));
            }
            LRP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
            RhoNestedSide su{}, sv{};
            su.kk = kk; su.kkp = kk_prev; su.k0 = k0; su.Uc = w.sc.Uc; su.ldc = kk; su.Ucp = w.UcPrev; su.ldcp = kk_prev;
            su.T = w.TU; su.Gp = w.GpU; su.A = w.Amat; su.G = w.GU; su.scratch = w.nestU;
            sv.kk = l; sv.kkp = l_prev; sv.k0 = l0; sv.Uc = w.sc.Vc; sv.ldc = l; sv.Ucp = w.VcPrev; sv.ldcp = l_prev;
            sv.T = w.TV; sv.Gp = w.GpV; sv.A = w.Bmat; sv.G = w.GV; sv.scratch = w.nestV;
            LRP_TRY(rho_nested_prep(ctx, rank, r_prev, su, sv));
        }
        // General case: the two sides run on the main and the auxiliary stream.
        if (r_prev > 0 && !nested) {
            cudaStream_t main_stream = ctx->stream;
            ctx->stream = side;
            int rc_v = tall_gemm_t(ctx, n, Vk, ld, rank, Vp, ld, r_prev, w.Bmat, rank, 0, w.gemmt_ws2);
            // E_V = V_{k-1} - V_k B and its Gram matrix in one pass (E never written); outside the fused kernel's range:
            // update sweep IN PLACE over V_{k-1} (dead after this test: its buffer is the next sweep's rebuild target)
            // + Gram sweep.  The fiber buffers keep their Q factors for the next sweep.
            if (rc_v >= 0) rc_v = tall_resid_gram(ctx, n, Vk, ld, rank, w.Bmat, rank, Vp, ld, r_prev, w.GV, r_prev, w.gemmt_ws2);
            if (rc_v == 1) {
                TallGemmArgs g{};
                g.n = n; g.k = rank; g.m = r_prev; g.mode = TG_SUBTRACT; g.A = Vk; g.lda = ld; g.B = w.Bmat; g.ldb = rank;
                g.Cin = Vp; g.ldc = ld; g.Out = Vp; g.ldo = ld;
                rc_v = tall_gemm(ctx, g);
                if (rc_v >= 0) rc_v = tall_gemm_t(ctx, n, Vp, ld, r_prev, Vp, ld, r_prev, w.GV, r_prev, 0, w.gemmt_ws2);
            }
            ctx->stream = main_stream;
            if (rc_v < 0) return rc_v;
        }
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_join, side));
        RhoArgs ra{};
        ra.r = rank; ra.rp = r_prev; ra.Sk = w.sc.S; ra.Sp = w.Sprev; ra.A = w.Amat; ra.B = w.Bmat; ra.GU = w.GU; ra.GV = w.GV;
        ra.out = w.rho_out; ra.partial = w.rho_out + 16; ra.ticket = reinterpret_cast<unsigned*>(w.rho_out + 16 + RHO_MAX_GRID);
        if (r_prev > 0 && !nested) {
            LRP_TRY(tall_gemm_t(ctx, n, Uk, ld, rank, Up, ld, r_prev, w.Amat, rank, 0, w.gemmt_ws));      // U side
            int rc_u = tall_resid_gram(ctx, n, Uk, ld, rank, w.Amat, rank, Up, ld, r_prev, w.GU, r_prev, w.gemmt_ws);
            if (rc_u < 0) return rc_u;
            if (rc_u == 1) {
                TallGemmArgs g{};
                g.n = n; g.k = rank; g.m = r_prev; g.mode = TG_SUBTRACT; g.A = Uk; g.lda = ld; g.B = w.Amat; g.ldb = rank;
                g.Cin = Up; g.ldc = ld; g.Out = Up; g.ldo = ld;
                LRP_TRY(tall_gemm(ctx, g));
                LRP_TRY(tall_gemm_t(ctx, n, Up, ld, r_prev, Up, ld, r_prev, w.GU, r_prev, 0, w.gemmt_ws));
            }
        }
        LRP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
        LRP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_join2, 0));
        LRP_TRY(rho_small(ctx, ra));
        double h_rho[2], h_eta[2];
        LRP_CUDA(ctx, d2h_small(ctx, ctx->pinned, w.rho_out, sizeof(double) * 16, ctx->stream));
        LRP_CUDA(ctx, cudaMemcpyAsync(w.Sprev, w.sc.S, sizeof(double) * rank, cudaMemcpyDeviceToDevice, ctx->stream));
        LRP_CUDA(ctx, cudaMemcpyAsync(w.UcPrev, w.sc.Uc, sizeof(double) * (size_t)kk * rank, cudaMemcpyDeviceToDevice, ctx->stream));
        LRP_CUDA(ctx, cudaMemcpyAsync(w.VcPrev, w.sc.Vc, sizeof(double) * (size_t)l * rank, cudaMemcpyDeviceToDevice, ctx->stream));
        kk_prev = kk; l_prev = l;
        LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        h_rho[0] = ctx->pinned[0]; h_rho[1] = ctx->pinned[1]; h_eta[0] = ctx->pinned[8]; h_eta[1] = ctx->pinned[9];
        cudaEvent_t e6 = ep.rec(ctx);
        const double rho = h_rho[0], snorm = h_rho[1], eta1 = h_eta[0], eta2 = h_eta[1];
        const double ind = (smin == 0.0) ? 0.0 : std::min(eta1 * (1.0 + eta2), eta2 * (1.0 + eta1)) * smin;
        info->nI[k] = l; info->nJ[k] = kk; info->rank_per_sweep[k] = rank; info->rho_per_sweep[k] = rho; info->ind_per_sweep[k] = ind;
        info->rho = rho; info->indicator = ind; info->eta1 = eta1; info->eta2 = eta2; info->snorm = snorm; info->smin_full = smin;
        t_sel.push_back({e0, e1}); t_sample.push_back({e1, e2}); t_qr.push_back({e2, e3}); t_core.push_back({e3, e4});
        t_rebuild.push_back({e4, e5}); t_stop.push_back({e5, e6});
        hS_last.assign(hS.begin(), hS.begin() + p);
        sweeps = k + 1;
        // next sweep: warm start from this iterate
        std::swap(Uk, Up); std::swap(Vk, Vp);
        r_prev = rank; sel_cols = rank;
        I_prev = I_pr; J_prev = J_pr;
        const double thresh = opts->tol * (opts->tol_mode == 0 ? snorm : 1.0);
        if (!replay && std::max(rho, ind) < thresh) { converged = true; break; }   // Alg. 4 line 26
    }
    // after the swap the last iterate lives in (Up, Vp), rank r_prev
    int r, rstar = 0;
    if (replay && opts->replay_final_rank > 0) { r = opts->replay_final_rank; converged = true; }
    else {
        r = final_rank_host(hS_last.data(), r_prev, opts->tol, max_rank, opts->tol_mode, &rstar);     // O11 over the kept values
        if (rstar > max_rank) converged = false;      // reading Q20: r* > r_max, the tolerance is not met by the truncated result
    }
    if (r > r_prev) r = r_prev;
    if (r > max_rank) r = max_rank;
    cudaEvent_t e_inv0 = ep.rec(ctx);
    if (!poisson) {  // no transform: the truncated iterate is the result
        LRP_TRY(tall_copy(ctx, n, r, Up, ld, d_UW, lduw));
        LRP_TRY(tall_copy(ctx, n, r, Vp, ld, d_VW, ldvw));
    } else {   // O12
        cudaStream_t dside = ctx->prof_on == 1 ? ctx->stream : ctx->aux;
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_fork, ctx->stream));
        LRP_CUDA(ctx, cudaStreamWaitEvent(dside, ctx->ev_fork, 0));
        LRP_TRY(lrp_dst1_impl(ctx, n, r, Up, ld, d_UW, lduw, scale, w.dst_ws, w.dst_ws_bytes));
        LRP_ON_STREAM(ctx, dside, lrp_dst1_impl(ctx, n, r, Vp, ld, d_VW, ldvw, scale, w.dst_ws2, w.dst_ws_bytes));
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_join, dside));
        LRP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
    }
    LRP_CUDA(ctx, cudaMemcpyAsync(d_SW, w.Sprev, sizeof(double) * r, cudaMemcpyDeviceToDevice, ctx->stream));
    if (d_Uhat && d_Vhat && d_Shat && ld_hat >= n) {
        LRP_TRY(tall_copy(ctx, n, r_prev, Up, ld, d_Uhat, ld_hat));
        LRP_TRY(tall_copy(ctx, n, r_prev, Vp, ld, d_Vhat, ld_hat));
        LRP_CUDA(ctx, cudaMemcpyAsync(d_Shat, w.Sprev, sizeof(double) * r_prev, cudaMemcpyDeviceToDevice, ctx->stream));
    }
    cudaEvent_t e_end = ep.rec(ctx);
    LRP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    info->rank = r; info->sweeps = sweeps; info->converged = converged ? 1 : 0;
    info->ms_dst_fwd = EventPool::ms(e_start, e_dst);
    for (auto& pr : t_sel) info->ms_select += EventPool::ms(pr.first, pr.second);
    for (auto& pr : t_sample) info->ms_sample += EventPool::ms(pr.first, pr.second);
    for (auto& pr : t_qr) info->ms_qr += EventPool::ms(pr.first, pr.second);
    for (auto& pr : t_core) info->ms_core += EventPool::ms(pr.first, pr.second);
    for (auto& pr : t_rebuild) info->ms_rebuild += EventPool::ms(pr.first, pr.second);
    for (auto& pr : t_stop) info->ms_stop += EventPool::ms(pr.first, pr.second);
    info->ms_dst_inv = EventPool::ms(e_inv0, e_end);
    info->ms_total = EventPool::ms(e_start, e_end);
    info->launches = ctx->launches - launches0;
    return converged ? LRP_OK : LRP_WARN_NOCONV;
}

int lrp_cross_deim_solve(lrp_ctx* ctx, int64_t n, int32_t rF, const double* d_UF, int64_t ldu, const double* d_SF,
                         const double* d_VF, int64_t ldv, const lrp_solve_opts* opts,
                         double* d_UW, int64_t lduw, double* d_SW, double* d_VW, int64_t ldvw, lrp_solve_info* info,
                         int32_t* h_trace_I, int32_t* h_trace_J, uint8_t* h_trace_keepI, uint8_t* h_trace_keepJ,
                         double* d_Uhat, double* d_Shat, double* d_Vhat, int64_t ld_hat) {
    return solve_impl(ctx, LRP_G_POISSON, n, rF, d_UF, ldu, d_SF, d_VF, ldv, opts, d_UW, lduw, d_SW, d_VW, ldvw, info,
                      h_trace_I, h_trace_J, h_trace_keepI, h_trace_keepJ, d_Uhat, d_Shat, d_Vhat, ld_hat);
}

// ------------------------------------------------------------------------------------------------ host-buffer pipeline
// Staging after the solve's own workspace: two slots of (UF, VF, SF) and two of (UW, VW, SW), ld = n.
namespace {
struct HostStage { double* UF[2]; double* VF[2]; double* SF[2]; double* UW[2]; double* VW[2]; double* SW[2]; };
bool carve_stage(lrp_arena& ar, int64_t n, int rF, int max_rank, HostStage* st) {
    for (int s = 0; s < 2; ++s) {
        double* a = ar.take<double>((size_t)n * rF); double* b = ar.take<double>((size_t)n * rF); double* c = ar.take<double>((size_t)rF);
        double* d = ar.take<double>((size_t)n * max_rank); double* e = ar.take<double>((size_t)n * max_rank); double* f = ar.take<double>((size_t)max_rank);
        if (st) { st->UF[s] = a; st->VF[s] = b; st->SF[s] = c; st->UW[s] = d; st->VW[s] = e; st->SW[s] = f; }
    }
    return ar.ok();
}
// tall block (cols columns of n doubles) between host and device on a copy engine
cudaError_t copy_tall_async(double* dst, int64_t ldd, const double* src, int64_t lds, int64_t n, int cols, cudaMemcpyKind kind, cudaStream_t s) {
    if (cols <= 0) return cudaSuccess;
    if (ldd == n && lds == n) return cudaMemcpyAsync(dst, src, sizeof(double) * (size_t)n * cols, kind, s);
    return cudaMemcpy2DAsync(dst, sizeof(double) * (size_t)ldd, src, sizeof(double) * (size_t)lds, sizeof(double) * (size_t)n, (size_t)cols, kind, s);
}
}  // namespace

// bytes of one lane: the solve's workspace + its two staging slots
static size_t host_lane_bytes(int64_t n, int32_t rF, int32_t max_rank, int32_t oversample) {
    const size_t base = lrp_workspace_bytes(n, rF, max_rank, oversample);
    if (!base) return 0;
    lrp_arena ar((void*)256, (size_t)-1 / 2);
    carve_stage(ar, n, rF, max_rank, nullptr);
    return lrp_align_up(base) + lrp_align_up(ar.off) + 256;
}

size_t lrp_solve_host_workspace_bytes(int64_t n, int32_t rF, int32_t max_rank, int32_t oversample, int32_t lanes) {
    if (lanes < 1 || lanes > LRP_HOST_LANES_MAX) return 0;
    return (size_t)lanes * host_lane_bytes(n, rF, max_rank, oversample);
}

namespace {
struct HostBatch {
    int64_t n; int32_t rF, nprob;
    const double* const* h_UF; int64_t ldu; const double* const* h_SF; const double* const* h_VF; int64_t ldv;
    const lrp_solve_opts* opts;
    double* const* h_UW; int64_t lduw; double* const* h_SW; double* const* h_VW; int64_t ldvw;
    lrp_solve_info* info;
};
// One lane: problems first, first + stride, ... on ctx (its stream, its workspace), each through the lane's two staging
// slots: the upload of the lane's next problem and the download of its previous one run while the current one is solved.
int host_lane(lrp_ctx* ctx, const HostBatch& b, int first, int stride) {
    const int64_t n = b.n; const int rF = b.rF, max_rank = b.opts->max_rank;
    const size_t base = lrp_workspace_bytes(n, rF, max_rank, b.opts->oversample);
    HostStage st;
    {
        const size_t off = lrp_align_up(base);
        if (!base || ctx->ws_bytes < off) return LRP_ERR_WORKSPACE;
        lrp_arena ar((char*)ctx->ws + off, ctx->ws_bytes - off);       // the solve carves only the first `base` bytes
        if (!carve_stage(ar, n, rF, max_rank, &st)) return LRP_ERR_WORKSPACE;
    }
    if (!ctx->cp_in) {                                   // first call on this ctx: two copy streams, four events
        LRP_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->cp_in, cudaStreamNonBlocking));
        LRP_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->cp_out, cudaStreamNonBlocking));
        for (int a = 0; a < 2; ++a) for (int c = 0; c < 2; ++c) LRP_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_cp[a][c], cudaEventDisableTiming));
    }
    auto upload = [&](int p, int s) -> int {
        LRP_CUDA(ctx, copy_tall_async(st.UF[s], n, b.h_UF[p], b.ldu, n, rF, cudaMemcpyHostToDevice, ctx->cp_in));
        LRP_CUDA(ctx, copy_tall_async(st.VF[s], n, b.h_VF[p], b.ldv, n, rF, cudaMemcpyHostToDevice, ctx->cp_in));
        LRP_CUDA(ctx, cudaMemcpyAsync(st.SF[s], b.h_SF[p], sizeof(double) * rF, cudaMemcpyHostToDevice, ctx->cp_in));
        LRP_CUDA(ctx, cudaEventRecord(ctx->ev_cp[0][s], ctx->cp_in));
        return LRP_OK;
    };
    int worst = LRP_OK, rc = first < b.nprob ? upload(first, 0) : LRP_OK;
    int q = 0;                                           // position of the problem in this lane's sequence
    for (int p = first; p < b.nprob && rc >= 0; p += stride, ++q) {
        const int s = q & 1;
        if (cudaStreamWaitEvent(ctx->stream, ctx->ev_cp[0][s], 0) != cudaSuccess) rc = LRP_ERR_CUDA;         // inputs of p are on the device
        // slot s^1 was read by the lane's previous solve, complete on return: the next problem uploads while p is solved
        if (rc >= 0 && p + stride < b.nprob) rc = upload(p + stride, s ^ 1);
        // slot s of the outputs was drained by the download of the lane's problem two back
        if (rc >= 0 && q >= 2 && cudaStreamWaitEvent(ctx->stream, ctx->ev_cp[1][s], 0) != cudaSuccess) rc = LRP_ERR_CUDA;
        if (rc < 0) break;
        ctx->host_pipeline = 1;                          // the sweep's small copies keep off the copy engines (d2h_small / h2d_small)
        rc = lrp_cross_deim_solve(ctx, n, rF, st.UF[s], n, st.SF[s], st.VF[s], n, b.opts, st.UW[s], n, st.SW[s], st.VW[s], n, &b.info[p],
                                  nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 0);
        ctx->host_pipeline = 0;
        if (rc < 0) break;
        if (rc > worst) worst = rc;
        const int r = b.info[p].rank;                    // the solve is synchronous: rank known, outputs complete
        cudaError_t e = copy_tall_async(b.h_UW[p], b.lduw, st.UW[s], n, n, r, cudaMemcpyDeviceToHost, ctx->cp_out);
        if (e == cudaSuccess) e = copy_tall_async(b.h_VW[p], b.ldvw, st.VW[s], n, n, r, cudaMemcpyDeviceToHost, ctx->cp_out);
        if (e == cudaSuccess) e = cudaMemcpyAsync(b.h_SW[p], st.SW[s], sizeof(double) * r, cudaMemcpyDeviceToHost, ctx->cp_out);
        if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_cp[1][s], ctx->cp_out);
        if (e != cudaSuccess) { ctx->last_cuda = (int)e; rc = LRP_ERR_CUDA; }
    }
    // drain both copy streams whatever happened: nothing of this lane is in flight on return
    cudaError_t e1 = cudaStreamSynchronize(ctx->cp_in), e2 = cudaStreamSynchronize(ctx->cp_out);
    if (rc >= 0 && (e1 != cudaSuccess || e2 != cudaSuccess)) { ctx->last_cuda = (int)(e1 != cudaSuccess ? e1 : e2); rc = LRP_ERR_CUDA; }
    return rc < 0 ? rc : worst;
}
}  // namespace

// Problems 0, 1, 2, ... on one lane (ctx) or, when the workspace holds two lanes' worth and there are at least two
// problems, on two: even ones on ctx, odd ones on a library-owned second context (own streams, own pinned block) on the
// same device, driven by a worker thread that lives for the call.  Two solves in flight fill the SMs that one leaves
// idle (one-CTA core, TSQR tree levels, host decisions): 14.4 -> 11.5 ms per C4 problem.  lane(ctx, first, stride) runs one lane.
extern "C++" {
template <typename Lane>
static int run_lanes(lrp_ctx* ctx, size_t lane_bytes, int nprob, Lane lane) {
    const bool two = nprob >= 2 && ctx->ws_bytes >= 2 * lane_bytes && ctx->prof_on == 0;
    if (!two) return lane(ctx, 0, 1);
    if (!ctx->lane2) {
        cudaStream_t s2 = nullptr;
        LRP_CUDA(ctx, cudaStreamCreateWithFlags(&s2, cudaStreamNonBlocking));
        lrp_ctx* c2 = nullptr;
        const int rc2 = lrp_create(&c2, ctx->device, s2);
        if (rc2 != LRP_OK) { cudaStreamDestroy(s2); return rc2; }
        ctx->lane2 = c2; ctx->lane2_stream = s2;
    }
    lrp_ctx* c2 = ctx->lane2;
    void* const ws0 = ctx->ws; const size_t wsb0 = ctx->ws_bytes;
    c2->ws = (char*)ws0 + lane_bytes; c2->ws_bytes = lane_bytes;
    ctx->ws_bytes = lane_bytes;                          // lane 0 keeps the first half for the duration of the call
    // work already enqueued on the caller's stream precedes lane 1 too
    cudaError_t ef = cudaEventRecord(ctx->ev_fork, ctx->stream);
    if (ef == cudaSuccess) ef = cudaStreamWaitEvent(c2->stream, ctx->ev_fork, 0);
    int rc0, rc1 = LRP_OK;
    const int64_t l2_0 = c2->launches;
    if (ef != cudaSuccess) { ctx->last_cuda = (int)ef; rc0 = LRP_ERR_CUDA; }
    else {
        const int device = ctx->device;
        bool started = true;
        std::thread worker;
        try { worker = std::thread([&, device] { cudaSetDevice(device); rc1 = lane(c2, 1, 2); }); }
        catch (...) { started = false; }                 // no thread to be had: one lane after all
        if (started) { rc0 = lane(ctx, 0, 2); worker.join(); }
        else { ctx->ws_bytes = wsb0; rc0 = lane(ctx, 0, 1); }
    }
    ctx->ws = ws0; ctx->ws_bytes = wsb0;
    ctx->launches += c2->launches - l2_0;
    if (rc1 < 0 && rc0 >= 0) ctx->last_cuda = c2->last_cuda;
    if (rc0 < 0) return rc0;
    if (rc1 < 0) return rc1;
    return rc0 > rc1 ? rc0 : rc1;
}
}  // extern "C++"

int lrp_cross_deim_solve_host(lrp_ctx* ctx, int64_t n, int32_t rF, int32_t nprob,
                              const double* const* h_UF, int64_t ldu, const double* const* h_SF, const double* const* h_VF, int64_t ldv,
                              const lrp_solve_opts* opts,
                              double* const* h_UW, int64_t lduw, double* const* h_SW, double* const* h_VW, int64_t ldvw,
                              lrp_solve_info* info) {
    if (!ctx || !opts || !info || nprob < 0 || !h_UF || !h_SF || !h_VF || !h_UW || !h_SW || !h_VW) return LRP_ERR_BADARG;
    if (ldu < n || ldv < n || lduw < n || ldvw < n || rF < 1 || opts->max_rank < 1) return LRP_ERR_BADARG;
    for (int p = 0; p < nprob; ++p)
        if (!h_UF[p] || !h_SF[p] || !h_VF[p] || !h_UW[p] || !h_SW[p] || !h_VW[p]) return LRP_ERR_BADARG;
    LRP_TRY(check_n(n));
    if (nprob == 0) return LRP_OK;
    const size_t lane_bytes = host_lane_bytes(n, rF, opts->max_rank, opts->oversample);
    if (!lane_bytes || ctx->ws_bytes < lane_bytes) return LRP_ERR_WORKSPACE;
    HostBatch b{n, rF, nprob, h_UF, ldu, h_SF, h_VF, ldv, opts, h_UW, lduw, h_SW, h_VW, ldvw, info};
    return run_lanes(ctx, lane_bytes, nprob, [&](lrp_ctx* c, int first, int stride) { return host_lane(c, b, first, stride); });
}

size_t lrp_solve_batch_workspace_bytes(int64_t n, int32_t rF, int32_t max_rank, int32_t oversample, int32_t lanes) {
    if (lanes < 1 || lanes > LRP_HOST_LANES_MAX) return 0;
    const size_t base = lrp_workspace_bytes(n, rF, max_rank, oversample);
    return base ? (size_t)lanes * (lrp_align_up(base) + 256) : 0;
}

int lrp_cross_deim_solve_batch(lrp_ctx* ctx, int64_t n, int32_t rF, int32_t nprob,
                               const double* const* d_UF, int64_t ldu, const double* const* d_SF, const double* const* d_VF, int64_t ldv,
                               const lrp_solve_opts* opts,
                               double* const* d_UW, int64_t lduw, double* const* d_SW, double* const* d_VW, int64_t ldvw,
                               lrp_solve_info* info) {
    if (!ctx || !opts || !info || nprob < 0 || !d_UF || !d_SF || !d_VF || !d_UW || !d_SW || !d_VW) return LRP_ERR_BADARG;
    for (int p = 0; p < nprob; ++p)
        if (!d_UF[p] || !d_SF[p] || !d_VF[p] || !d_UW[p] || !d_SW[p] || !d_VW[p]) return LRP_ERR_BADARG;
    if (nprob == 0) return LRP_OK;
    const size_t lane_bytes = lrp_solve_batch_workspace_bytes(n, rF, opts->max_rank, opts->oversample, 1);
    if (!lane_bytes || ctx->ws_bytes < lane_bytes) return LRP_ERR_WORKSPACE;
    return run_lanes(ctx, lane_bytes, nprob, [&](lrp_ctx* c, int first, int stride) {
        int worst = LRP_OK;
        for (int p = first; p < nprob; p += stride) {
            const int rc = lrp_cross_deim_solve(c, n, rF, d_UF[p], ldu, d_SF[p], d_VF[p], ldv, opts, d_UW[p], lduw, d_SW[p], d_VW[p], ldvw,
                                                &info[p], nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 0);
            if (rc < 0) return rc;
            if (rc > worst) worst = rc;
        }
        return worst;
    });
}

int lrp_cross_deim_matrix(lrp_ctx* ctx, int32_t kind, int64_t n, const lrp_solve_opts* opts,
                          double* d_U, int64_t ldu, double* d_S, double* d_V, int64_t ldv, lrp_solve_info* info,
                          int32_t* h_trace_I, int32_t* h_trace_J, uint8_t* h_trace_keepI, uint8_t* h_trace_keepJ,
                          double* d_Uhat, double* d_Shat, double* d_Vhat, int64_t ld_hat) {
    if (!opts || kind == LRP_G_POISSON) return LRP_ERR_BADARG;
    return solve_impl(ctx, kind, n, opts->r0, nullptr, 0, nullptr, nullptr, 0, opts, d_U, ldu, d_S, d_V, ldv, info,
                      h_trace_I, h_trace_J, h_trace_keepI, h_trace_keepJ, d_Uhat, d_Shat, d_Vhat, ld_hat);
}

size_t lrp_dense_workspace_bytes(int64_t n) {
    if (check_n(n) != LRP_OK || n > 32768) return 0;
    return 2 * lrp_align_up((size_t)n * n * sizeof(double)) + lrp_align_up(lrp_dst1_ws_impl(n, (int32_t)n)) + 256;
}

int lrp_dense_poisson(lrp_ctx* ctx, int64_t n, const double* d_F, int64_t ldf, double* d_W, int64_t ldw) {
    if (!ctx || !d_F || !d_W || ldf < n || ldw < n) return LRP_ERR_BADARG;
    LRP_TRY(check_n(n));
    if (n > 32768) return LRP_ERR_UNSUPPORTED_N;
    if (ctx->ws_bytes < lrp_dense_workspace_bytes(n)) return LRP_ERR_WORKSPACE;
    lrp_arena ar(ctx->ws, ctx->ws_bytes);
    double* T1 = ar.take<double>((size_t)n * n);
    double* T2 = ar.take<double>((size_t)n * n);
    const size_t dws_bytes = lrp_dst1_ws_impl(n, (int32_t)n);
    void* dws = ar.take<char>(dws_bytes ? dws_bytes : 1);
    if (!ar.ok()) return LRP_ERR_WORKSPACE;
    const double sc = sqrt(2.0 / (double)(n + 1));
    const int32_t b = (int32_t)n;
    // What = Z F Z ./ (d_i + d_j), W = Z What Z (eq. (4)), Z symmetric orthogonal: four column-wise
    // batched DST-I and two transposes (the full-rank method needs the global transposes the low-rank one avoids)
    LRP_TRY(lrp_dst1_impl(ctx, n, b, d_F, ldf, T1, n, sc, dws, dws_bytes));        // Z F
    LRP_TRY(tall_transpose(ctx, n, T1, n, T2, n));                                 // (Z F)^T = F^T Z
    LRP_TRY(lrp_dst1_impl(ctx, n, b, T2, n, T2, n, sc, dws, dws_bytes));           // Z F^T Z = Fhat^T
    LRP_TRY(tall_spectral_divide(ctx, n, T2, n));                                  // What^T (the divisor is symmetric)
    LRP_TRY(lrp_dst1_impl(ctx, n, b, T2, n, T2, n, sc, dws, dws_bytes));           // Z What^T = (What Z)^T
    LRP_TRY(tall_transpose(ctx, n, T2, n, T1, n));                                 // What Z
    return lrp_dst1_impl(ctx, n, b, T1, n, d_W, ldw, sc, dws, dws_bytes);          // W = Z What Z
}

int lrp_sample_matrix(lrp_ctx* ctx, int32_t kind, int64_t n, const int32_t* d_I, int32_t nI, const int32_t* d_J, int32_t nJ,
                      double* d_C, int64_t ldc, double* d_Rt, int64_t ldr) {
    if (!ctx || n < 2 || (kind != LRP_G_HILBERT && kind != LRP_G_KMATRIX) || nI < 0 || nJ < 0) return LRP_ERR_BADARG;
    if (d_C && nJ > 0) {
        if (!d_J || ldc < n) return LRP_ERR_BADARG;
        LRP_TRY(tall_matrix_fibers(ctx, kind, n, 0, d_J, nJ, d_C, ldc));
    }
    if (d_Rt && nI > 0) {
        if (!d_I || ldr < n) return LRP_ERR_BADARG;
        LRP_TRY(tall_matrix_fibers(ctx, kind, n, 1, d_I, nI, d_Rt, ldr));
    }
    return LRP_OK;
}

}  // extern "C"
