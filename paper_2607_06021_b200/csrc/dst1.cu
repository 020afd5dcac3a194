// dst1.cu -- batched DST-I for n + 1 = N = 2^p, fp64, one column per FFT,
// every column transformed along its own contiguous dimension (no transpose).
//
// Algorithm: the odd extension of x has a purely imaginary spectrum; instead of the
// length-2N complex FFT the column is folded into ONE complex FFT of length L = N/2:
//   t_0 = 0,  t_m = sin(pi m/N) (x_m + x_{N-m}) + (x_m - x_{N-m})/2           (real, length N)
//   z_j = t_{2j} + i t_{2j+1},  Z = FFT_L(z),  T_k = E_k + e^{-2 pi i k/N} O_k   (real-FFT untangle)
//   X_{2k} = -Im T_k,   X_1 = T_0/2,   X_{2k+1} = X_{2k-1} + Re T_k            (prefix sum over k)
// Regimes: N < 64 definition sum; N <= 16384 one CTA per column group, column resident in shared memory,
// one HBM pass; larger N a four-step split L = L1*L2 (two strided/contiguous shared-memory FFT sweeps,
// twiddle between) followed by the untangle + scan sweep.
#include "common.cuh"
#include "fft_smem.cuh"
#include <math.h>

namespace {

// ------------------------------------------------------------------------------------------ tiny n
__global__ void dst1_naive_kernel(int n, const double* __restrict__ in, int64_t ld_in,
                                  double* __restrict__ out, int64_t ld_out, double scale) {
    __shared__ double xs[64];
    const int N = n + 1;
    const double* x = in + (int64_t)blockIdx.x * ld_in;
    for (int j = threadIdx.x; j < n; j += blockDim.x) xs[j] = x[j];
    __syncthreads();
    for (int k = threadIdx.x + 1; k <= n; k += blockDim.x) {
        double acc = 0.0;
        for (int j = 1; j <= n; ++j) acc += xs[j - 1] * sinpi((double)((j * k) % (2 * N)) / (double)N);
        out[(int64_t)blockIdx.x * ld_out + (k - 1)] = scale * acc;
    }
}

// ------------------------------------------------------------------------------------------ one-pass regime
template <int Q> struct SmallCfg {
    static constexpr int L = 1 << Q, N = 2 * L, GS = L / 8;
    static constexpr int CPB = GS >= 256 ? 1 : 256 / GS;
    static constexpr int NT = GS * CPB;
    static constexpr int PL = L + 1;
    static constexpr int NHI = N / 64 + 1;
    static constexpr size_t SMEM = sizeof(double2) * (64 + NHI) + sizeof(double) * ((size_t)CPB * 2 * PL + 64 * CPB);
};

template <int Q>
__global__ void __launch_bounds__(SmallCfg<Q>::NT)
dst1_small_kernel(int batch, const double* __restrict__ in, int64_t ld_in,
                  double* __restrict__ out, int64_t ld_out, double scale) {
    using C = SmallCfg<Q>;
    constexpr int L = C::L, N = C::N, GS = C::GS, PL = C::PL;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* lo = (double2*)smem_raw;
    double2* hi = lo + 64;
    double* data = (double*)(hi + C::NHI);
    const int tid = threadIdx.x;
    const int g = tid / GS, gt = tid % GS;
    const int col = blockIdx.x * C::CPB + g;
    const bool active = col < batch;
    double* re = data + (size_t)g * 2 * PL;
    double* im = re + PL;
    double* wsum = data + (size_t)C::CPB * 2 * PL + 64 * g;
    const double* x = in + (int64_t)(active ? col : 0) * ld_in;      // x_m = x[m-1]

    // global loads first (8 pairs in flight per thread), table build overlaps their latency
    double xa[8], xb[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int m = gt + i * GS;                                         // 0 .. L-1
        xa[i] = (active && m >= 1) ? x[m - 1] : 0.0;
        xb[i] = (active && m >= 1) ? x[N - m - 1] : 0.0;
    }
    double xmid = (active && gt == 0) ? x[L - 1] : 0.0;
    tw_build(lo, hi, 2 * N, C::NHI, tid, C::NT);                      // exp(-2 pi i u/(2N)) = exp(-i pi u/N)
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int m = gt + i * GS;
        double s = -tw_get(lo, hi, m).y;                             // sin(pi m / N)
        double sum = s * (xa[i] + xb[i]), dif = 0.5 * (xa[i] - xb[i]);
        double* arr = (m & 1) ? im : re;
        arr[PADI(m >> 1)] = sum + dif;                               // t_m   (t_0 = 0 since xa = xb = 0)
        if (m >= 1) arr[PADI((N - m) >> 1)] = sum - dif;             // t_{N-m}
    }
    if (gt == 0) ((L & 1) ? im : re)[PADI(L >> 1)] = 2.0 * xmid;     // t_L = 2 x_L
    __syncthreads();

    fft_smem<Q, C::CPB>(re, im, gt, g, lo, hi, 4);                              // exp(-2 pi i mm/L) = tw(4 mm)

    // untangle: pairs (k, L-k), k = 0 .. L/2
    for (int k = gt; k <= L / 2; k += GS) {
        if (k == 0) {
            double a = re[0], b = im[0];
            re[0] = 0.5 * (a + b);                                   // X_1 = T_0 / 2
            im[0] = 0.5 * (b - a);                                   // X_{N-1} = -T_L / 2 = (Im Z_0 - Re Z_0)/2
        } else {
            int km = L - k;
            double ak = re[PADI(k)], bk = im[PADI(k)], am = re[PADI(km)], bm = im[PADI(km)];
            double2 E = make_double2(0.5 * (ak + am), 0.5 * (bk - bm));
            double2 O = make_double2(0.5 * (bk + bm), -0.5 * (ak - am));
            double2 wO = cmul(tw_get(lo, hi, 2 * k), O);             // exp(-2 pi i k/N) O_k
            re[PADI(k)] = E.x + wO.x;      im[PADI(k)] = -(E.y + wO.y);     // R_k, X_{2k}
            re[PADI(km)] = E.x - wO.x;     im[PADI(km)] = E.y - wO.y;       // R_{L-k}, X_{2(L-k)}
        }
    }
    __syncthreads();

    // Odd outputs P_k = X_{2k+1}: a TWO-SIDED prefix sum.  Lower half forward from P_0 = X_1 (P_k = P_{k-1} + R_k), upper
    // half backward from the independently known P_{L-1} = X_{N-1} (P_{k-1} = P_k - R_k): every output is reached
    // through the shorter chain, and the (small) tail of a decaying spectrum is summed from small terms only.
    {
        constexpr int HS = GS / 2;                                   // threads per half
        const int half = gt / HS, ht = gt % HS;
        double loc[8];
        double run = 0.0;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int j = ht * 8 + i;                                // position in the half's sequence
            double v;
            if (half == 0) v = re[PADI(j)];                          // R_j (re[0] = X_1)
            else v = (j == 0) ? im[0] : -re[PADI(L - j)];            // u_0 = X_{N-1}, u_j = -R_{L-j}
            run += v; loc[i] = run;
        }
        __syncthreads();                                             // all inputs read before any output is written
        double incl = group_scan_incl<HS>(run, ht, wsum + 32 * half);
        double off = incl - run;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int j = ht * 8 + i;
            re[PADI(half == 0 ? j : L - 1 - j)] = loc[i] + off;      // P_j  /  P_{L-1-j}
        }
    }
    __syncthreads();

    if (active) {
        double* o = out + (int64_t)col * ld_out;
        for (int idx = gt; idx < N - 1; idx += GS) {                 // X_m at o[m-1]
            double val = (idx & 1) ? im[PADI((idx + 1) >> 1)] : re[PADI(idx >> 1)];
            o[idx] = scale * val;
        }
    }
}

template <int Q>
int launch_small(lrp_ctx* ctx, int batch, const double* in, int64_t ld_in, double* out, int64_t ld_out, double scale) {
    using C = SmallCfg<Q>;
    int grid = (batch + C::CPB - 1) / C::CPB;
    LRP_PROF(ctx, K_DST_SMALL, 16.0 * (2 * C::L - 1) * batch, 0);
    dst1_small_kernel<Q><<<grid, C::NT, C::SMEM, ctx->stream>>>(batch, in, ld_in, out, ld_out, scale);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}
#define LRP_Q_SWITCH(q, FN, ...)                        \
    switch (q) {                                        \
        case 5: return FN<5>(__VA_ARGS__);              \
        case 6: return FN<6>(__VA_ARGS__);              \
        case 7: return FN<7>(__VA_ARGS__);              \
        case 8: return FN<8>(__VA_ARGS__);              \
        case 9: return FN<9>(__VA_ARGS__);              \
        case 10: return FN<10>(__VA_ARGS__);            \
        case 11: return FN<11>(__VA_ARGS__);            \
        case 12: return FN<12>(__VA_ARGS__);            \
        case 13: return FN<13>(__VA_ARGS__);            \
        default: return LRP_ERR_UNSUPPORTED_N;          \
    }
int dispatch_small(int q, lrp_ctx* ctx, int batch, const double* in, int64_t ld_in, double* out, int64_t ld_out, double scale) {
    LRP_Q_SWITCH(q, launch_small, ctx, batch, in, ld_in, out, ld_out, scale)
}
template <int Q>
int init_small(lrp_ctx* ctx) {
    LRP_CUDA(ctx, cudaFuncSetAttribute(dst1_small_kernel<Q>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SmallCfg<Q>::SMEM));
    return LRP_OK;
}
}  // namespace

// dynamic shared memory opt-in of every DST-I kernel: once per context (lrp_create), not per call
int lrp_dst1_init(lrp_ctx* ctx) {
    LRP_TRY(init_small<5>(ctx)); LRP_TRY(init_small<6>(ctx)); LRP_TRY(init_small<7>(ctx)); LRP_TRY(init_small<8>(ctx));
    LRP_TRY(init_small<9>(ctx)); LRP_TRY(init_small<10>(ctx)); LRP_TRY(init_small<11>(ctx)); LRP_TRY(init_small<12>(ctx));
    LRP_TRY(init_small<13>(ctx));
    LRP_TRY(dst1_large_init(ctx));
    return dst1_bluestein_init(ctx);
}

size_t lrp_dst1_ws_impl(int64_t n, int32_t batch) {
    int64_t N = n + 1;
    if (batch <= 0) return 0;
    if (!lrp_is_pow2(N)) return dst1_bluestein_ws(n, batch);
    if (N <= 16384) return 0;
    return dst1_large_ws(N, batch);
}

int lrp_dst1_impl(lrp_ctx* ctx, int64_t n, int32_t batch, const double* d_in, int64_t ld_in,
                  double* d_out, int64_t ld_out, double scale, void* ws, size_t ws_bytes) {
    if (batch == 0) return LRP_OK;
    const int64_t N = n + 1;
    if (!lrp_is_pow2(N)) return dst1_bluestein(ctx, n, batch, d_in, ld_in, d_out, ld_out, scale, ws, ws_bytes);
    if (N < 64) {
        LRP_PROF(ctx, K_DST_NAIVE, 16.0 * n * batch, 0);
        dst1_naive_kernel<<<batch, 32, 0, ctx->stream>>>((int)n, d_in, ld_in, d_out, ld_out, scale);
        LRP_LAUNCHED(ctx);
        return LRP_OK;
    }
    const int log2N = lrp_ilog2(N);
    if (N <= 16384) return dispatch_small(log2N - 1, ctx, batch, d_in, ld_in, d_out, ld_out, scale);
    if (ws_bytes < dst1_large_ws(N, batch)) return LRP_ERR_WORKSPACE;
    return dst1_large(ctx, log2N, batch, d_in, ld_in, d_out, ld_out, scale, ws, ws_bytes);
}
