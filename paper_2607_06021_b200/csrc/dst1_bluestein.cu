// dst1_bluestein.cu -- batched DST-I for GENERAL n (n + 1 = N not a power of two; the paper's own grids are n = 2^10..2^18,
// PAPER.md:274), by Bluestein's chirp-z identity  j k = (j^2 + k^2 - (k - j)^2) / 2:
//     X_k = sum_{j=1..n} x_j sin(pi j k / N) = Im[ w_k  sum_j (x_j w_j) conj(w_{k-j}) ],    w_m = exp(i pi m^2 / (2N)),
// a linear convolution of a_j = x_j w_j with the chirp c_m = conj(w_m), |m| < n, evaluated as a circular convolution of
// power-of-two length P >= 2N:  y = IFFT_P( FFT_P(a) . FFT_P(c) ).  The chirp arguments are reduced exactly in integer
// arithmetic (m^2 mod 4N) before sincospi.  Every column is transformed along its own contiguous dimension (no
// transpose between the dimensions of the 2-D problem).
//   P <= 8192 : one CTA per column, everything in shared memory (radix-8 Stockham FFT of fft_smem.cuh).
//   P <= 2^24 : four-step split P = L1 * L2 through a complex workspace, three kernels per transform and NO transpose:
//               A  (tile of j2, all j1): chirp multiply, FFTs over j1, twiddle          -> W[k1][j2]
//               B  (rows k1):            FFT over j2, times Chat[k1][k2], inverse FFT over k2 (same rows!) -> W[k1][j2']
//               A' (tile of j2', all k1): conjugate twiddle, inverse FFTs over k1, post-chirp, Im     -> out[j1 L2 + j2' - 1]
//               (the inverse four-step runs the stages backwards, so the [k1][k2] layout of the forward result is
//               exactly what it consumes).
// About 8-16x the work of the power-of-two path of dst1.cu / dst1_large.cu (three complex FFTs of 2-4x the length).
#include "common.cuh"
#include "fft_smem.cuh"
#include <math.h>

namespace {

// w_m = exp(i pi m^2 / (2N)), argument reduced exactly: m^2 mod 4N
__device__ __forceinline__ double2 chirp(int64_t m, int64_t N) {
    const int64_t q = (m * m) % (4 * N);
    double s, c; sincospi((double)q / (double)(2 * N), &s, &c);
    return make_double2(c, s);
}
__device__ __forceinline__ double2 conj2(double2 a) { return make_double2(a.x, -a.y); }

// ------------------------------------------------------------------------------------------------ P <= 8192
template <int Q> struct BsCfg {
    static constexpr int P = 1 << Q, GS = P / 8, NT = GS;          // Q >= 8: whole warps
    static constexpr int NHI = P / 64 + 1;
    static constexpr size_t SMEM = sizeof(double) * 2 * (P + 16) + sizeof(double2) * (64 + NHI);
};

// mode 0: Chat = FFT_P(c wrapped) -> chat (one CTA).  mode 1: transform column blockIdx.x.
template <int Q>
__global__ void __launch_bounds__(BsCfg<Q>::NT)
bluestein_small_kernel(int mode, int64_t n, const double* __restrict__ in, int64_t ld_in, double* __restrict__ out, int64_t ld_out,
                       double scale, double2* __restrict__ chat) {
    using C = BsCfg<Q>;
    constexpr int P = C::P, GS = C::GS, NT = C::NT;
    extern __shared__ __align__(16) unsigned char bs_raw[];
    double* re = (double*)bs_raw;
    double* im = re + P + 16;
    double2* lo = (double2*)(im + P + 16);
    double2* hi = lo + 64;
    const int tid = threadIdx.x;
    const int64_t N = n + 1;
    tw_build(lo, hi, P, C::NHI, tid, NT);
    if (mode == 0) {
        for (int e = tid; e < P; e += NT) {
            // wrapped index e <-> m = e (0 <= e < n) or m = e - P (P - n < e < P)
            double2 v = make_double2(0.0, 0.0);
            if (e < n) v = conj2(chirp(e, N));
            else if (e > P - n) v = conj2(chirp((int64_t)e - P, N));
            re[PADI(e)] = v.x; im[PADI(e)] = v.y;
        }
    } else {
        const double* x = in + (int64_t)blockIdx.x * ld_in;
        for (int e = tid; e < P; e += NT) {
            double2 v = make_double2(0.0, 0.0);
            if (e >= 1 && e <= n) { const double2 w = chirp(e, N); const double xv = x[e - 1]; v = make_double2(xv * w.x, xv * w.y); }
            re[PADI(e)] = v.x; im[PADI(e)] = v.y;
        }
    }
    __syncthreads();
    fft_smem<Q, 1>(re, im, tid, 0, lo, hi, 1);
    __syncthreads();
    if (mode == 0) {
        for (int e = tid; e < P; e += NT) chat[e] = make_double2(re[PADI(e)], im[PADI(e)]);
        return;
    }
    for (int e = tid; e < P; e += NT) {              // times Chat, conjugated: IFFT(z) = conj(FFT(conj z)) / P
        const double2 z = cmul(make_double2(re[PADI(e)], im[PADI(e)]), chat[e]);
        re[PADI(e)] = z.x; im[PADI(e)] = -z.y;
    }
    __syncthreads();
    fft_smem<Q, 1>(re, im, tid, 0, lo, hi, 1);
    __syncthreads();
    double* o = out + (int64_t)blockIdx.x * ld_out;
    const double sc = scale / (double)P;
    for (int e = tid + 1; e <= n; e += NT) {
        const double2 y = make_double2(re[PADI(e)], -im[PADI(e)]);
        const double2 w = chirp(e, N);
        o[e - 1] = sc * (w.x * y.y + w.y * y.x);      // Im(w y)
    }
}

// ------------------------------------------------------------------------------------------------ P > 8192: four-step
constexpr int BL_TL = 13, BL_NT = (1 << BL_TL) / 8;      // 8192 points, 1024 threads per CTA

template <int QF> struct BlRowCfg {                      // a CTA holds R rows of length LF = 2^QF
    static constexpr int LF = 1 << QF, GS = LF / 8, R = (1 << BL_TL) / LF;
    static constexpr int RS = LF + 16;
    static constexpr int NHI = LF / 64 + 1;
    static constexpr size_t SMEM = sizeof(double) * 2 * (size_t)R * RS + sizeof(double2) * (64 + NHI);
};

__device__ __forceinline__ double2 twid(int64_t prod, int64_t P) {      // exp(-2 pi i prod / P), prod already reduced mod P
    double s, c; sincospi(-2.0 * (double)prod / (double)P, &s, &c);
    return make_double2(c, s);
}

// stage A (forward, mode 0/1) and stage A' (inverse, mode 2): the CTA owns R = T2 consecutive j2 and all L1 values of the
// strided index.  mode 0: input = wrapped chirp c; mode 1: input = x_j w_j; both: FFT over j1, twiddle, W[k1 L2 + j2].
// mode 2: input W[k1 L2 + j2], conjugate twiddle, inverse FFT over k1, out[j - 1] = scale/P Im(w_j y_j), j = j1 L2 + j2.
template <int Q1>
__global__ void __launch_bounds__(BL_NT)
bluestein_a_kernel(int mode, int64_t n, int q2, const double* __restrict__ in, int64_t ld_in, double* __restrict__ out,
                   int64_t ld_out, double scale, double2* __restrict__ W) {
    using C = BlRowCfg<Q1>;
    constexpr int L1 = C::LF, GS = C::GS, R = C::R, RS = C::RS;
    extern __shared__ __align__(16) unsigned char bl_raw[];
    double* re = (double*)bl_raw;
    double* im = re + (size_t)R * RS;
    double2* lo = (double2*)(im + (size_t)R * RS);
    double2* hi = lo + 64;
    const int tid = threadIdx.x;
    const int64_t N = n + 1, L2 = (int64_t)1 << q2, P = (int64_t)L1 << q2;
    const int64_t j2base = (int64_t)blockIdx.x * R;
    double2* Wc = W + (int64_t)blockIdx.y * P;
    tw_build(lo, hi, L1, C::NHI, tid, BL_NT);
    for (int e = tid; e < R * L1; e += BL_NT) {
        const int s = e % R, a1 = e / R;                   // s: j2 offset, a1: j1 (modes 0, 1) or k1 (mode 2)
        const int64_t j2 = j2base + s;
        double2 v = make_double2(0.0, 0.0);
        if (mode == 2) {
            const double2 z = __ldcg(Wc + (int64_t)a1 * L2 + j2);
            const double2 t = twid((j2 * a1) & (P - 1), P);       // forward twiddle; inverse needs its conjugate:
            const double2 zz = cmul(z, conj2(t));                   // z conj(t), then conj for the conj-FFT-conj trick
            v = make_double2(zz.x, -zz.y);
        } else {
            const int64_t j = (int64_t)a1 * L2 + j2;
            if (mode == 0) {
                if (j < n) v = conj2(chirp(j, N));
                else if (j > P - n) v = conj2(chirp(j - P, N));
            } else if (j >= 1 && j <= n) {
                const double2 w = chirp(j, N); const double xv = in[(int64_t)blockIdx.y * ld_in + j - 1];
                v = make_double2(xv * w.x, xv * w.y);
            }
        }
        re[s * RS + PADI(a1)] = v.x; im[s * RS + PADI(a1)] = v.y;
    }
    __syncthreads();
    {
        const int g = tid / GS, gt = tid % GS;             // R groups of GS threads: R * GS = 1024
        fft_smem<Q1, R>(re + g * RS, im + g * RS, gt, g, lo, hi, 1);      // R groups: named barriers, or CTA-wide when R > 15
    }
    __syncthreads();
    for (int e = tid; e < R * L1; e += BL_NT) {
        const int s = e % R, b1 = e / R;                   // b1: k1 (modes 0, 1) or j1 (mode 2)
        const int64_t j2 = j2base + s;
        const double2 v = make_double2(re[s * RS + PADI(b1)], im[s * RS + PADI(b1)]);
        if (mode == 2) {
            const int64_t j = (int64_t)b1 * L2 + j2;
            if (j >= 1 && j <= n) {
                const double2 y = make_double2(v.x, -v.y);
                const double2 w = chirp(j, N);
                out[(int64_t)blockIdx.y * ld_out + j - 1] = (scale / (double)P) * (w.x * y.y + w.y * y.x);
            }
        } else {
            __stcg(Wc + (int64_t)b1 * L2 + j2, cmul(v, twid((j2 * b1) & (P - 1), P)));
        }
    }
}

// stage B: rows k1 of W (length L2): forward FFT over j2.  mode 0: store (this is Chat, [k1][k2] layout).
// mode 1: times Chat[k1][k2], inverse FFT over k2 (the first stage of the inverse four-step acts on the same rows), store.
template <int Q2>
__global__ void __launch_bounds__(BL_NT)
bluestein_b_kernel(int mode, int q1, double2* __restrict__ W, const double2* __restrict__ chat) {
    using C = BlRowCfg<Q2>;
    constexpr int L2 = C::LF, GS = C::GS, R = C::R, RS = C::RS;
    extern __shared__ __align__(16) unsigned char bl_raw[];
    double* re = (double*)bl_raw;
    double* im = re + (size_t)R * RS;
    double2* lo = (double2*)(im + (size_t)R * RS);
    double2* hi = lo + 64;
    const int tid = threadIdx.x;
    const int64_t P = (int64_t)L2 << q1;
    const int64_t row0 = (int64_t)blockIdx.x * R;
    double2* Wc = W + (int64_t)blockIdx.y * P;
    tw_build(lo, hi, L2, C::NHI, tid, BL_NT);
    for (int e = tid; e < R * L2; e += BL_NT) {
        const int rr = e / L2, c = e % L2;
        const double2 z = __ldcg(Wc + (row0 + rr) * L2 + c);
        re[rr * RS + PADI(c)] = z.x; im[rr * RS + PADI(c)] = z.y;
    }
    __syncthreads();
    const int g = tid / GS, gt = tid % GS;
    fft_smem<Q2, R>(re + g * RS, im + g * RS, gt, g, lo, hi, 1);
    __syncthreads();
    if (mode == 1) {
        for (int e = tid; e < R * L2; e += BL_NT) {
            const int rr = e / L2, c = e % L2;
            const double2 z = cmul(make_double2(re[rr * RS + PADI(c)], im[rr * RS + PADI(c)]), chat[(row0 + rr) * L2 + c]);
            re[rr * RS + PADI(c)] = z.x; im[rr * RS + PADI(c)] = -z.y;          // conj: inverse by conj-FFT-conj
        }
        __syncthreads();
        fft_smem<Q2, R>(re + g * RS, im + g * RS, gt, g, lo, hi, 1);
        __syncthreads();
    }
    for (int e = tid; e < R * L2; e += BL_NT) {
        const int rr = e / L2, c = e % L2;
        const double sgn = mode == 1 ? -1.0 : 1.0;
        __stcg(Wc + (row0 + rr) * L2 + c, make_double2(re[rr * RS + PADI(c)], sgn * im[rr * RS + PADI(c)]));
    }
}

typedef void (*BsSmall)(int, int64_t, const double*, int64_t, double*, int64_t, double, double2*);
typedef void (*BlA)(int, int64_t, int, const double*, int64_t, double*, int64_t, double, double2*);
typedef void (*BlB)(int, int, double2*, const double2*);

struct SmallEntry { int q; BsSmall fn; size_t smem; int nt; };
const SmallEntry* small_table(int* cnt) {
    static const SmallEntry t[] = {
        {8, bluestein_small_kernel<8>, BsCfg<8>::SMEM, BsCfg<8>::NT}, {9, bluestein_small_kernel<9>, BsCfg<9>::SMEM, BsCfg<9>::NT},
        {10, bluestein_small_kernel<10>, BsCfg<10>::SMEM, BsCfg<10>::NT}, {11, bluestein_small_kernel<11>, BsCfg<11>::SMEM, BsCfg<11>::NT},
        {12, bluestein_small_kernel<12>, BsCfg<12>::SMEM, BsCfg<12>::NT}, {13, bluestein_small_kernel<13>, BsCfg<13>::SMEM, BsCfg<13>::NT}};
    *cnt = 6; return t;
}
struct RowEntry { int q; BlA fa; BlB fb; size_t smem; };
const RowEntry* row_table(int* cnt) {
    static const RowEntry t[] = {
        {7, bluestein_a_kernel<7>, bluestein_b_kernel<7>, BlRowCfg<7>::SMEM}, {8, bluestein_a_kernel<8>, bluestein_b_kernel<8>, BlRowCfg<8>::SMEM},
        {9, bluestein_a_kernel<9>, bluestein_b_kernel<9>, BlRowCfg<9>::SMEM}, {10, bluestein_a_kernel<10>, bluestein_b_kernel<10>, BlRowCfg<10>::SMEM},
        {11, bluestein_a_kernel<11>, bluestein_b_kernel<11>, BlRowCfg<11>::SMEM}, {12, bluestein_a_kernel<12>, bluestein_b_kernel<12>, BlRowCfg<12>::SMEM}};
    *cnt = 6; return t;
}

int bluestein_logP(int64_t n) { int q = 8; while (((int64_t)1 << q) < 2 * (n + 1)) ++q; return q; }
int group_cols(int q, int batch) {                     // columns per pass: W of a group <= 512 MB
    int64_t g = ((int64_t)512 << 20) / ((int64_t)16 << q);
    if (g < 1) g = 1;
    return (int)(g < batch ? g : batch);
}

}  // namespace

int dst1_bluestein_init(lrp_ctx* ctx) {
    int c; const SmallEntry* st = small_table(&c);
    for (int i = 0; i < c; ++i) LRP_CUDA(ctx, cudaFuncSetAttribute(st[i].fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)st[i].smem));
    const RowEntry* rt = row_table(&c);
    for (int i = 0; i < c; ++i) {
        LRP_CUDA(ctx, cudaFuncSetAttribute(rt[i].fa, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rt[i].smem));
        LRP_CUDA(ctx, cudaFuncSetAttribute(rt[i].fb, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rt[i].smem));
    }
    return LRP_OK;
}

bool dst1_bluestein_supported(int64_t n) { return n >= 1 && bluestein_logP(n) <= 24; }

size_t dst1_bluestein_ws(int64_t n, int32_t batch) {
    if (!dst1_bluestein_supported(n) || batch <= 0) return 0;
    const int q = bluestein_logP(n);
    size_t b = lrp_align_up(sizeof(double2) << q);                                   // Chat
    if (q > 13) b += lrp_align_up(((size_t)group_cols(q, batch) * sizeof(double2)) << q);   // W
    return b;
}

int dst1_bluestein(lrp_ctx* ctx, int64_t n, int32_t batch, const double* d_in, int64_t ld_in, double* d_out, int64_t ld_out,
                   double scale, void* ws, size_t ws_bytes) {
    if (!dst1_bluestein_supported(n)) return LRP_ERR_UNSUPPORTED_N;
    if (ws_bytes < dst1_bluestein_ws(n, batch)) return LRP_ERR_WORKSPACE;
    const int q = bluestein_logP(n);
    double2* chat = (double2*)ws;
    if (q <= 13) {
        int c; const SmallEntry* st = small_table(&c); const SmallEntry* e = nullptr;
        for (int i = 0; i < c; ++i) if (st[i].q == q) e = &st[i];
        if (!e) return LRP_ERR_UNSUPPORTED_N;
        LRP_PROF(ctx, K_DST_BLUESTEIN, 0, 0);
        e->fn<<<1, e->nt, e->smem, ctx->stream>>>(0, n, nullptr, 0, nullptr, 0, 1.0, chat);
        LRP_LAUNCHED(ctx);
        LRP_PROF(ctx, K_DST_BLUESTEIN, 16.0 * n * batch, 0);
        e->fn<<<batch, e->nt, e->smem, ctx->stream>>>(1, n, d_in, ld_in, d_out, ld_out, scale, chat);
        LRP_LAUNCHED(ctx);
        return LRP_OK;
    }
    const int q1 = q / 2, q2 = q - q1;                   // 7 <= q1 <= q2 <= 12
    int c; const RowEntry* rt = row_table(&c); const RowEntry *e1 = nullptr, *e2 = nullptr;
    for (int i = 0; i < c; ++i) { if (rt[i].q == q1) e1 = &rt[i]; if (rt[i].q == q2) e2 = &rt[i]; }
    if (!e1 || !e2) return LRP_ERR_UNSUPPORTED_N;
    double2* W = (double2*)((char*)ws + lrp_align_up(sizeof(double2) << q));
    const int RA = (1 << BL_TL) >> q1, RB = (1 << BL_TL) >> q2;
    const unsigned gA = (unsigned)(((int64_t)1 << q2) / RA), gB = (unsigned)(((int64_t)1 << q1) / RB);
    // Chat in the [k1][k2] layout of the forward four-step
    LRP_PROF(ctx, K_DST_BLUESTEIN, 0, 0);
    e1->fa<<<dim3(gA, 1), BL_NT, e1->smem, ctx->stream>>>(0, n, q2, nullptr, 0, nullptr, 0, 1.0, chat);
    LRP_LAUNCHED(ctx);
    LRP_PROF(ctx, K_DST_BLUESTEIN, 0, 0);
    e2->fb<<<dim3(gB, 1), BL_NT, e2->smem, ctx->stream>>>(0, q1, chat, nullptr);
    LRP_LAUNCHED(ctx);
    const int gc = group_cols(q, batch);
    for (int c0 = 0; c0 < batch; c0 += gc) {
        const int cols = batch - c0 < gc ? batch - c0 : gc;
        const double* in = d_in + (int64_t)c0 * ld_in; double* out = d_out + (int64_t)c0 * ld_out;
        LRP_PROF(ctx, K_DST_BLUESTEIN, 16.0 * n * cols, 0);
        e1->fa<<<dim3(gA, cols), BL_NT, e1->smem, ctx->stream>>>(1, n, q2, in, ld_in, nullptr, 0, 1.0, W);
        LRP_LAUNCHED(ctx);
        LRP_PROF(ctx, K_DST_BLUESTEIN, 0, 0);
        e2->fb<<<dim3(gB, cols), BL_NT, e2->smem, ctx->stream>>>(1, q1, W, chat);
        LRP_LAUNCHED(ctx);
        LRP_PROF(ctx, K_DST_BLUESTEIN, 0, 0);
        e1->fa<<<dim3(gA, cols), BL_NT, e1->smem, ctx->stream>>>(2, n, q2, nullptr, 0, out, ld_out, scale, W);
        LRP_LAUNCHED(ctx);
    }
    return LRP_OK;
}
