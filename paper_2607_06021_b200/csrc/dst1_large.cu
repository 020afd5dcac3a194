// dst1_large.cu -- batched DST-I for N = n + 1 = 2^p > 16384: the column no longer fits one CTA's shared memory.
//
// Same folding as dst1.cu (t -> z, complex FFT of length L = N/2, untangle, prefix sum), with the FFT split
// four-step style, L = L1 * L2, j = j1*L2 + j2, k = k1 + L1*k2:
//   sweep A: fold x on the fly (every x element enters exactly two t's: the CTA owns a j2 tile AND its mirror tile,
//            so each element is fetched from HBM once), length-L1 FFTs over the strided index j1, four-step twiddle,
//            W[k1*L2 + j2] (complex, 8N bytes per column);
//   sweep B: the CTA owns T rows k1 and their mirror rows L1 - k1: length-L2 FFTs, real-FFT untangle of the pairs
//            (k, L-k) in shared memory, writes X_{2k} (final) and R_k = X_{2k+1} - X_{2k-1} in natural order;
//   sweep C: in-place prefix sum over the odd outputs (chunk sums, scan of the chunk sums, apply).
// Columns are processed in groups whose W + output footprint stays L2-resident, so that ideally only the read of x
// and the final write of the output reach HBM.
#include "common.cuh"
#include "fft_smem.cuh"
#include <math.h>
#include <stdlib.h>

namespace {

constexpr int row_stride(int Lrow, int nrows) {            // padded row length with (stride mod 16) == max(1, 16/nrows)
    int want = (16 / nrows) > 0 ? (16 / nrows) : 1;
    int base = Lrow;
    return base + (((want - base) % 16) + 16) % 16;
}

// ------------------------------------------------------------------------------------------------ sweep A
template <int Q1, int TL> struct PACfg {
    static constexpr int L1 = 1 << Q1, GS = L1 / 8;
    static constexpr int T2 = (1 << TL) / L1, T = T2 / 2;        // sub-FFTs per CTA: T of the tile + T of its mirror
    static constexpr int NT = (1 << TL) / 8;
    static constexpr int RS = row_stride(L1, T2);
    static constexpr int IMOFF = T2 * RS + 8;
    static constexpr int NHI = (2 * L1) / 64 + 1;
    static constexpr int TW_LO = 32, TW_HI = (L1 + 31) / 32;
    static constexpr int CH = 4;                  // loads in flight per thread (register budget)
    static constexpr size_t SMEM = sizeof(double2) * (64 + NHI + 2 * T2 + (size_t)T2 * (TW_LO + TW_HI)) +
                                   sizeof(double) * ((size_t)2 * IMOFF);
};

template <int Q1, int TL>
__global__ void __launch_bounds__(PACfg<Q1, TL>::NT, TL <= 12 ? 2 : 1)
dst1_pa_kernel(int log2N, const double* __restrict__ in, int64_t ld_in, double2* __restrict__ W) {
    using C = PACfg<Q1, TL>;
    constexpr int L1 = C::L1, GS = C::GS, T2 = C::T2, T = C::T, RS = C::RS, NT = C::NT;
    const int64_t N = (int64_t)1 << log2N, L = N >> 1;
    const int L2 = (int)(L >> Q1);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* lo = (double2*)smem_raw;
    double2* hi = lo + 64;
    double2* tB = hi + C::NHI;                       // [T2][2]   exp(-i pi (2 j2 + b)/N)
    double2* t4lo = tB + 2 * T2;                     // [T2][32]  exp(-2 pi i j2 l / L)
    double2* t4hi = t4lo + T2 * C::TW_LO;            // [T2][L1/32] exp(-2 pi i j2 (32 h) / L)
    double* re = (double*)(t4hi + T2 * C::TW_HI);
    double* im = re + C::IMOFF;
    const int tid = threadIdx.x;
    const int c = blockIdx.x;
    const double* x = in + (int64_t)blockIdx.y * ld_in;            // x_m = x[m-1]
    double2* Wc = W + (int64_t)blockIdx.y * L;
    auto j2_of = [&](int s) { return s < T ? c * T + s : L2 - c * T - T + (s - T); };

    tw_build(lo, hi, 2 * L1, C::NHI, tid, NT);
    for (int i = tid; i < 2 * T2; i += NT) {
        double sn, cs; sincospi(-(double)(2 * j2_of(i >> 1) + (i & 1)) / (double)N, &sn, &cs); tB[i] = make_double2(cs, sn);
    }
    for (int i = tid; i < T2 * (C::TW_LO + C::TW_HI); i += NT) {
        int s, kk; double2* dst;
        if (i < T2 * C::TW_LO) { s = i / C::TW_LO; kk = i % C::TW_LO; dst = t4lo + i; }
        else { int q = i - T2 * C::TW_LO; s = q / C::TW_HI; kk = (q % C::TW_HI) * 32; dst = t4hi + q; }
        int64_t prod = ((int64_t)j2_of(s) * kk) & (L - 1);
        double sn, cs; sincospi(-2.0 * (double)prod / (double)L, &sn, &cs); *dst = make_double2(cs, sn);
    }
    __syncthreads();
    // fold: t_m = sin(pi m/N)(x_m + x_{N-m}) + (x_m - x_{N-m})/2 for m = 2j, 2j+1;  z_j = t_{2j} + i t_{2j+1}
#pragma unroll 1
    for (int i0 = 0; i0 < 8; i0 += C::CH) {
        double x0[C::CH], x1[C::CH], y0[C::CH], y1[C::CH];
#pragma unroll
        for (int i = 0; i < C::CH; ++i) {
            int e = tid + (i0 + i) * NT;
            int s = e % T2, j1 = e / T2;
            int64_t m0 = 2 * ((int64_t)j1 * L2 + j2_of(s));
            x0[i] = (m0 >= 1) ? x[m0 - 1] : 0.0;
            x1[i] = x[m0];
            y0[i] = (m0 >= 1) ? x[N - m0 - 1] : 0.0;
            y1[i] = x[N - m0 - 2];
        }
#pragma unroll
        for (int i = 0; i < C::CH; ++i) {
            int e = tid + (i0 + i) * NT;
            int s = e % T2, j1 = e / T2;
            double2 a = tw_get(lo, hi, j1);                       // exp(-i pi j1 / L1)
            double2 b0 = tB[2 * s], b1 = tB[2 * s + 1];
            double s0 = -(a.x * b0.y + a.y * b0.x);               // sin(pi m0 / N)
            double s1 = -(a.x * b1.y + a.y * b1.x);
            re[s * RS + PADI(j1)] = s0 * (x0[i] + y0[i]) + 0.5 * (x0[i] - y0[i]);
            im[s * RS + PADI(j1)] = s1 * (x1[i] + y1[i]) + 0.5 * (x1[i] - y1[i]);
        }
    }
    __syncthreads();
    {
        const int g = tid / GS, gt = tid % GS;
        fft_smem<Q1>(re + g * RS, im + g * RS, gt, lo, hi, 2);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int s = e % T2, k1 = e / T2;
        double2 v = make_double2(re[s * RS + PADI(k1)], im[s * RS + PADI(k1)]);
        double2 w = cmul(t4hi[s * C::TW_HI + (k1 >> 5)], t4lo[s * C::TW_LO + (k1 & 31)]);
        Wc[(int64_t)k1 * L2 + j2_of(s)] = cmul(v, w);
    }
}

// ------------------------------------------------------------------------------------------------ sweep B
template <int Q2, int TL> struct PBCfg {
    static constexpr int L2 = 1 << Q2, GS = L2 / 8;
    static constexpr int R2 = (1 << TL) / L2, T = R2 / 2;        // rows per CTA: T rows k1 + their T mirror rows
    static constexpr int NT = (1 << TL) / 8;
    static constexpr int RS = row_stride(L2, R2);
    static constexpr int IMOFF = R2 * RS + 8;
    static constexpr int NHI = (2 * L2) / 64 + 1;
    static constexpr size_t SMEM = sizeof(double2) * (64 + NHI + R2) + sizeof(double) * ((size_t)2 * IMOFF);
};

// untangle one pair (k, L-k): in (zk, zm) = (Z_k, Z_{L-k}), w = exp(-2 pi i k/N);
// out zk <- (R_k, X_{2k}),  zm <- (R_{L-k}, X_{2(L-k)})       (same algebra as dst1.cu)
__device__ __forceinline__ void untangle_pair(double2& zk, double2& zm, double2 w) {
    double2 E = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y));
    double2 O = make_double2(0.5 * (zk.y + zm.y), -0.5 * (zk.x - zm.x));
    double2 wO = cmul(w, O);
    zk = make_double2(E.x + wO.x, -(E.y + wO.y));
    zm = make_double2(E.x - wO.x, E.y - wO.y);
}

template <int Q2, int TL>
__global__ void __launch_bounds__(PBCfg<Q2, TL>::NT, TL <= 12 ? 2 : 1)
dst1_pb_kernel(int log2N, const double2* __restrict__ W, double* __restrict__ out, int64_t ld_out, double scale,
               double* __restrict__ xlast, int xstride) {
    using C = PBCfg<Q2, TL>;
    constexpr int L2 = C::L2, GS = C::GS, R2 = C::R2, T = C::T, RS = C::RS, NT = C::NT;
    const int64_t N = (int64_t)1 << log2N, L = N >> 1;
    const int L1 = (int)(L >> Q2);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* lo = (double2*)smem_raw;
    double2* hi = lo + 64;
    double2* rowtw = hi + C::NHI;                    // [R2] exp(-2 pi i row/N)
    double* re = (double*)(rowtw + R2);
    double* im = re + C::IMOFF;
    const int tid = threadIdx.x;
    const int c = blockIdx.x;
    const double2* Wc = W + (int64_t)blockIdx.y * L;
    double* o = out + (int64_t)blockIdx.y * ld_out;
    auto row_of = [&](int slot) {
        int rho = c * T + (slot < T ? slot : slot - T);
        return slot < T ? rho : (rho == 0 ? L1 / 2 : L1 - rho);
    };
    double2 v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        v[i] = Wc[(int64_t)row_of(e / L2) * L2 + (e % L2)];
    }
    tw_build(lo, hi, 2 * L2, C::NHI, tid, NT);        // exp(-2 pi i u/(2 L2)) = exp(-2 pi i (L1 u)/N)
    for (int i = tid; i < R2; i += NT) {
        double sn, cs; sincospi(-2.0 * (double)row_of(i) / (double)N, &sn, &cs); rowtw[i] = make_double2(cs, sn);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int slot = e / L2, j2 = e % L2;
        re[slot * RS + PADI(j2)] = v[i].x; im[slot * RS + PADI(j2)] = v[i].y;
    }
    __syncthreads();
    {
        const int g = tid / GS, gt = tid % GS;
        fft_smem<Q2>(re + g * RS, im + g * RS, gt, lo, hi, 2);      // exp(-2 pi i mm/L2) = tw(2 mm)
    }
    // untangle: thread owns the pair {(slot r, k2), its mirror}; k = row + L1*k2
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        int e = tid + i * NT;
        int r = e / L2, k2 = e % L2;
        if (c * T + r >= 1) {                                      // general rows: mirror is (slot T+r, L2-1-k2)
            int ia = r * RS + PADI(k2), ib = (T + r) * RS + PADI(L2 - 1 - k2);
            double2 zk = make_double2(re[ia], im[ia]), zm = make_double2(re[ib], im[ib]);
            untangle_pair(zk, zm, cmul(rowtw[r], tw_get(lo, hi, k2)));
            re[ia] = zk.x; im[ia] = zk.y; re[ib] = zm.x; im[ib] = zm.y;
        } else {
            // row 0 pairs with itself: (k2, L2-k2), k2 = 1..L2/2; k2 = 0 holds T_0
            if (k2 == 0) {
                double a = re[0], b = im[0];
                re[0] = 0.5 * (a + b); im[0] = 0.0;               // R_0 := X_1 = T_0/2
                xlast[(int64_t)blockIdx.y * xstride] = scale * 0.5 * (b - a);   // X_{N-1} = -T_L/2, start of the backward sum
            } else if (k2 <= L2 / 2) {
                int ia = PADI(k2), ib = PADI(L2 - k2);
                double2 zk = make_double2(re[ia], im[ia]), zm = make_double2(re[ib], im[ib]);
                untangle_pair(zk, zm, tw_get(lo, hi, k2));
                re[ia] = zk.x; im[ia] = zk.y; re[ib] = zm.x; im[ib] = zm.y;
            }
            // slot T holds row L1/2, which also pairs with itself: (k2, L2-1-k2), k2 < L2/2
            if (k2 < L2 / 2) {
                int ia = T * RS + PADI(k2), ib = T * RS + PADI(L2 - 1 - k2);
                double2 zk = make_double2(re[ia], im[ia]), zm = make_double2(re[ib], im[ib]);
                untangle_pair(zk, zm, cmul(rowtw[T], tw_get(lo, hi, k2)));
                re[ia] = zk.x; im[ia] = zk.y; re[ib] = zm.x; im[ib] = zm.y;
            }
        }
    }
    __syncthreads();
    // natural-order output: X_{2k} at o[2k-1], R_k at o[2k]; for fixed k2 the T rows of a tile are 2T consecutive doubles
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int slot = e % R2, k2 = e / R2;
        int64_t k = (int64_t)row_of(slot) + (int64_t)L1 * k2;
        int ia = slot * RS + PADI(k2);
        o[2 * k] = scale * re[ia];
        if (k >= 1) o[2 * k - 1] = scale * im[ia];
    }
}

// ------------------------------------------------------------------------------------------------ sweep C
// Odd outputs P_k = X_{2k+1} from R_k = P_k - P_{k-1} (stored at o[2k], R_0 = X_1): a TWO-SIDED in-place sum over the
// even-index elements.  Lower half of the chunks forward from P_0 = X_1, upper half backward from the independently
// known P_{L-1} = X_{N-1} (sweep B, xlast): every output is reached through the shorter chain and the small tail of a
// decaying spectrum is summed from small terms only.  sums: per column nchunks chunk sums + 1 slot for X_{N-1}.
constexpr int SC_CHUNK = 4096, SC_NT = 512;       // k's per chunk

__global__ void __launch_bounds__(SC_NT)
dst1_chunksum_kernel(int log2N, const double* __restrict__ out, int64_t ld_out, double* __restrict__ sums) {
    const int64_t L = (int64_t)1 << (log2N - 1);
    const int nch = (int)(L / SC_CHUNK);
    const double* o = out + (int64_t)blockIdx.y * ld_out + 2 * (int64_t)blockIdx.x * SC_CHUNK;
    __shared__ double ws[32];
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < SC_CHUNK / SC_NT; ++i) acc += o[2 * (threadIdx.x + i * SC_NT)];
    for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < SC_NT / 32; ++w) t += ws[w];
        sums[(int64_t)blockIdx.y * (nch + 1) + blockIdx.x] = t;
    }
}

// per column (one CTA): chunks c < nch/2 get the exclusive prefix of the chunk sums, chunks c >= nch/2 the exclusive
// suffix (sum of the chunks above them, accumulated from the top)
__global__ void __launch_bounds__(1024)
dst1_scansums_kernel(int nchunks, double* __restrict__ sums) {
    double* s = sums + (int64_t)blockIdx.x * (nchunks + 1);
    __shared__ double wsum[32];
    __shared__ double tot;
    const int half = nchunks / 2;
    for (int dir = 0; dir < 2; ++dir) {
        const int cnt = dir == 0 ? half : nchunks - half;
        double carry = 0.0;
        for (int base = 0; base < cnt; base += 1024) {
            const int q = base + threadIdx.x;
            const int i = dir == 0 ? q : nchunks - 1 - q;
            double v = q < cnt ? s[i] : 0.0;
            double incl = group_scan_incl<1024>(v, threadIdx.x, wsum);
            if (q < cnt) s[i] = carry + incl - v;
            if (threadIdx.x == 1023) tot = incl;
            __syncthreads();
            carry += tot;
            __syncthreads();
        }
    }
}

__global__ void __launch_bounds__(SC_NT)
dst1_scanapply_kernel(int log2N, double* __restrict__ out, int64_t ld_out, const double* __restrict__ sums) {
    const int64_t L = (int64_t)1 << (log2N - 1);
    const int nch = (int)(L / SC_CHUNK);
    const bool fwd = (int)blockIdx.x < nch / 2;
    double* o = out + (int64_t)blockIdx.y * ld_out + 2 * (int64_t)blockIdx.x * SC_CHUNK;
    const double* sc = sums + (int64_t)blockIdx.y * (nch + 1);
    __shared__ double wsum[32];
    constexpr int PER = SC_CHUNK / SC_NT;          // 8 consecutive positions of the (possibly reversed) chunk per thread
    double loc[PER], val[PER]; double run = 0.0;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const int q = threadIdx.x * PER + i;
        val[i] = o[2 * (fwd ? q : SC_CHUNK - 1 - q)];
        run += val[i]; loc[i] = run;
    }
    double incl = group_scan_incl<SC_NT>(run, threadIdx.x, wsum);
    const double off = incl - run;
    if (fwd) {
        const double base = sc[blockIdx.x];
#pragma unroll
        for (int i = 0; i < PER; ++i) o[2 * (threadIdx.x * PER + i)] = base + off + loc[i];                    // P_k
    } else {
        const double xl = sc[nch], above = sc[blockIdx.x];
#pragma unroll
        for (int i = 0; i < PER; ++i)                                // P_k = X_{N-1} - sum_{m > k} R_m
            o[2 * (SC_CHUNK - 1 - (threadIdx.x * PER + i))] = xl - (above + (off + loc[i] - val[i]));
    }
}

// ------------------------------------------------------------------------------------------------ host side
template <int Q1, int TL>
int launch_pa(lrp_ctx* ctx, int log2N, int cols, const double* in, int64_t ld_in, double2* W) {
    using C = PACfg<Q1, TL>;
    LRP_CUDA(ctx, cudaFuncSetAttribute(dst1_pa_kernel<Q1, TL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    const int L2 = 1 << (log2N - 1 - Q1);
    LRP_PROF(ctx, K_DST_P1, 16.0 * ((int64_t)1 << log2N) * cols, 0);
    dst1_pa_kernel<Q1, TL><<<dim3(L2 / C::T2, cols), C::NT, C::SMEM, ctx->stream>>>(log2N, in, ld_in, W);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}
template <int Q2, int TL>
int launch_pb(lrp_ctx* ctx, int log2N, int cols, const double2* W, double* out, int64_t ld_out, double scale,
              double* xlast, int xstride) {
    using C = PBCfg<Q2, TL>;
    LRP_CUDA(ctx, cudaFuncSetAttribute(dst1_pb_kernel<Q2, TL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    const int L1 = 1 << (log2N - 1 - Q2);
    LRP_PROF(ctx, K_DST_P2, 16.0 * ((int64_t)1 << log2N) * cols, 0);
    dst1_pb_kernel<Q2, TL><<<dim3(L1 / C::R2, cols), C::NT, C::SMEM, ctx->stream>>>(log2N, W, out, ld_out, scale, xlast, xstride);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

#define LRP_QL_SWITCH(q, TLV, FN, ...)                  \
    switch (q) {                                        \
        case 7: return FN<7, TLV>(__VA_ARGS__);         \
        case 8: return FN<8, TLV>(__VA_ARGS__);         \
        case 9: return FN<9, TLV>(__VA_ARGS__);         \
        case 10: return FN<10, TLV>(__VA_ARGS__);       \
        case 11: return FN<11, TLV>(__VA_ARGS__);       \
        default: return LRP_ERR_UNSUPPORTED_N;          \
    }
int dispatch_pa(int q1, int tl, lrp_ctx* ctx, int log2N, int cols, const double* in, int64_t ld_in, double2* W) {
    if (tl == 12) { LRP_QL_SWITCH(q1, 12, launch_pa, ctx, log2N, cols, in, ld_in, W) }
    if (q1 == 12) return launch_pa<12, 13>(ctx, log2N, cols, in, ld_in, W);
    LRP_QL_SWITCH(q1, 13, launch_pa, ctx, log2N, cols, in, ld_in, W)
}
int dispatch_pb(int q2, int tl, lrp_ctx* ctx, int log2N, int cols, const double2* W, double* out, int64_t ld_out, double scale,
                double* xlast, int xstride) {
    if (tl == 12) { LRP_QL_SWITCH(q2, 12, launch_pb, ctx, log2N, cols, W, out, ld_out, scale, xlast, xstride) }
    if (q2 == 12) return launch_pb<12, 13>(ctx, log2N, cols, W, out, ld_out, scale, xlast, xstride);
    LRP_QL_SWITCH(q2, 13, launch_pb, ctx, log2N, cols, W, out, ld_out, scale, xlast, xstride)
}

// tile size and split: L = 2^q = L1 * L2 with both factors <= 2^(TL-1)
void plan(int log2N, int* tl, int* q1, int* q2) {
    const int q = log2N - 1;
    *tl = q <= 22 ? 12 : 13;
    *q2 = q / 2; *q1 = q - *q2;
    if (const char* e = getenv("LRP_DST_TL")) { int v = atoi(e); if (v == 13 && q >= 14) *tl = 13; }
    if (const char* e = getenv("LRP_DST_Q1")) { int v = atoi(e); if (v >= 7 && v <= *tl - 1 && q - v >= 7 && q - v <= *tl - 1) { *q1 = v; *q2 = q - v; } }
}

// columns per group: W + output of one group should stay L2-resident between the sweeps
int group_cols(int64_t N, int batch) {
    int64_t per_col = N * 16;
    static int64_t budget_mb = 0;
    if (budget_mb == 0) { const char* e = getenv("LRP_DST_GROUP_MB"); budget_mb = e ? atoll(e) : 4096; if (budget_mb < 1) budget_mb = 4096; }
    int g = (int)((budget_mb << 20) / per_col);
    if (g < 1) g = 1;
    if (g > batch) g = batch;
    return g;
}

}  // namespace

size_t dst1_large_ws(int64_t N, int32_t batch) {
    const int g = group_cols(N, batch);
    const int64_t L = N / 2;
    return lrp_align_up((size_t)g * L * sizeof(double2)) + lrp_align_up((size_t)g * (L / SC_CHUNK + 1) * sizeof(double));
}

int dst1_large(lrp_ctx* ctx, int log2N, int32_t batch, const double* d_in, int64_t ld_in,
               double* d_out, int64_t ld_out, double scale, void* ws, size_t ws_bytes) {
    const int64_t N = (int64_t)1 << log2N, L = N / 2;
    if (log2N > 25) return LRP_ERR_UNSUPPORTED_N;
    int tl, q1, q2; plan(log2N, &tl, &q1, &q2);
    const int g = group_cols(N, batch);
    lrp_arena ar(ws, ws_bytes);
    double2* W = ar.take<double2>((size_t)g * L);
    double* sums = ar.take<double>((size_t)g * (L / SC_CHUNK + 1));
    if (!ar.ok()) return LRP_ERR_WORKSPACE;
    const int nchunks = (int)(L / SC_CHUNK);
    for (int c0 = 0; c0 < batch; c0 += g) {
        const int cols = (batch - c0) < g ? (batch - c0) : g;
        double* o = d_out + (int64_t)c0 * ld_out;
        LRP_TRY(dispatch_pa(q1, tl, ctx, log2N, cols, d_in + (int64_t)c0 * ld_in, ld_in, W));
        LRP_TRY(dispatch_pb(q2, tl, ctx, log2N, cols, W, o, ld_out, scale, sums + nchunks, nchunks + 1));
        LRP_PROF(ctx, K_DST_CHUNKSUM, 8.0 * N * cols, 0);
        dst1_chunksum_kernel<<<dim3(nchunks, cols), SC_NT, 0, ctx->stream>>>(log2N, o, ld_out, sums);
        LRP_LAUNCHED(ctx);
        LRP_PROF(ctx, K_DST_SCANSUMS, 0, 0);
        dst1_scansums_kernel<<<cols, 1024, 0, ctx->stream>>>(nchunks, sums);
        LRP_LAUNCHED(ctx);
        LRP_PROF(ctx, K_DST_FINISH, 16.0 * N * cols, 0);
        dst1_scanapply_kernel<<<dim3(nchunks, cols), SC_NT, 0, ctx->stream>>>(log2N, o, ld_out, sums);
        LRP_LAUNCHED(ctx);
    }
    return LRP_OK;
}
