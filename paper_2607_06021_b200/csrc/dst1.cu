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
#include <math.h>

namespace {

__host__ __device__ constexpr int PADI(int i) { return i + (i >> 5); }

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// two-level table of exp(-2 pi i u / M):  hi[u >> 6] * lo[u & 63]
__device__ __forceinline__ double2 tw_get(const double2* lo, const double2* hi, int u) {
    return cmul(hi[u >> 6], lo[u & 63]);
}
__device__ __forceinline__ void tw_build(double2* lo, double2* hi, int M, int nhi, int tid, int nt) {
    const double inv = 1.0 / (double)M;     // M is a power of two: every argument below is exact
    for (int i = tid; i < 64; i += nt) {
        double s, c; sincospi(-2.0 * (double)i * inv, &s, &c); lo[i] = make_double2(c, s);
    }
    for (int i = tid; i < nhi; i += nt) {
        double s, c; sincospi(-2.0 * (double)(i * 64) * inv, &s, &c); hi[i] = make_double2(c, s);
    }
}

template <int R> struct Bfly;
template <> struct Bfly<2> {
    __device__ __forceinline__ static void run(double2 (&v)[2]) {
        double2 a = v[0], b = v[1];
        v[0] = make_double2(a.x + b.x, a.y + b.y);
        v[1] = make_double2(a.x - b.x, a.y - b.y);
    }
};
__device__ __forceinline__ void fft4(double2& v0, double2& v1, double2& v2, double2& v3) {
    double2 t0 = make_double2(v0.x + v2.x, v0.y + v2.y);
    double2 t1 = make_double2(v0.x - v2.x, v0.y - v2.y);
    double2 t2 = make_double2(v1.x + v3.x, v1.y + v3.y);
    double2 d  = make_double2(v1.x - v3.x, v1.y - v3.y);
    double2 t3 = make_double2(d.y, -d.x);                       // (v1 - v3) * (-i)
    v0 = make_double2(t0.x + t2.x, t0.y + t2.y);
    v2 = make_double2(t0.x - t2.x, t0.y - t2.y);
    v1 = make_double2(t1.x + t3.x, t1.y + t3.y);
    v3 = make_double2(t1.x - t3.x, t1.y - t3.y);
}
template <> struct Bfly<4> {
    __device__ __forceinline__ static void run(double2 (&v)[4]) { fft4(v[0], v[1], v[2], v[3]); }
};
template <> struct Bfly<8> {
    __device__ __forceinline__ static void run(double2 (&v)[8]) {
        const double c = 0.70710678118654752440;
        double2 a0 = make_double2(v[0].x + v[4].x, v[0].y + v[4].y);
        double2 a1 = make_double2(v[1].x + v[5].x, v[1].y + v[5].y);
        double2 a2 = make_double2(v[2].x + v[6].x, v[2].y + v[6].y);
        double2 a3 = make_double2(v[3].x + v[7].x, v[3].y + v[7].y);
        double2 b0 = make_double2(v[0].x - v[4].x, v[0].y - v[4].y);
        double2 d1 = make_double2(v[1].x - v[5].x, v[1].y - v[5].y);
        double2 d2 = make_double2(v[2].x - v[6].x, v[2].y - v[6].y);
        double2 d3 = make_double2(v[3].x - v[7].x, v[3].y - v[7].y);
        double2 b1 = make_double2(c * (d1.x + d1.y), c * (d1.y - d1.x));     // * exp(-i pi/4)
        double2 b2 = make_double2(d2.y, -d2.x);                                // * (-i)
        double2 b3 = make_double2(c * (d3.y - d3.x), -c * (d3.x + d3.y));     // * exp(-3 i pi/4)
        fft4(a0, a1, a2, a3);
        fft4(b0, b1, b2, b3);
        v[0] = a0; v[2] = a1; v[4] = a2; v[6] = a3;
        v[1] = b0; v[3] = b1; v[5] = b2; v[7] = b3;
    }
};

// One Stockham pass of radix R over a length-2^Q complex sequence held in (re, im) (padded with PADI),
// executed by the GS = 2^Q/8 threads of a group (gt = thread in group); every thread keeps its 8 complex
// values in registers across the barrier, so the pass is in place.  Twiddle exp(-2 pi i mm / L) = tw(tw_mul*mm).
template <int Q, int R, bool FIRST>
__device__ __forceinline__ void fft_pass(double* re, double* im, int gt, int log2Ns,
                                         const double2* lo, const double2* hi, int tw_mul) {
    constexpr int L = 1 << Q, GS = L / 8, ITEMS = 8 / R, STRIDE = L / R;
    double2 v[ITEMS][R];
#pragma unroll
    for (int it = 0; it < ITEMS; ++it)
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int idx = PADI(gt + it * GS + r * STRIDE);
            v[it][r] = make_double2(re[idx], im[idx]);
        }
    __syncthreads();
    const int Ns = 1 << log2Ns;
#pragma unroll
    for (int it = 0; it < ITEMS; ++it) {
        int j = gt + it * GS;
        int k = j & (Ns - 1);
        if (!FIRST) {
            int mm = k * (STRIDE >> log2Ns);
            double2 w1 = tw_get(lo, hi, tw_mul * mm);
            if constexpr (R == 2) {
                v[it][1] = cmul(v[it][1], w1);
            } else if constexpr (R == 4) {
                double2 w2 = cmul(w1, w1), w3 = cmul(w2, w1);
                v[it][1] = cmul(v[it][1], w1); v[it][2] = cmul(v[it][2], w2); v[it][3] = cmul(v[it][3], w3);
            } else {
                double2 w2 = cmul(w1, w1), w3 = cmul(w2, w1), w4 = cmul(w2, w2);
                double2 w5 = cmul(w4, w1), w6 = cmul(w4, w2), w7 = cmul(w4, w3);
                v[it][1] = cmul(v[it][1], w1); v[it][2] = cmul(v[it][2], w2); v[it][3] = cmul(v[it][3], w3);
                v[it][4] = cmul(v[it][4], w4); v[it][5] = cmul(v[it][5], w5);
                v[it][6] = cmul(v[it][6], w6); v[it][7] = cmul(v[it][7], w7);
            }
        }
        Bfly<R>::run(v[it]);
        int base = (j - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int idx = PADI(base + (r << log2Ns));
            re[idx] = v[it][r].x; im[idx] = v[it][r].y;
        }
    }
    __syncthreads();
}

// forward complex FFT of length 2^Q in shared memory, natural order in and out (Stockham autosort).
template <int Q>
__device__ __forceinline__ void fft_smem(double* re, double* im, int gt,
                                         const double2* lo, const double2* hi, int tw_mul) {
    constexpr int A = Q / 3, B = Q % 3;
    fft_pass<Q, 8, true>(re, im, gt, 0, lo, hi, tw_mul);
#pragma unroll
    for (int p = 1; p < A; ++p) fft_pass<Q, 8, false>(re, im, gt, 3 * p, lo, hi, tw_mul);
    if (B == 1) fft_pass<Q, 2, false>(re, im, gt, 3 * A, lo, hi, tw_mul);
    if (B == 2) fft_pass<Q, 4, false>(re, im, gt, 3 * A, lo, hi, tw_mul);
}

// inclusive scan of one value per thread over the GS (power of two) threads of a group; wsum: >= 32 doubles
// of shared memory per group (used when GS > 32).  Contains barriers: call from all threads.
template <int GS>
__device__ __forceinline__ double group_scan_incl(double v, int gt, double* wsum) {
    constexpr int W = GS < 32 ? GS : 32;
#pragma unroll
    for (int d = 1; d < W; d <<= 1) {
        double o = __shfl_up_sync(0xffffffffu, v, d, W);
        if ((gt & (W - 1)) >= d) v += o;
    }
    if (GS > 32) {
        constexpr int NW = GS / 32;
        if ((gt & 31) == 31) wsum[gt >> 5] = v;
        __syncthreads();
        if (gt < 32) {
            double s = gt < NW ? wsum[gt] : 0.0;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                double o = __shfl_up_sync(0xffffffffu, s, d, 32);
                if (gt >= d) s += o;
            }
            if (gt < NW) wsum[gt] = s;
        }
        __syncthreads();
        if (gt >= 32) v += wsum[(gt >> 5) - 1];
        __syncthreads();
    }
    return v;
}

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
    static constexpr int PL = PADI(L) + 1;
    static constexpr int NHI = N / 64 + 1;
    static constexpr size_t SMEM = sizeof(double2) * (64 + NHI) + sizeof(double) * ((size_t)CPB * 2 * PL + 32 * CPB);
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
    double* wsum = data + (size_t)C::CPB * 2 * PL + 32 * g;
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

    fft_smem<Q>(re, im, gt, lo, hi, 4);                              // exp(-2 pi i mm/L) = tw(4 mm)

    // untangle: pairs (k, L-k), k = 0 .. L/2
    for (int k = gt; k <= L / 2; k += GS) {
        if (k == 0) {
            double a = re[0], b = im[0];
            re[0] = 0.5 * (a + b);                                   // X_1 = T_0 / 2
            im[0] = 0.0;
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

    // X_{2k+1} = X_1 + sum_{m<=k} R_m : inclusive scan over re[0..L)
    {
        double loc[8];
        double run = 0.0;
#pragma unroll
        for (int i = 0; i < 8; ++i) { run += re[PADI(gt * 8 + i)]; loc[i] = run; }
        double incl = group_scan_incl<GS>(run, gt, wsum);
        double off = incl - run;
#pragma unroll
        for (int i = 0; i < 8; ++i) re[PADI(gt * 8 + i)] = loc[i] + off;
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

// ------------------------------------------------------------------------------------------ four-step regime
// L = L1 * L2, j = j1*L2 + j2, k = k1 + L1*k2:
//   Z[k1 + L1 k2] = sum_{j2} w_{L2}^{j2 k2} [ w_L^{j2 k1} sum_{j1} z[j1 L2 + j2] w_{L1}^{j1 k1} ].
template <int Q1> struct P1Cfg {
    static constexpr int L1 = 1 << Q1, GS = L1 / 8;
    static constexpr int T = L1 >= 4096 ? 1 : 4096 / L1;             // j2 values per CTA
    static constexpr int NT = T * GS;
    static constexpr int WANT = (16 / T) > 0 ? (16 / T) : 1;
    static constexpr int RS = PADI(L1) + (((WANT - PADI(L1)) % 16) + 16) % 16;   // row stride: RS = WANT mod 16
    static constexpr int NHI = (2 * L1) / 64 + 1;
    static constexpr int TW_LO = 32, TW_HI = L1 / 32;
    static constexpr size_t SMEM = sizeof(double2) * (64 + NHI + 2 * T + (size_t)T * (TW_LO + TW_HI)) +
                                   sizeof(double) * ((size_t)T * 2 * RS);
};

// sweep 1: fold x into z on the fly, length-L1 FFTs over the strided index j1, four-step twiddle, write W[k1*L2 + j2].
template <int Q1>
__global__ void __launch_bounds__(P1Cfg<Q1>::NT)
dst1_p1_kernel(int log2N, const double* __restrict__ in, int64_t ld_in, double2* __restrict__ W) {
    using C = P1Cfg<Q1>;
    constexpr int L1 = C::L1, GS = C::GS, T = C::T, RS = C::RS, NT = C::NT;
    const int64_t N = (int64_t)1 << log2N;
    const int64_t L = N >> 1;
    const int L2 = (int)(L >> Q1);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* lo = (double2*)smem_raw;
    double2* hi = lo + 64;
    double2* tB = hi + C::NHI;                                        // exp(-i pi (2 j2 + b)/N), 2T entries
    double2* t4lo = tB + 2 * T;                                       // [T][32]  exp(-2 pi i j2 l / L)
    double2* t4hi = t4lo + T * C::TW_LO;                              // [T][L1/32] exp(-2 pi i j2 (32 h)/L)
    double* data = (double*)(t4hi + T * C::TW_HI);
    const int tid = threadIdx.x;
    const int j2_0 = blockIdx.x * T;
    const double* x = in + (int64_t)blockIdx.y * ld_in;
    double2* Wc = W + (int64_t)blockIdx.y * L;

    // loads: element e -> (j1 = e / T, j2l = e % T), 8 per thread
    double x0[8], x1[8], y0[8], y1[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int j2l = e % T, j1 = e / T;
        int64_t m0 = 2 * ((int64_t)j1 * L2 + j2_0 + j2l);            // even index, m1 = m0 + 1
        x0[i] = (m0 >= 1) ? x[m0 - 1] : 0.0;
        x1[i] = x[m0];                                                // m1 <= N-1 always
        y0[i] = (m0 >= 1) ? x[N - m0 - 1] : 0.0;                      // x_{N-m0}
        y1[i] = x[N - m0 - 2];                                        // x_{N-m1}, N - m1 >= 1 always
    }
    tw_build(lo, hi, 2 * L1, C::NHI, tid, NT);
    for (int i = tid; i < 2 * T; i += NT) {
        double s, c; sincospi(-(double)(2 * j2_0 + i) / (double)N, &s, &c); tB[i] = make_double2(c, s);
    }
    for (int i = tid; i < T * (C::TW_LO + C::TW_HI); i += NT) {
        int j2l, kk; double2* dst;
        if (i < T * C::TW_LO) { j2l = i / C::TW_LO; kk = i % C::TW_LO; dst = t4lo + i; }
        else { int q = i - T * C::TW_LO; j2l = q / C::TW_HI; kk = (q % C::TW_HI) * 32; dst = t4hi + q; }
        int64_t prod = ((int64_t)(j2_0 + j2l) * kk) & (L - 1);
        double s, c; sincospi(-2.0 * (double)prod / (double)L, &s, &c); *dst = make_double2(c, s);
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int j2l = e % T, j1 = e / T;
        double2 a = tw_get(lo, hi, j1);                               // exp(-i pi j1 / L1)
        double2 b0 = tB[2 * j2l], b1 = tB[2 * j2l + 1];
        double s0 = -(a.x * b0.y + a.y * b0.x);                       // sin(pi m0 / N)
        double s1 = -(a.x * b1.y + a.y * b1.x);
        double t0 = s0 * (x0[i] + y0[i]) + 0.5 * (x0[i] - y0[i]);
        double t1 = s1 * (x1[i] + y1[i]) + 0.5 * (x1[i] - y1[i]);
        data[(size_t)j2l * 2 * RS + PADI(j1)] = t0;
        data[(size_t)j2l * 2 * RS + RS + PADI(j1)] = t1;
    }
    __syncthreads();
    {
        const int g = tid / GS, gt = tid % GS;
        fft_smem<Q1>(data + (size_t)g * 2 * RS, data + (size_t)g * 2 * RS + RS, gt, lo, hi, 2);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int j2l = e % T, k1 = e / T;
        double2 v = make_double2(data[(size_t)j2l * 2 * RS + PADI(k1)], data[(size_t)j2l * 2 * RS + RS + PADI(k1)]);
        double2 w = cmul(t4hi[j2l * C::TW_HI + (k1 >> 5)], t4lo[j2l * C::TW_LO + (k1 & 31)]);
        Wc[(int64_t)k1 * L2 + j2_0 + j2l] = cmul(v, w);
    }
}

template <int Q2> struct P2Cfg {
    static constexpr int L2 = 1 << Q2, GS = L2 / 8;
    static constexpr int T = L2 >= 4096 ? 1 : 4096 / L2;             // k1 rows per CTA
    static constexpr int NT = T * GS;
    static constexpr int WANT = (16 / T) > 0 ? (16 / T) : 1;
    static constexpr int RS = PADI(L2) + (((WANT - PADI(L2)) % 16) + 16) % 16;
    static constexpr int NHI = L2 / 64 + 1;
    static constexpr size_t SMEM = sizeof(double2) * (64 + NHI) + sizeof(double) * ((size_t)T * 2 * RS);
};

// sweep 2: contiguous length-L2 FFTs over j2 for T adjacent k1, write Z[k1 + L1 k2].
template <int Q2>
__global__ void __launch_bounds__(P2Cfg<Q2>::NT)
dst1_p2_kernel(int log2N, const double2* __restrict__ W, double2* __restrict__ Z) {
    using C = P2Cfg<Q2>;
    constexpr int L2 = C::L2, GS = C::GS, T = C::T, RS = C::RS, NT = C::NT;
    const int64_t L = (int64_t)1 << (log2N - 1);
    const int L1 = (int)(L >> Q2);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* lo = (double2*)smem_raw;
    double2* hi = lo + 64;
    double* data = (double*)(hi + C::NHI);
    const int tid = threadIdx.x;
    const int k1_0 = blockIdx.x * T;
    const double2* Wc = W + (int64_t)blockIdx.y * L;
    double2* Zc = Z + (int64_t)blockIdx.y * L;
    double2 v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;                                          // row r = e / L2, j2 = e % L2
        v[i] = Wc[(int64_t)(k1_0 + e / L2) * L2 + (e % L2)];
    }
    tw_build(lo, hi, L2, C::NHI, tid, NT);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int r = e / L2, j2 = e % L2;
        data[(size_t)r * 2 * RS + PADI(j2)] = v[i].x;
        data[(size_t)r * 2 * RS + RS + PADI(j2)] = v[i].y;
    }
    __syncthreads();
    {
        const int g = tid / GS, gt = tid % GS;
        fft_smem<Q2>(data + (size_t)g * 2 * RS, data + (size_t)g * 2 * RS + RS, gt, lo, hi, 1);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int r = e % T, k2 = e / T;
        double2 o = make_double2(data[(size_t)r * 2 * RS + PADI(k2)], data[(size_t)r * 2 * RS + RS + PADI(k2)]);
        Zc[(int64_t)k2 * L1 + k1_0 + r] = o;
    }
}

// sweep 3a: real-FFT untangle of Z into R (prefix-sum terms) and E (even outputs), both length L per column.
__global__ void dst1_untangle_kernel(int log2N, const double2* __restrict__ Z, double* __restrict__ RE, double scale) {
    const int64_t N = (int64_t)1 << log2N, L = N >> 1;
    const double2* Zc = Z + (int64_t)blockIdx.y * L;
    double* R = RE + (int64_t)blockIdx.y * N;
    double* E = R + L;
    const double invN = 1.0 / (double)N;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k <= L / 2; k += (int64_t)gridDim.x * blockDim.x) {
        if (k == 0) {
            double2 z = Zc[0];
            R[0] = scale * 0.5 * (z.x + z.y);
            E[0] = 0.0;
        } else {
            int64_t km = L - k;
            double2 zk = Zc[k], zm = Zc[km];
            double2 Ev = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y));
            double2 Ov = make_double2(0.5 * (zk.y + zm.y), -0.5 * (zk.x - zm.x));
            double s, c; sincospi(-2.0 * (double)k * invN, &s, &c);
            double2 wO = cmul(make_double2(c, s), Ov);
            R[k] = scale * (Ev.x + wO.x);   E[k] = -scale * (Ev.y + wO.y);
            R[km] = scale * (Ev.x - wO.x);  E[km] = scale * (Ev.y - wO.y);
        }
    }
}

constexpr int SCAN_CHUNK = 4096, SCAN_NT = 512;

// sweep 3b: per-chunk sums of R
__global__ void __launch_bounds__(SCAN_NT)
dst1_chunksum_kernel(int log2N, const double* __restrict__ RE, double* __restrict__ sums) {
    const int64_t N = (int64_t)1 << log2N, L = N >> 1;
    const double* R = RE + (int64_t)blockIdx.y * N + (int64_t)blockIdx.x * SCAN_CHUNK;
    __shared__ double ws[32];
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < SCAN_CHUNK / SCAN_NT; ++i) acc += R[threadIdx.x + i * SCAN_NT];
    for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < SCAN_NT / 32; ++w) t += ws[w];
        sums[(int64_t)blockIdx.y * (L / SCAN_CHUNK) + blockIdx.x] = t;
    }
    (void)L;
}
// sweep 3c: exclusive scan of the chunk sums of one column (one CTA per column)
__global__ void __launch_bounds__(1024)
dst1_scansums_kernel(int nchunks, double* __restrict__ sums) {
    double* s = sums + (int64_t)blockIdx.x * nchunks;
    __shared__ double wsum[32];
    double carry = 0.0;
    for (int base = 0; base < nchunks; base += 1024) {
        int i = base + threadIdx.x;
        double v = i < nchunks ? s[i] : 0.0;
        double incl = group_scan_incl<1024>(v, threadIdx.x, wsum);
        if (i < nchunks) s[i] = carry + incl - v;
        __shared__ double tot;
        if (threadIdx.x == 1023) tot = incl;
        __syncthreads();
        carry += tot;
        __syncthreads();
    }
}
// sweep 3d: scan each chunk of R with its offset and interleave with E into the natural-order output.
__global__ void __launch_bounds__(SCAN_NT)
dst1_finish_kernel(int log2N, const double* __restrict__ RE, const double* __restrict__ sums,
                   double* __restrict__ out, int64_t ld_out) {
    const int64_t N = (int64_t)1 << log2N, L = N >> 1;
    const int64_t k0 = (int64_t)blockIdx.x * SCAN_CHUNK;
    const double* R = RE + (int64_t)blockIdx.y * N;
    const double* E = R + L;
    double* o = out + (int64_t)blockIdx.y * ld_out;
    __shared__ double sm[SCAN_CHUNK + SCAN_CHUNK / 32 + 8];
    __shared__ double wsum[32];
    for (int i = threadIdx.x; i < SCAN_CHUNK; i += SCAN_NT) sm[PADI(i)] = R[k0 + i];
    __syncthreads();
    constexpr int PER = SCAN_CHUNK / SCAN_NT;
    double loc[PER]; double run = 0.0;
#pragma unroll
    for (int i = 0; i < PER; ++i) { run += sm[PADI(threadIdx.x * PER + i)]; loc[i] = run; }
    double incl = group_scan_incl<SCAN_NT>(run, threadIdx.x, wsum);
    double off = incl - run + sums[(int64_t)blockIdx.y * (L / SCAN_CHUNK) + blockIdx.x];
#pragma unroll
    for (int i = 0; i < PER; ++i) sm[PADI(threadIdx.x * PER + i)] = loc[i] + off;
    __syncthreads();
    // outputs X_m, m = 2 k0 .. 2 k0 + 2*CHUNK - 1, at o[m-1]
    for (int i = threadIdx.x; i < 2 * SCAN_CHUNK; i += SCAN_NT) {
        int64_t m = 2 * k0 + i;
        if (m >= 1) {
            double val = (i & 1) ? sm[PADI(i >> 1)] : E[k0 + (i >> 1)];
            o[m - 1] = val;
        }
    }
}

template <int Q>
int launch_small(lrp_ctx* ctx, int batch, const double* in, int64_t ld_in, double* out, int64_t ld_out, double scale) {
    using C = SmallCfg<Q>;
    LRP_CUDA(ctx, cudaFuncSetAttribute(dst1_small_kernel<Q>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    int grid = (batch + C::CPB - 1) / C::CPB;
    LRP_PROF(ctx, K_DST_SMALL, 16.0 * (2 * C::L - 1) * batch, 0);
    dst1_small_kernel<Q><<<grid, C::NT, C::SMEM, ctx->stream>>>(batch, in, ld_in, out, ld_out, scale);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}
template <int Q1>
int launch_p1(lrp_ctx* ctx, int log2N, int cols, const double* in, int64_t ld_in, double2* W) {
    using C = P1Cfg<Q1>;
    LRP_CUDA(ctx, cudaFuncSetAttribute(dst1_p1_kernel<Q1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    int L2 = 1 << (log2N - 1 - Q1);
    dim3 grid(L2 / C::T, cols);
    LRP_PROF(ctx, K_DST_P1, 16.0 * ((int64_t)1 << log2N) * cols, 0);
    dst1_p1_kernel<Q1><<<grid, C::NT, C::SMEM, ctx->stream>>>(log2N, in, ld_in, W);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}
template <int Q2>
int launch_p2(lrp_ctx* ctx, int log2N, int cols, const double2* W, double2* Z) {
    using C = P2Cfg<Q2>;
    LRP_CUDA(ctx, cudaFuncSetAttribute(dst1_p2_kernel<Q2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    int L1 = 1 << (log2N - 1 - Q2);
    dim3 grid(L1 / C::T, cols);
    LRP_PROF(ctx, K_DST_P2, 16.0 * ((int64_t)1 << log2N) * cols, 0);
    dst1_p2_kernel<Q2><<<grid, C::NT, C::SMEM, ctx->stream>>>(log2N, W, Z);
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
int dispatch_p1(int q1, lrp_ctx* ctx, int log2N, int cols, const double* in, int64_t ld_in, double2* W) {
    LRP_Q_SWITCH(q1, launch_p1, ctx, log2N, cols, in, ld_in, W)
}
int dispatch_p2(int q2, lrp_ctx* ctx, int log2N, int cols, const double2* W, double2* Z) {
    LRP_Q_SWITCH(q2, launch_p2, ctx, log2N, cols, W, Z)
}

// columns per group in the four-step regime: keep one group's intermediates around L2 size
int group_cols(int64_t N, int batch) {
    int64_t per_col = N * 8 * 3;                                      // W/RE + Z + output column
    int g = (int)((int64_t)(96 << 20) / per_col);
    if (g < 1) g = 1;
    if (g > batch) g = batch;
    return g;
}

}  // namespace

size_t lrp_dst1_ws_impl(int64_t n, int32_t batch) {
    int64_t N = n + 1;
    if (N <= 16384 || batch <= 0) return 0;
    int g = group_cols(N, batch);
    int64_t L = N / 2;
    size_t bytes = 0;
    bytes += lrp_align_up((size_t)g * L * sizeof(double2));           // W, reused as R | E
    bytes += lrp_align_up((size_t)g * L * sizeof(double2));           // Z
    bytes += lrp_align_up((size_t)g * (L / SCAN_CHUNK) * sizeof(double));
    return bytes;
}

int lrp_dst1_impl(lrp_ctx* ctx, int64_t n, int32_t batch, const double* d_in, int64_t ld_in,
                  double* d_out, int64_t ld_out, double scale, void* ws, size_t ws_bytes) {
    if (batch == 0) return LRP_OK;
    const int64_t N = n + 1;
    if (N < 64) {
        LRP_PROF(ctx, K_DST_NAIVE, 16.0 * n * batch, 0);
        dst1_naive_kernel<<<batch, 32, 0, ctx->stream>>>((int)n, d_in, ld_in, d_out, ld_out, scale);
        LRP_LAUNCHED(ctx);
        return LRP_OK;
    }
    const int log2N = lrp_ilog2(N);
    if (N <= 16384) return dispatch_small(log2N - 1, ctx, batch, d_in, ld_in, d_out, ld_out, scale);

    if (ws_bytes < lrp_dst1_ws_impl(n, batch)) return LRP_ERR_WORKSPACE;
    const int q = log2N - 1, q1 = q / 2, q2 = q - q1;
    const int64_t L = N / 2;
    const int g = group_cols(N, batch);
    lrp_arena ar(ws, ws_bytes);
    double2* W = ar.take<double2>((size_t)g * L);
    double2* Z = ar.take<double2>((size_t)g * L);
    double* sums = ar.take<double>((size_t)g * (L / SCAN_CHUNK));
    if (!ar.ok()) return LRP_ERR_WORKSPACE;
    const int nchunks = (int)(L / SCAN_CHUNK);
    for (int c0 = 0; c0 < batch; c0 += g) {
        const int cols = (batch - c0) < g ? (batch - c0) : g;
        LRP_TRY(dispatch_p1(q1, ctx, log2N, cols, d_in + (int64_t)c0 * ld_in, ld_in, W));
        LRP_TRY(dispatch_p2(q2, ctx, log2N, cols, W, Z));
        {
            int64_t work = L / 2 + 1;
            int bx = (int)((work + 255) / 256); if (bx > 4096) bx = 4096;
            LRP_PROF(ctx, K_DST_UNTANGLE, 16.0 * N * cols, 0);
            dst1_untangle_kernel<<<dim3(bx, cols), 256, 0, ctx->stream>>>(log2N, Z, (double*)W, scale);
            LRP_LAUNCHED(ctx);
        }
        LRP_PROF(ctx, K_DST_CHUNKSUM, 4.0 * N * cols, 0);
        dst1_chunksum_kernel<<<dim3(nchunks, cols), SCAN_NT, 0, ctx->stream>>>(log2N, (const double*)W, sums);
        LRP_LAUNCHED(ctx);
        LRP_PROF(ctx, K_DST_SCANSUMS, 0, 0);
        dst1_scansums_kernel<<<cols, 1024, 0, ctx->stream>>>(nchunks, sums);
        LRP_LAUNCHED(ctx);
        LRP_PROF(ctx, K_DST_FINISH, 16.0 * N * cols, 0);
        dst1_finish_kernel<<<dim3(nchunks, cols), SCAN_NT, 0, ctx->stream>>>(log2N, (const double*)W, sums,
                                                                            d_out + (int64_t)c0 * ld_out, ld_out);
        LRP_LAUNCHED(ctx);
    }
    return LRP_OK;
}
