// dst1_large.cu -- batched DST-I for N = n + 1 = 2^p > 16384: the column no longer fits one CTA's shared memory.
//
// Same folding as dst1.cu (t -> z, complex FFT of length L = N/2, untangle, odd outputs from R_k = X_{2k+1} - X_{2k-1}),
// with the FFT split four-step style, L = L1 * L2, j = j1*L2 + j2, k = k1 + L1*k2.  ONE persistent kernel runs the
// whole batch: its CTAs pull work items from a queue in global memory, and the complex intermediate W (8N bytes per
// column) lives in a two-slot ring of column groups small enough to stay in the 126 MB L2, so that HBM sees each
// element once on the way in and once on the way out (the r01 version made three full HBM sweeps).  Items, per column:
//   A (nA tiles): fold x on the fly (the CTA owns a j2 tile AND its mirror tile: every x element is fetched once),
//       length-L1 FFTs over the strided index j1, four-step twiddle, W[k1*L2 + j2]; the same pass accumulates the
//       folded sums y_r = sum_{m = r mod Mc, m < L} (x_m + x_{N-m}) e^{i pi m/N} that the anchors need;
//   D (1 item): exact anchors  X_{2 c CH + 1} = x_L + Im sum_r y_r e^{2 pi i r c / Mc},  Mc = N/CH, CH = 4096: the odd
//       outputs at the start of every chunk of 4096 k, by one shared-memory FFT of the Mc folded sums;
//   B (nB tiles): rows k1 and their mirror rows L1 - k1: length-L2 FFTs, real-FFT untangle of the pairs (k, L-k) in
//       shared memory; (R_k, X_{2k}) go back IN PLACE into the rows of W;
//   C (nC = L/4096 chunks): gathers its (R, X_even) from the [k1][k2] layout of W, transposes through shared memory,
//       sums R forward from the chunk's own anchor over the first half and backward from the next chunk's anchor over
//       the second half (every odd output is reached through a chain of <= 2048 terms from an independently computed
//       value: the rounding error no longer grows with N as in a global prefix sum), writes the natural-order output.
// Dependencies (A -> D, A -> B, B + D -> C, C of the group two back -> A: ring slot free) are per-column arrival counters;
// items are queued in an order in which every dependency points backwards, and a CTA that holds an item is running, so
// the waits cannot deadlock whatever the number of resident CTAs.
// Measured alternatives (scratch microbenchmarks, figures in DESIGN.md section 4): distributed shared memory in a 16-CTA cluster exchanges
// 3.2 TB/s over the 112 SMs such clusters can occupy, L2-resident traffic 12 TB/s over all 148 -- hence L2, not DSMEM,
// also for the sizes (N <= 2^18) whose column would fit a cluster.
#include "common.cuh"
#include "fft_smem.cuh"
#include <math.h>
#include <cuda/atomic>

#ifdef LRP_DST_STATS
__device__ unsigned long long g_sub[32];
#define SUBT(i) do { if (threadIdx.x == 0) { long long t_ = clock64(); atomicAdd(&g_sub[i], (unsigned long long)(t_ - tsub)); tsub = t_; } } while (0)
#define SUBT0() long long tsub = clock64()
extern "C" int lrp_debug_dst_sub(unsigned long long* out) { cudaDeviceSynchronize(); int rc = (int)cudaMemcpyFromSymbol(out, g_sub, sizeof(g_sub)); unsigned long long z[32] = {0}; cudaMemcpyToSymbol(g_sub, z, sizeof(z)); return rc; }
#else
#define SUBT(i) do {} while (0)
#define SUBT0() do {} while (0)
#endif
namespace {

constexpr int SC_CHUNK = 4096;                                  // k's per chunk of phase C = anchor spacing
constexpr int64_t RING_SLOT_BYTES = 24ll << 20;                 // W bytes per ring slot (two slots live in L2)

constexpr int row_stride(int Lrow, int nrows) {            // padded row length with (stride mod 16) == max(1, 16/nrows)
    int want = (16 / nrows) > 0 ? (16 / nrows) : 1;
    int base = Lrow;
    return base + (((want - base) % 16) + 16) % 16;
}

__device__ __forceinline__ double2 ldcg2(const double2* p) { return __ldcg(p); }

// ------------------------------------------------------------------------------------------------ phase A
template <int Q1, int TL> struct PACfg {
    static constexpr int L1 = 1 << Q1, GS = L1 / 8;
    static constexpr int T2 = (1 << TL) / L1, T = T2 / 2;        // sub-FFTs per CTA: T of the tile + T of its mirror
    static constexpr int NT = (1 << TL) / 8;
    static constexpr int RS = row_stride(L1, T2);
    static constexpr int IMOFF = T2 * RS + 8;
    static constexpr int NHI = (2 * L1) / 64 + 1;
    static constexpr int TW_LO = 32, TW_HI = (L1 + 31) / 32;
    static constexpr int SLO = 33, SHI = TW_HI | 1;        // odd row strides: the T2 rows are read side by side
    static constexpr int CH = 4;                  // loads in flight per thread (register budget)
    static constexpr size_t SMEM = sizeof(double2) * (64 + NHI + 2 * T2 + (size_t)T2 * (SLO + SHI)) +
                                   sizeof(double) * ((size_t)2 * IMOFF);
    static_assert(sizeof(double) * 2 * IMOFF >= sizeof(double) * 4 * NT, "anchor partial reduction reuses the FFT arrays");
};

// Column-independent twiddles of phase A, built once per call (dst1_tables_kernel) and read by every tile from L2:
//   gB   [2 L2]          exp(-i pi m / N), m = 2 j2 + b
//   g4lo [L2][32]        exp(-2 pi i j2 l / L)
//   g4hi [L2][L1/32]     exp(-2 pi i j2 (32 h) / L)
//   twA  [64 + NHI_A]    two-level table (tw_get) of exp(-2 pi i u / (2 L1)): lo[64] then hi[2 L1 / 64 + 1]
//   twB  [64 + NHI_B]    the same for exp(-2 pi i u / (2 L2))   (phase B)
struct ATables { const double2* gB; const double2* g4lo; const double2* g4hi; const double2* twA; const double2* twB; };

// copy a two-level twiddle table (tw_get layout: lo[64], hi[nhi]) from the per-call global table into shared memory
__device__ __forceinline__ void tw_fetch(double2* lo, double2* hi, const double2* __restrict__ src, int nhi, int tid, int nt) {
    for (int i = tid; i < 64 + nhi; i += nt) { const double2 v = __ldg(src + i); if (i < 64) lo[i] = v; else hi[i - 64] = v; }
}

// tile c of one column: x -> W (L complex), ypart[2 j2 + b] (2 L2 complex): the CTA's folded anchor sums
template <int Q1, int TL>
__device__ __forceinline__ void phase_a(unsigned char* smem_raw, int log2N, int c, const double* __restrict__ x,
                                        double2* __restrict__ Wc, double2* __restrict__ ypart, const ATables tabs) {
    using C = PACfg<Q1, TL>;
    constexpr int L1 = C::L1, GS = C::GS, T2 = C::T2, T = C::T, RS = C::RS, NT = C::NT;
    const int64_t N = (int64_t)1 << log2N, L = N >> 1;
    const int L2 = (int)(L >> Q1);
    double2* lo = (double2*)smem_raw;
    double2* hi = lo + 64;
    double2* tB = hi + C::NHI;                       // [T2][2]   exp(-i pi (2 j2 + b)/N)
    double2* t4lo = tB + 2 * T2;                     // [T2][32]  exp(-2 pi i j2 l / L)
    double2* t4hi = t4lo + T2 * C::SLO;            // [T2][L1/32] exp(-2 pi i j2 (32 h) / L)
    double* re = (double*)(t4hi + T2 * C::SHI);
    double* im = re + C::IMOFF;
    const int tid = threadIdx.x;
    auto j2_of = [&](int s) { return s < T ? c * T + s : L2 - c * T - T + (s - T); };

    // the first half of the tile's x elements is requested before anything else: the table loads and the barrier below
    // overlap its latency
    double x0[C::CH], x1[C::CH], y0[C::CH], y1[C::CH];
    auto load_half = [&](int i0) {
#pragma unroll
        for (int i = 0; i < C::CH; ++i) {
            int e = tid + (i0 + i) * NT;
            int s = e % T2, j1 = e / T2;
            int64_t m0 = 2 * ((int64_t)j1 * L2 + j2_of(s));
            x0[i] = (m0 >= 1) ? __ldca(x + m0 - 1) : 0.0;
            x1[i] = __ldca(x + m0);
            y0[i] = (m0 >= 1) ? __ldca(x + N - m0 - 1) : 0.0;
            y1[i] = __ldca(x + N - m0 - 2);
        }
    };
    SUBT0();
    load_half(0);
    tw_fetch(lo, hi, tabs.twA, C::NHI, tid, NT);
    for (int i = tid; i < 2 * T2; i += NT) tB[i] = __ldg(tabs.gB + 2 * j2_of(i >> 1) + (i & 1));
    for (int i = tid; i < T2 * (C::TW_LO + C::TW_HI); i += NT) {
        if (i < T2 * C::TW_LO) { const int s = i / C::TW_LO, kk = i % C::TW_LO; t4lo[s * C::SLO + kk] = __ldg(tabs.g4lo + (int64_t)j2_of(s) * C::TW_LO + kk); }
        else { const int q = i - T2 * C::TW_LO, s = q / C::TW_HI, h = q % C::TW_HI; t4hi[s * C::SHI + h] = __ldg(tabs.g4hi + (int64_t)j2_of(s) * C::TW_HI + h); }
    }
    __syncthreads();
    SUBT(0);
    // fold: t_m = sin(pi m/N)(x_m + x_{N-m}) + (x_m - x_{N-m})/2 for m = 2j, 2j+1;  z_j = t_{2j} + i t_{2j+1}
    // anchors: ya[b] += (x_m + x_{N-m}) e^{+i pi m/N} for m = m0 + b < L  (the thread's s = tid % T2 is the same for all its e)
    // The thread's elements share s = tid % T2 and have j1 = q + (L1/8) i, q = tid / T2: e^{-i pi m/N} for m = m0 + b is
    // e^{-i pi q/L1} e^{-i pi (2 j2 + b)/N} (once per thread) times e^{-i pi i/8} (compile-time constants; i + 4: times -i).
    double2 ya0 = make_double2(0.0, 0.0), ya1 = make_double2(0.0, 0.0);
    static_assert(NT / T2 == L1 / 8 && C::CH == 4, "j1 = q + (L1/8) i");
    const int fs = tid % T2, fq = tid / T2;
    double2 ab0, ab1;
    {
        const double2 aq = tw_get(lo, hi, fq);                    // exp(-i pi q / L1)
        ab0 = cmul(aq, tB[2 * fs]); ab1 = cmul(aq, tB[2 * fs + 1]);
    }
    constexpr double W16C[4] = {1.0, 0.92387953251128675613, 0.70710678118654752440, 0.38268343236508977173};
    constexpr double W16S[4] = {0.0, -0.38268343236508977173, -0.70710678118654752440, -0.92387953251128675613};
#pragma unroll 1
    for (int i0 = 0; i0 < 8; i0 += C::CH) {
        if (i0 > 0) {
            load_half(i0);
            ab0 = make_double2(ab0.y, -ab0.x); ab1 = make_double2(ab1.y, -ab1.x);      // times e^{-i pi/2}
        }
#pragma unroll
        for (int i = 0; i < C::CH; ++i) {
            const int j1 = fq + (i0 + i) * (L1 / 8);
            const double2 wi = make_double2(W16C[i], W16S[i]);
            const double2 e0 = i == 0 ? ab0 : cmul(ab0, wi), e1 = i == 0 ? ab1 : cmul(ab1, wi);     // (cos, -sin)(pi m / N)
            const double s0 = -e0.y, s1 = -e1.y;
            const double sum0 = x0[i] + y0[i], sum1 = x1[i] + y1[i];
            re[fs * RS + PADI(j1)] = s0 * sum0 + 0.5 * (x0[i] - y0[i]);
            im[fs * RS + PADI(j1)] = s1 * sum1 + 0.5 * (x1[i] - y1[i]);
            if (j1 < L1 / 2) {                                    // m0, m0 + 1 < L
                ya0.x = fma(sum0, e0.x, ya0.x); ya0.y = fma(sum0, s0, ya0.y);
                ya1.x = fma(sum1, e1.x, ya1.x); ya1.y = fma(sum1, s1, ya1.y);
            }
        }
    }
    __syncthreads();
    SUBT(1);
    {
        const int g = tid / GS, gt = tid % GS;
        fft_smem<Q1, NT / GS>(re + g * RS, im + g * RS, gt, g, lo, hi, 2);
    }
    __syncthreads();                                  // the sub-FFTs synchronise per group; the store below reads across groups
    SUBT(2);
    {
        // k1 = q + (L1/8) i: for L1 = 256 the low table entry (k1 & 31 = q) and the column j2 are the thread's own
        const double2 wlo = t4lo[fs * C::SLO + (fq & 31)];
        const int j2s = j2_of(fs);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int k1 = fq + i * (L1 / 8);
            const double2 v = make_double2(re[fs * RS + PADI(k1)], im[fs * RS + PADI(k1)]);
            const double2 w = cmul(t4hi[fs * C::SHI + (k1 >> 5)], (L1 / 8) % 32 == 0 ? wlo : t4lo[fs * C::SLO + (k1 & 31)]);
            __stcg(&Wc[(int64_t)k1 * L2 + j2s], cmul(v, w));
        }
    }
    __syncthreads();
    SUBT(3);
    // anchor partials: sum over the NT / T2 threads that share s (fixed order), one entry per (j2, b)
    double* red = re;                                 // [NT][4]
    red[4 * tid + 0] = ya0.x; red[4 * tid + 1] = ya0.y; red[4 * tid + 2] = ya1.x; red[4 * tid + 3] = ya1.y;
    __syncthreads();
    if (tid < 2 * T2) {
        const int s = tid >> 1, b = tid & 1;
        double ar = 0.0, ai = 0.0;
        for (int q = 0; q < NT / T2; ++q) { ar += red[4 * (s + q * T2) + 2 * b]; ai += red[4 * (s + q * T2) + 2 * b + 1]; }
        __stcg(&ypart[2 * j2_of(s) + b], make_double2(ar, ai));
    }
    SUBT(4);
}

// one thread per table entry; exact arguments (powers of two), sincospi
__global__ void dst1_tables_kernel(int log2N, int q1, double2* __restrict__ gB, double2* __restrict__ g4lo, double2* __restrict__ g4hi,
                                   double2* __restrict__ twA, double2* __restrict__ twB) {
    const int64_t N = (int64_t)1 << log2N, L = N >> 1, L2 = L >> q1;
    const int nhi = ((1 << q1) + 31) / 32;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t nB = 2 * L2, nlo = L2 * 32, nh = L2 * nhi;
    double sn, cs;
    if (blockIdx.x == 0) {                            // the two-level tables of the sub-FFTs: M = 2 L1 and M = 2 L2
        for (int t = threadIdx.x; t < 2 * 64 + 2 + (int)((2 << q1) / 64) + (int)(2 * L2 / 64); t += blockDim.x) {
            const int nA = 64 + (int)((2 << q1) / 64) + 1;
            const bool isA = t < nA;
            const int u = isA ? t : t - nA;
            const double inv = 1.0 / (double)(isA ? ((int64_t)2 << q1) : 2 * L2);       // powers of two: exact arguments
            const double arg = u < 64 ? -2.0 * (double)u * inv : -2.0 * (double)((u - 64) * 64) * inv;
            sincospi(arg, &sn, &cs);
            (isA ? twA : twB)[u] = make_double2(cs, sn);
        }
    }
    if (i < nB) { sincospi(-(double)i / (double)N, &sn, &cs); gB[i] = make_double2(cs, sn); }
    else if (i < nB + nlo) {
        const int64_t e = i - nB, j2 = e / 32, kk = e % 32;
        sincospi(-2.0 * (double)((j2 * kk) & (L - 1)) / (double)L, &sn, &cs); g4lo[e] = make_double2(cs, sn);
    } else if (i < nB + nlo + nh) {
        const int64_t e = i - nB - nlo, j2 = e / nhi, kk = (e % nhi) * 32;
        sincospi(-2.0 * (double)((j2 * kk) & (L - 1)) / (double)L, &sn, &cs); g4hi[e] = make_double2(cs, sn);
    }
}

// ------------------------------------------------------------------------------------------------ phase D (anchors)
// anchors[c] = scale * X_{2 c CH + 1} = scale * (x_L + Im sum_{r < Mc} y_r e^{2 pi i r c / Mc}),  c < nch = Mc / 2
template <int NT, int QM>
__device__ __forceinline__ void phase_d(unsigned char* smem_raw, int log2N, int log2L1, const double* __restrict__ x,
                                        const double2* __restrict__ ypart, double scale, double* __restrict__ anchors) {
    constexpr int Mc = 1 << QM, nch = Mc / 2;
    const int64_t L = (int64_t)1 << (log2N - 1);
    const int nfold = SC_CHUNK >> log2L1;             // entries of ypart per residue: 2 L2 / Mc = CH / L1
    const int tid = threadIdx.x;
    const double xL = x[L - 1];
    if constexpr (QM <= 7) {                          // Mc <= 128: direct DFT with a full table
        double2* y = (double2*)smem_raw;              // [Mc]
        double2* tab = y + Mc;                        // [Mc] e^{2 pi i u / Mc}
        for (int r = tid; r < Mc; r += NT) {
            double ar = 0.0, ai = 0.0;
            for (int q = 0; q < nfold; ++q) { double2 v = ldcg2(ypart + r + (int64_t)q * Mc); ar += v.x; ai += v.y; }
            y[r] = make_double2(ar, ai);
            double sn, cs; sincospi(2.0 * (double)r / (double)Mc, &sn, &cs); tab[r] = make_double2(cs, sn);
        }
        __syncthreads();
        for (int c = tid; c < nch; c += NT) {
            double a0 = 0.0, a1 = 0.0;
            int u = 0;
            for (int r = 0; r < Mc; r += 2) {
                double2 y0 = y[r], w0 = tab[u]; u = (u + c) & (Mc - 1);
                double2 y1 = y[r + 1], w1 = tab[u]; u = (u + c) & (Mc - 1);
                a0 = fma(y0.x, w0.y, fma(y0.y, w0.x, a0));
                a1 = fma(y1.x, w1.y, fma(y1.y, w1.x, a1));
            }
            anchors[c] = scale * (xL + (a0 + a1));
        }
    } else {                                          // Im IDFT(y) = -Im FFT(conj y): one shared-memory FFT of length Mc
        constexpr int GS = Mc / 8;
        double* re = (double*)smem_raw;               // [Mc + 16]
        double* im = re + Mc + 16;
        double2* lo = (double2*)(im + Mc + 16);       // [64]
        double2* hi = lo + 64;                        // [Mc/64 + 1]
        for (int r = tid; r < Mc; r += NT) {
            double ar = 0.0, ai = 0.0;
            for (int q = 0; q < nfold; ++q) { double2 v = ldcg2(ypart + r + (int64_t)q * Mc); ar += v.x; ai += v.y; }
            re[PADI(r)] = ar; im[PADI(r)] = -ai;
        }
        tw_build(lo, hi, Mc, Mc / 64 + 1, tid, NT);
        __syncthreads();
        // the first GS threads (whole warps, GS >= 32) run the FFT; their passes synchronise on named barrier 1
        if (tid < GS) fft_smem<QM, (GS < NT ? 2 : 1)>(re, im, tid, 0, lo, hi, 1);
        __syncthreads();
        for (int c = tid; c < nch; c += NT) anchors[c] = scale * (xL - im[PADI(c)]);
    }
}

// ------------------------------------------------------------------------------------------------ phase B
// Rows of L2 >= 512 points (SPLIT): decimation in frequency by 8.  The first radix-8 butterfly runs on the registers the
// coalesced row load delivers (v[r] = row[gt + r L2/8]), its outputs are twiddled and stored as EIGHT CONTIGUOUS blocks
// of Ls = L2/8 points (block r' at r' * BS), and block r' is then an independent length-Ls FFT whose result is
// X[8 k' + r'] -- one warp (or less) per block, so the remaining passes synchronise with __syncwarp instead of a
// 256-thread named barrier per pass.  POS(k2) is where X[k2] ends up; BS = Ls + 2 keeps the untangle's and the store
// loop's consecutive k2 (8 blocks x 2 neighbouring k') on 16 different banks.
template <int Q2, int TL> struct PBCfg {
    static constexpr int L2 = 1 << Q2, GS = L2 / 8;
    static constexpr int R2 = (1 << TL) / L2, T = R2 / 2;        // rows per CTA: T rows k1 + their T mirror rows
    static constexpr int NT = (1 << TL) / 8;
    static constexpr bool SPLIT = Q2 >= 9;
    static constexpr int LS = L2 / 8, BS = LS + 2;
    static constexpr int RS = SPLIT ? 8 * BS : row_stride(L2, R2);
    static constexpr int IMOFF = R2 * RS + 8;
    __device__ __forceinline__ static int POS(int k2) { return SPLIT ? (k2 & 7) * BS + PADI(k2 >> 3) : PADI(k2); }
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

// tile c of one column: rows of W -> (R_k, X_{2k}) in place, scaled;  *xlast = scale X_{N-1}  (tile 0)
template <int Q2, int TL>
__device__ __forceinline__ void phase_b(unsigned char* smem_raw, int log2N, int c, double2* __restrict__ Wc, double scale,
                                        double* __restrict__ xlast, const ATables tabs) {
    using C = PBCfg<Q2, TL>;
    constexpr int L2 = C::L2, GS = C::GS, R2 = C::R2, T = C::T, RS = C::RS, NT = C::NT;
    const int64_t N = (int64_t)1 << log2N, L = N >> 1;
    const int L1 = (int)(L >> Q2);
    double2* lo = (double2*)smem_raw;
    double2* hi = lo + 64;
    double2* rowtw = hi + C::NHI;                    // [R2] exp(-2 pi i row/N)
    double* re = (double*)(rowtw + R2);
    double* im = re + C::IMOFF;
    const int tid = threadIdx.x;
    auto row_of = [&](int slot) {
        int rho = c * T + (slot < T ? slot : slot - T);
        return slot < T ? rho : (rho == 0 ? L1 / 2 : L1 - rho);
    };
    const int g = tid / GS, gt = tid % GS;           // group g transforms row slot g; v[r] = row[gt + r*GS]: first-pass operands
    double2 v[8];
    SUBT0();
    {
        const double2* row = Wc + (int64_t)row_of(g) * L2;
#pragma unroll
        for (int r = 0; r < 8; ++r) v[r] = ldcg2(row + gt + r * GS);
    }
    tw_fetch(lo, hi, tabs.twB, C::NHI, tid, NT);      // exp(-2 pi i u/(2 L2)) = exp(-2 pi i (L1 u)/N)
    for (int i = tid; i < R2; i += NT) {
        double sn, cs; sincospi(-2.0 * (double)row_of(i) / (double)N, &sn, &cs); rowtw[i] = make_double2(cs, sn);
    }
    if constexpr (C::SPLIT) {
        constexpr int QS = Q2 - 3, GSS = C::LS / 8;                   // sub-FFT: 2^QS points, GSS threads
        Bfly<8>::run(v);
        {   // v[r'] *= exp(-2 pi i gt r'/L2) = tw(2 gt r'); the shared tables are not published yet: w1 from the global copy
            const int u = 2 * gt;
            const double2 w1 = cmul(__ldg(tabs.twB + 64 + (u >> 6)), __ldg(tabs.twB + (u & 63)));
            const double2 w2 = cmul(w1, w1), w3 = cmul(w2, w1), w4 = cmul(w2, w2);
            const double2 w5 = cmul(w4, w1), w6 = cmul(w4, w2), w7 = cmul(w4, w3);
            v[1] = cmul(v[1], w1); v[2] = cmul(v[2], w2); v[3] = cmul(v[3], w3); v[4] = cmul(v[4], w4);
            v[5] = cmul(v[5], w5); v[6] = cmul(v[6], w6); v[7] = cmul(v[7], w7);
        }
        double* rg = re + g * RS; double* ig = im + g * RS;
#pragma unroll
        for (int r = 0; r < 8; ++r) { const int idx = r * C::BS + PADI(gt); rg[idx] = v[r].x; ig[idx] = v[r].y; }
        __syncthreads();                              // blocks complete (written by the whole row group); tables published
        const int sg = gt / GSS, lt = gt % GSS;
        fft_smem<QS, NT / GSS>(rg + sg * C::BS, ig + sg * C::BS, lt, tid / GSS, lo, hi, 16);      // exp(-2 pi i mm/Ls) = tw(16 mm)
    } else {
        fft_smem_from_regs<Q2, NT / GS>(v, re + g * RS, im + g * RS, gt, g, lo, hi, 2);      // exp(-2 pi i mm/L2) = tw(2 mm)
    }
    __syncthreads();                                  // per-group barriers inside; the untangle pairs rows of different groups
    SUBT(8);
    // untangle: thread owns the pair {(slot r, k2), its mirror}; k = row + L1*k2
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        int e = tid + i * NT;
        int r = e / L2, k2 = e % L2;
        if (c * T + r >= 1) {                                      // general rows: mirror is (slot T+r, L2-1-k2)
            int ia = r * RS + C::POS(k2), ib = (T + r) * RS + C::POS(L2 - 1 - k2);
            double2 zk = make_double2(re[ia], im[ia]), zm = make_double2(re[ib], im[ib]);
            untangle_pair(zk, zm, cmul(rowtw[r], tw_get(lo, hi, k2)));
            re[ia] = zk.x; im[ia] = zk.y; re[ib] = zm.x; im[ib] = zm.y;
        } else {
            // row 0 pairs with itself: (k2, L2-k2), k2 = 1..L2/2; k2 = 0 holds T_0
            if (k2 == 0) {
                double a = re[0], b = im[0];                    // POS(0) = 0
                re[0] = 0.5 * (a + b); im[0] = 0.0;               // R_0 := X_1 = T_0/2
                *xlast = scale * 0.5 * (b - a);                    // X_{N-1} = -T_L/2: where the last chunk's backward sum starts
            } else if (k2 <= L2 / 2) {
                int ia = C::POS(k2), ib = C::POS(L2 - k2);
                double2 zk = make_double2(re[ia], im[ia]), zm = make_double2(re[ib], im[ib]);
                untangle_pair(zk, zm, tw_get(lo, hi, k2));
                re[ia] = zk.x; im[ia] = zk.y; re[ib] = zm.x; im[ib] = zm.y;
            }
            // slot T holds row L1/2, which also pairs with itself: (k2, L2-1-k2), k2 < L2/2
            if (k2 < L2 / 2) {
                int ia = T * RS + C::POS(k2), ib = T * RS + C::POS(L2 - 1 - k2);
                double2 zk = make_double2(re[ia], im[ia]), zm = make_double2(re[ib], im[ib]);
                untangle_pair(zk, zm, cmul(rowtw[T], tw_get(lo, hi, k2)));
                re[ia] = zk.x; im[ia] = zk.y; re[ib] = zm.x; im[ib] = zm.y;
            }
        }
    }
    __syncthreads();
    SUBT(9);
    // (R_k, X_{2k}) back into the CTA's own rows of W
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int slot = e / L2, k2 = e % L2;
        int ia = slot * RS + C::POS(k2);
        __stcg(&Wc[(int64_t)row_of(slot) * L2 + k2], make_double2(scale * re[ia], scale * im[ia]));
    }
    SUBT(10);
}

// ------------------------------------------------------------------------------------------------ phase C
// Odd outputs P_k = X_{2k+1} of chunk c (k in [c CH, (c+1) CH)) from R_k = P_k - P_{k-1}: first half forward from the
// chunk's anchor P_{c CH}, second half backward from the next chunk's anchor P_{(c+1) CH} (last chunk: from X_{N-1}).
// shared-memory index of local k (0..4095): +1 per 8 (blocked scan reads), +PM per row of K1C (transposed stores: a
// half-warp holds consecutive k2 of one k1, i.e. k's that are K1C apart)
__device__ __forceinline__ int sc_pad(int k, int log2K1C, int PM) { return k + (k >> 3) + (k >> log2K1C) * PM; }
constexpr int SC_ARR = SC_CHUNK + SC_CHUNK / 8 + 32 * 16 + 8;       // doubles per array
static_assert(SC_ARR % 16 == 8, "R and X_even banks interleave in the output loop");
constexpr size_t SC_SMEM = 2 * (size_t)SC_ARR * sizeof(double) + 64 * sizeof(double);

template <int NT>
__device__ __forceinline__ void phase_c(unsigned char* smem_raw, int log2N, int log2L1, int c, const double2* __restrict__ Wc,
                                        double* __restrict__ o, const double* __restrict__ anchors) {
    const int64_t L = (int64_t)1 << (log2N - 1);
    const int nch = (int)(L / SC_CHUNK);
    const int L1 = 1 << log2L1;
    const int64_t L2 = L >> log2L1;
    const int CW = L1 >= SC_CHUNK ? 1 : SC_CHUNK / L1;                // k2's per chunk
    const int log2K1C = L1 >= SC_CHUNK ? 12 : log2L1;                 // k1's per chunk K1C = min(L1, 4096)
    const int K1C = 1 << log2K1C;
    const int PM = CW >= 16 ? 1 : 16 / CW;
    double* sR = (double*)smem_raw;
    double* sX = sR + SC_ARR;
    double* wsum = sX + SC_ARR;                                        // [2][32]
    const int tid = threadIdx.x;
    // chunk c holds k = k1 + L1*k2: (L1 <= 4096) all k1, k2 in [c*CW, (c+1)*CW); (L1 > 4096) one k2 and a range of k1
    const int64_t k2base = L1 >= SC_CHUNK ? ((int64_t)c * SC_CHUNK) / L1 : (int64_t)c * CW;
    const int k1base = L1 >= SC_CHUNK ? (int)(((int64_t)c * SC_CHUNK) % L1) : 0;
    constexpr int PER = SC_CHUNK / NT;
    SUBT0();
    {
        double2 v[PER];
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            const int e = tid + i * NT;
            const int k2o = e % CW, k1 = e / CW;
            v[i] = ldcg2(Wc + (int64_t)(k1base + k1) * L2 + k2base + k2o);
        }
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            const int e = tid + i * NT;
            const int k2o = e % CW, k1 = e / CW;
            const int ix = sc_pad(k1 + K1C * k2o, log2K1C, PM);
            sR[ix] = v[i].x; sX[ix] = v[i].y;
        }
    }
    // bases: forward half starts at the anchor; backward half at P_{(c+1)CH - 1} = anchor_{c+1} - R_{(c+1) CH}
    double base;
    constexpr int HT = NT / 2;                                         // threads per half
    const int half = tid / HT, ht = tid % HT;
    if (half == 0) base = __ldcg(anchors + c);
    else if (c + 1 < nch) {
        const int64_t kn = (int64_t)(c + 1) * SC_CHUNK;               // first k of the next chunk
        base = __ldcg(anchors + c + 1) - ldcg2(Wc + (kn & (L1 - 1)) * L2 + (kn >> log2L1)).x;
    } else base = __ldcg(anchors + nch);                               // X_{N-1}
    __syncthreads();
    SUBT(16);
    // both halves: inclusive scan of a sequence whose first term is dropped (forward u_q = R_q, q >= 1; backward
    // w_j = R_{CH-j}, j >= 1): P_q = base + incl (forward),  P_{CH-1-j} = base - incl (backward)
    double loc[PER]; double run = 0.0;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const int q = ht * PER + i;
        const double val = q == 0 ? 0.0 : sR[sc_pad(half == 0 ? q : SC_CHUNK - q, log2K1C, PM)];
        run += val; loc[i] = run;
    }
    const double incl = group_scan_incl<HT>(run, ht, wsum + 32 * half);       // barriers inside: reads done before the writes below
    const double off = incl - run;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const int q = ht * PER + i;
        if (half == 0) sR[sc_pad(q, log2K1C, PM)] = base + (off + loc[i]);
        else sR[sc_pad(SC_CHUNK - 1 - q, log2K1C, PM)] = base - (off + loc[i]);
    }
    __syncthreads();
    SUBT(17);
    // natural order: X_{2k} at o[2k-1], P_k = X_{2k+1} at o[2k]; the chunk's 8192 outputs are contiguous from o[2 k0 - 1]
    const int64_t obase = 2 * (int64_t)c * SC_CHUNK - 1;
#pragma unroll
    for (int i = 0; i < 2 * PER; ++i) {
        const int j = tid + i * NT;
        const int ix = sc_pad(j >> 1, log2K1C, PM);
        const double val2 = (j & 1) ? sR[ix] : sX[ix];
        if (obase + j >= 0) __stcs(o + obase + j, val2);
    }
    SUBT(18);
}

// ------------------------------------------------------------------------------------------------ the persistent kernel
struct LargeArgs {
    int log2N, batch, gc, G, nA, nB, nC;
    const double* in; int64_t ld_in; double* out; int64_t ld_out; double scale;
    double2* W;            // [2 gc][L]      ring of two column groups
    double2* ypart;        // [2 gc][2 L2]
    double* anchors;       // [2 gc][nch + 1]   (last entry: scale * X_{N-1})
    ATables tabs;          // phase A twiddles (dst1_tables_kernel)
    int* counters;         // [0]: queue head; [1 + 4 col + {0,1,2,3}]: A tiles, B tiles, D, C chunks done for column col
};
enum { PH_A = 0, PH_B = 1, PH_D = 2, PH_C = 3, PH_DONE = 4 };

// queue order: A(0); then for every group g: D(g), B(g), A(g+1), C(g) -- every dependency points at least one phase back
__device__ __forceinline__ void decode_item(const LargeArgs& a, int item, int& phase, int& g, int& local) {
    auto cols = [&](int gg) { int r = a.batch - gg * a.gc; return r < a.gc ? r : a.gc; };
    int i = item;
    const int c0 = cols(0) * a.nA;
    if (i < c0) { phase = PH_A; g = 0; local = i; return; }
    i -= c0;
    const int full = a.gc * (1 + a.nB + a.nA + a.nC);
    const int nfull = a.G >= 2 ? a.G - 2 : 0;                 // groups 0 .. G-3 and their successors are full
    int gg = i / full; if (gg > nfull) gg = nfull;
    i -= gg * full;
    for (; gg < a.G; ++gg) {
        const int cg = cols(gg), cn = gg + 1 < a.G ? cols(gg + 1) : 0;
        if (i < cg) { phase = PH_D; g = gg; local = i; return; }
        i -= cg;
        if (i < a.nB * cg) { phase = PH_B; g = gg; local = i; return; }
        i -= a.nB * cg;
        if (i < a.nA * cn) { phase = PH_A; g = gg + 1; local = i; return; }
        i -= a.nA * cn;
        if (i < a.nC * cg) { phase = PH_C; g = gg; local = i; return; }
        i -= a.nC * cg;
    }
    phase = PH_DONE; g = 0; local = 0;
}

// arrival counters: release increment by one thread after the CTA barrier (the barrier orders the other threads' writes
// before it), acquire load by the waiting CTA's thread 0 before its barrier -- no device-wide fence per thread
__device__ __forceinline__ void wait_count(int* p, int need) {
    cuda::atomic_ref<int, cuda::thread_scope_device> a(*p);
    while (a.load(cuda::memory_order_acquire) < need) __nanosleep(100);
}
__device__ __forceinline__ void arrive_count(int* p) {
    cuda::atomic_ref<int, cuda::thread_scope_device> a(*p);
    a.fetch_add(1, cuda::memory_order_release);
}

template <int Q1, int Q2, int TL> struct FusedCfg {
    static constexpr int NT = (1 << TL) / 8;
    static constexpr int QM = Q1 + Q2 + 1 - 12;                        // log2 of the folded anchor sums per column (Mc = N / 4096)
    static constexpr int MC = 1 << QM;
    static constexpr size_t DSMEM = QM <= 7 ? sizeof(double2) * 2 * MC : sizeof(double) * 2 * (MC + 16) + sizeof(double2) * (64 + MC / 64 + 1);
    static constexpr size_t m1 = PACfg<Q1, TL>::SMEM > PBCfg<Q2, TL>::SMEM ? PACfg<Q1, TL>::SMEM : PBCfg<Q2, TL>::SMEM;
    static constexpr size_t m2 = SC_SMEM > DSMEM ? SC_SMEM : DSMEM;
    static constexpr size_t SMEM = m1 > m2 ? m1 : m2;
};

template <int Q1, int Q2, int TL>
__global__ void __launch_bounds__(FusedCfg<Q1, Q2, TL>::NT, TL <= 12 ? 2 : 1)
dst1_fused_kernel(LargeArgs a) {
    constexpr int NT = FusedCfg<Q1, Q2, TL>::NT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int s_item[4];
    const int64_t L = (int64_t)1 << (a.log2N - 1);
    const int64_t L2 = L >> Q1;
    const int nch = (int)(L / SC_CHUNK);
    const int tid = threadIdx.x;
#ifdef LRP_DST_STATS
    unsigned long long* stats = (unsigned long long*)(a.counters + 1 + 4 * a.batch + 1);      // [5 phases incl. wait][cycles, items]
    long long t_prev = clock64();
#endif
    int next_item = 0;
    if (tid == 0) next_item = atomicAdd(a.counters, 1);
    for (;;) {
        __syncthreads();                                   // previous item's shared memory is dead; s_item reusable
        if (tid == 0) {
            const int item = next_item;
            next_item = atomicAdd(a.counters, 1);          // the queue is read one item ahead: its latency hides behind this item
            int phase, g, local;
            decode_item(a, item, phase, g, local);
            int col = 0, tile = 0;
            if (phase != PH_DONE) {
                const int nt = phase == PH_A ? a.nA : (phase == PH_B ? a.nB : (phase == PH_C ? a.nC : 1));
                col = g * a.gc + local / nt; tile = local % nt;
                int* cnt = a.counters + 1 + 4 * col;
                if (phase == PH_A) { if (g >= 2) wait_count(cnt - 4 * 2 * a.gc + 3, a.nC); }          // ring slot free
                else if (phase == PH_C) { wait_count(cnt + 1, a.nB); wait_count(cnt + 2, 1); }
                else wait_count(cnt, a.nA);                                                            // B, D
            }
#ifdef LRP_DST_STATS
            { long long t = clock64(); atomicAdd(&stats[8], (unsigned long long)(t - t_prev)); atomicAdd(&stats[9], 1ull); t_prev = t; }
#endif
            s_item[0] = phase; s_item[1] = col; s_item[2] = tile; s_item[3] = g;
        }
        __syncthreads();
        const int phase = s_item[0], col = s_item[1], tile = s_item[2], g = s_item[3];
        if (phase == PH_DONE) break;
        const int slot = (g & 1) * a.gc + (col - g * a.gc);
        double2* Wc = a.W + (int64_t)slot * L;
        double2* yp = a.ypart + (int64_t)slot * 2 * L2;
        double* anc = a.anchors + (int64_t)slot * (nch + 1);
        const double* x = a.in + (int64_t)col * a.ld_in;
        if (phase == PH_A) phase_a<Q1, TL>(smem_raw, a.log2N, tile, x, Wc, yp, a.tabs);
        else if (phase == PH_B) phase_b<Q2, TL>(smem_raw, a.log2N, tile, Wc, a.scale, anc + nch, a.tabs);
        else if (phase == PH_D) phase_d<NT, FusedCfg<Q1, Q2, TL>::QM>(smem_raw, a.log2N, Q1, x, yp, a.scale, anc);
        else phase_c<NT>(smem_raw, a.log2N, Q1, tile, Wc, a.out + (int64_t)col * a.ld_out, anc);
        __syncthreads();                                   // every thread's global writes of this item ...
        if (tid == 0) arrive_count(a.counters + 1 + 4 * col + phase);      // ... are released by this increment
#ifdef LRP_DST_STATS
        if (tid == 0) { long long t = clock64(); atomicAdd(&stats[2 * phase], (unsigned long long)(t - t_prev)); atomicAdd(&stats[2 * phase + 1], 1ull); t_prev = t; }
#endif
    }
}

// split L = 2^q = L1 * L2 and the tile size (2^tl points per CTA).  L1 = 256 wherever a pair of rows of L2 still
// fits a CTA (phase A then moves x and W in 128-byte runs and its sub-FFTs are one warp each).
struct Plan { int q1, q2, tl, nA, nB, nC; };
Plan plan(int log2N) {
    const int q = log2N - 1;
    Plan p;
    p.q1 = q <= 14 ? 7 : 8;
    if (q - p.q1 > 12) p.q1 = q - 12;
    p.q2 = q - p.q1;
    p.tl = (p.q1 >= 9 || p.q2 >= 12) ? 13 : 12;
    p.nA = (1 << p.q2) / ((1 << p.tl) >> p.q1);               // L2 / T2
    p.nB = (1 << p.q1) / ((1 << p.tl) >> p.q2);               // L1 / R2
    p.nC = (int)(((int64_t)1 << q) / SC_CHUNK);
    return p;
}

// entries of the two sub-FFT twiddle tables (twA, twB): 64 + NHI each
size_t sub_table_entries(int q1, int q2) { return (size_t)(64 + ((2 << q1) / 64 + 1)) + (size_t)(64 + ((2 << q2) / 64 + 1)); }

// columns per ring slot
int group_cols(int64_t N, int batch) {
    int64_t g = RING_SLOT_BYTES / (N * 8);
    if (g < 1) g = 1;
    if (g > batch) g = batch;
    return (int)g;
}

typedef void (*FusedKernel)(LargeArgs);
struct KernelEntry { int q1, q2, tl; FusedKernel fn; size_t smem; int nt; };
template <int Q1, int Q2, int TL> KernelEntry entry() {
    return KernelEntry{Q1, Q2, TL, dst1_fused_kernel<Q1, Q2, TL>, FusedCfg<Q1, Q2, TL>::SMEM, FusedCfg<Q1, Q2, TL>::NT};
}
const KernelEntry* kernel_table(int* count) {
    static const KernelEntry tab[] = {
        entry<7, 7, 12>(), entry<8, 7, 12>(), entry<8, 8, 12>(), entry<8, 9, 12>(), entry<8, 10, 12>(), entry<8, 11, 12>(),
        entry<8, 12, 13>(), entry<9, 12, 13>(), entry<10, 12, 13>(), entry<11, 12, 13>(), entry<12, 12, 13>()};
    *count = (int)(sizeof(tab) / sizeof(tab[0]));
    return tab;
}

}  // namespace

int dst1_large_init(lrp_ctx* ctx) {
    int cnt; const KernelEntry* tab = kernel_table(&cnt);
    for (int i = 0; i < cnt; ++i)
        LRP_CUDA(ctx, cudaFuncSetAttribute(tab[i].fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tab[i].smem));
    return LRP_OK;
}

size_t dst1_large_ws(int64_t N, int32_t batch) {
    const int gc = group_cols(N, batch);
    const int64_t L = N / 2;
    const Plan p = plan(lrp_ilog2(N));
    const int64_t L2 = (int64_t)1 << p.q2;
    const size_t tab = (size_t)(2 * L2 + L2 * 32 + L2 * (((int64_t)1 << p.q1) + 31) / 32) + sub_table_entries(p.q1, p.q2);
    return lrp_align_up(tab * sizeof(double2)) + lrp_align_up((size_t)2 * gc * L * sizeof(double2)) + lrp_align_up((size_t)2 * gc * 2 * L2 * sizeof(double2)) +
           lrp_align_up((size_t)2 * gc * (p.nC + 1) * sizeof(double)) + lrp_align_up((size_t)(1 + 4 * (size_t)batch + 32) * sizeof(int));
}

#ifdef LRP_DST_STATS
static int* g_dbg_counters = nullptr; static int g_dbg_batch = 0;
extern "C" int lrp_debug_dst_stats(unsigned long long* out) {      // work builds only: 10 values [phase A,B,D,C,wait] x [cycles, items]
    cudaDeviceSynchronize();
    return (int)cudaMemcpy(out, g_dbg_counters + 1 + 4 * g_dbg_batch + 1, 10 * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
}
#endif

int dst1_large(lrp_ctx* ctx, int log2N, int32_t batch, const double* d_in, int64_t ld_in,
               double* d_out, int64_t ld_out, double scale, void* ws, size_t ws_bytes) {
    const int64_t N = (int64_t)1 << log2N, L = N / 2;
    if (log2N > 25) return LRP_ERR_UNSUPPORTED_N;
    const Plan p = plan(log2N);
    const int64_t L2 = (int64_t)1 << p.q2;
    LargeArgs a{};
    a.log2N = log2N; a.batch = batch; a.gc = group_cols(N, batch); a.G = (batch + a.gc - 1) / a.gc;
    a.nA = p.nA; a.nB = p.nB; a.nC = p.nC;
    a.in = d_in; a.ld_in = ld_in; a.out = d_out; a.ld_out = ld_out; a.scale = scale;
    lrp_arena ar(ws, ws_bytes);
    const int64_t nhi = (((int64_t)1 << p.q1) + 31) / 32;
    const int64_t ntab = 2 * L2 + L2 * 32 + L2 * nhi;
    double2* twt = ar.take<double2>((size_t)ntab + sub_table_entries(p.q1, p.q2));
    a.tabs.gB = twt; a.tabs.g4lo = twt + 2 * L2; a.tabs.g4hi = twt + 2 * L2 + L2 * 32;
    double2* twA = twt + ntab; double2* twB = twA + 64 + ((2 << p.q1) / 64 + 1);
    a.tabs.twA = twA; a.tabs.twB = twB;
    a.W = ar.take<double2>((size_t)2 * a.gc * L);
    a.ypart = ar.take<double2>((size_t)2 * a.gc * 2 * L2);
    a.anchors = ar.take<double>((size_t)2 * a.gc * (p.nC + 1));
    a.counters = ar.take<int>(1 + 4 * (size_t)batch + 32);
    if (!ar.ok()) return LRP_ERR_WORKSPACE;
    int cnt; const KernelEntry* tab = kernel_table(&cnt);
    const KernelEntry* ke = nullptr;
    for (int i = 0; i < cnt; ++i) if (tab[i].q1 == p.q1 && tab[i].q2 == p.q2 && tab[i].tl == p.tl) ke = &tab[i];
    if (!ke) return LRP_ERR_UNSUPPORTED_N;
    LRP_CUDA(ctx, cudaMemsetAsync(a.counters, 0, (1 + 4 * (size_t)batch + 32) * sizeof(int), ctx->stream));
    const int64_t items = (int64_t)batch * (p.nA + p.nB + p.nC + 1);
    int64_t grid = (int64_t)ctx->sm_count * (p.tl <= 12 ? 2 : 1);
    if (grid > items) grid = items;
#ifdef LRP_DST_STATS
    g_dbg_counters = a.counters; g_dbg_batch = batch;
#endif
    {
        LRP_PROF(ctx, K_DST_FUSED, 0, 0);
        dst1_tables_kernel<<<(unsigned)((ntab + 255) / 256), 256, 0, ctx->stream>>>(log2N, p.q1, twt, twt + 2 * L2, twt + 2 * L2 + L2 * 32, twA, twB);
        LRP_LAUNCHED(ctx);
    }
    LRP_PROF(ctx, K_DST_FUSED, 16.0 * (double)N * batch, 0);
    ke->fn<<<(unsigned)grid, ke->nt, ke->smem, ctx->stream>>>(a);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}
