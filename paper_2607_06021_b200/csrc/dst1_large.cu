// dst1_large.cu -- batched DST-I for N = n + 1 = 2^p > 16384: the column no longer fits one CTA's shared memory.
//
// Same folding as dst1.cu (t -> z, complex FFT of length L = N/2, untangle, prefix sum), with the FFT split
// four-step style, L = L1 * L2, j = j1*L2 + j2, k = k1 + L1*k2:
//   sweep A: fold x on the fly (every x element enters exactly two t's: the CTA owns a j2 tile AND its mirror tile,
//            so each element is fetched from HBM once), length-L1 FFTs over the strided index j1, four-step twiddle,
//            W[k1*L2 + j2] (complex, 8N bytes per column);
//   sweep B: the CTA owns T rows k1 and their mirror rows L1 - k1: length-L2 FFTs, real-FFT untangle of the pairs
//            (k, L-k) in shared memory; (R_k, X_{2k}) with R_k = X_{2k+1} - X_{2k-1} go back IN PLACE into the rows of W
//            (fully coalesced), and the CTA's partial sums of R over every 4096-wide chunk of k go to a small table;
//   sweep C: one CTA per chunk of 4096 consecutive k: gathers its (R, X_even) from the [k1][k2] layout of W (runs of
//            4096/L1 entries), transposes through shared memory, two-sided prefix sum of R from the scanned chunk sums,
//            writes the natural-order output contiguously.
// L1 is kept small (256 where the row of L2 still fits a CTA) so that sweep A reads x and writes W in >= 128-byte runs.
#include "common.cuh"
#include "fft_smem.cuh"
#include <math.h>

namespace {

constexpr int SC_CHUNK = 4096, SC_NT = 512;       // sweep C: k's per chunk, threads per chunk

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
    static constexpr int SLO = 33, SHI = TW_HI | 1;        // odd row strides: the T2 rows are read side by side
    static constexpr int CH = 4;                  // loads in flight per thread (register budget)
    static constexpr size_t SMEM = sizeof(double2) * (64 + NHI + 2 * T2 + (size_t)T2 * (SLO + SHI)) +
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
    double2* t4hi = t4lo + T2 * C::SLO;            // [T2][L1/32] exp(-2 pi i j2 (32 h) / L)
    double* re = (double*)(t4hi + T2 * C::SHI);
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
        if (i < T2 * C::TW_LO) { s = i / C::TW_LO; kk = i % C::TW_LO; dst = t4lo + s * C::SLO + kk; }
        else { int q = i - T2 * C::TW_LO; s = q / C::TW_HI; kk = (q % C::TW_HI) * 32; dst = t4hi + s * C::SHI + (q % C::TW_HI); }
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
        fft_smem<Q1, NT / GS>(re + g * RS, im + g * RS, gt, g, lo, hi, 2);
    }
    __syncthreads();                                  // the sub-FFTs synchronise per group; the store below reads across groups
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int s = e % T2, k1 = e / T2;
        double2 v = make_double2(re[s * RS + PADI(k1)], im[s * RS + PADI(k1)]);
        double2 w = cmul(t4hi[s * C::SHI + (k1 >> 5)], t4lo[s * C::SLO + (k1 & 31)]);
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
dst1_pb_kernel(int log2N, double2* __restrict__ W, double scale, double* __restrict__ xlast, int xstride,
               double* __restrict__ part) {
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
    double2* Wc = W + (int64_t)blockIdx.y * L;
    auto row_of = [&](int slot) {
        int rho = c * T + (slot < T ? slot : slot - T);
        return slot < T ? rho : (rho == 0 ? L1 / 2 : L1 - rho);
    };
    const int g = tid / GS, gt = tid % GS;           // group g transforms row slot g; v[r] = row[gt + r*GS]: first-pass operands
    double2 v[8];
    {
        const double2* row = Wc + (int64_t)row_of(g) * L2;
#pragma unroll
        for (int r = 0; r < 8; ++r) v[r] = row[gt + r * GS];
    }
    tw_build(lo, hi, 2 * L2, C::NHI, tid, NT);        // exp(-2 pi i u/(2 L2)) = exp(-2 pi i (L1 u)/N)
    for (int i = tid; i < R2; i += NT) {
        double sn, cs; sincospi(-2.0 * (double)row_of(i) / (double)N, &sn, &cs); rowtw[i] = make_double2(cs, sn);
    }
    fft_smem_from_regs<Q2, NT / GS>(v, re + g * RS, im + g * RS, gt, g, lo, hi, 2);      // exp(-2 pi i mm/L2) = tw(2 mm)
    __syncthreads();                                  // per-group barriers inside; the untangle pairs rows of different groups
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
    // (R_k, X_{2k}) back into the CTA's own rows of W
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int e = tid + i * NT;
        int slot = e / L2, k2 = e % L2;
        int ia = slot * RS + PADI(k2);
        Wc[(int64_t)row_of(slot) * L2 + k2] = make_double2(scale * re[ia], scale * im[ia]);
    }
    // partial chunk sums of R: chunk of k = row + L1*k2 is k2 / CW (L1 <= SC_CHUNK), fixed order -> deterministic
    {
        const int CW = SC_CHUNK / L1 > 0 ? SC_CHUNK / L1 : 1;
        const int nch = L2 / CW;
        double* pc = part + ((int64_t)blockIdx.y * gridDim.x + c) * nch;
        for (int ch = tid; ch < nch; ch += NT) {
            double acc = 0.0;
            for (int slot = 0; slot < R2; ++slot)
                for (int j = 0; j < CW; ++j) acc += re[slot * RS + PADI(ch * CW + j)];
            pc[ch] = scale * acc;
        }
    }
}

// ------------------------------------------------------------------------------------------------ sweep C
// Odd outputs P_k = X_{2k+1} from R_k = P_k - P_{k-1} (R_0 = X_1): a TWO-SIDED sum.  Lower half of the chunks forward
// from P_0 = X_1, upper half backward from the independently known P_{L-1} = X_{N-1} (sweep B, xlast): every output is
// reached through the shorter chain and the small tail of a decaying spectrum is summed from small terms only.
// sums: per column nchunks chunk sums + 1 slot for X_{N-1}; part: per column [nB][nchunks] partial sums of sweep B.

// chunk sums from sweep B's partials: one thread per chunk, fixed order over the nB contributing CTAs (deterministic)
__global__ void __launch_bounds__(128)
dst1_chunkreduce_kernel(int nchunks, int nB, const double* __restrict__ part, double* __restrict__ sums) {
    const int ch = blockIdx.x * 128 + threadIdx.x;
    if (ch >= nchunks) return;
    const double* pc = part + (int64_t)blockIdx.y * nB * nchunks + ch;
    double acc = 0.0;
    int b = 0;
    for (; b + 4 <= nB; b += 4) {
        double v0 = pc[(int64_t)b * nchunks], v1 = pc[(int64_t)(b + 1) * nchunks];
        double v2 = pc[(int64_t)(b + 2) * nchunks], v3 = pc[(int64_t)(b + 3) * nchunks];
        acc += v0; acc += v1; acc += v2; acc += v3;
    }
    for (; b < nB; ++b) acc += pc[(int64_t)b * nchunks];
    sums[(int64_t)blockIdx.y * (nchunks + 1) + ch] = acc;
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

// shared-memory index of local k (0..4095): +1 per 8 (blocked scan reads: thread t owns k = 8t..8t+7), +PM per row of
// K1C (transposed stores: a half-warp holds consecutive k2 of one k1, i.e. k's that are K1C apart)
__device__ __forceinline__ int sc_pad(int k, int log2K1C, int PM) { return k + (k >> 3) + (k >> log2K1C) * PM; }
constexpr int SC_ARR = SC_CHUNK + SC_CHUNK / 8 + 32 * 16 + 8;       // doubles per array
static_assert(SC_ARR % 16 == 8, "R and X_even banks interleave in the output loop");

__global__ void __launch_bounds__(SC_NT)
dst1_scanapply_kernel(int log2N, int log2L1, const double2* __restrict__ W, double* __restrict__ out, int64_t ld_out,
                      const double* __restrict__ sums) {
    const int64_t L = (int64_t)1 << (log2N - 1);
    const int nch = (int)(L / SC_CHUNK);
    const int L1 = 1 << log2L1;
    const int64_t L2 = L >> log2L1;
    const int CW = L1 >= SC_CHUNK ? 1 : SC_CHUNK / L1;                // k2's per chunk
    const int log2K1C = L1 >= SC_CHUNK ? 12 : log2L1;                 // k1's per chunk K1C = min(L1, 4096)
    const int K1C = 1 << log2K1C;
    const int PM = CW >= 16 ? 1 : 16 / CW;
    const int c = blockIdx.x;
    const bool fwd = c < nch / 2;
    const double2* Wc = W + (int64_t)blockIdx.y * L;
    double* o = out + (int64_t)blockIdx.y * ld_out;
    const double* sc = sums + (int64_t)blockIdx.y * (nch + 1);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* sR = (double*)smem_raw;
    double* sX = sR + SC_ARR;
    __shared__ double wsum[32];
    // chunk c holds k = k1 + L1*k2: (L1 <= 4096) all k1, k2 in [c*CW, (c+1)*CW); (L1 > 4096) one k2 and a range of k1
    const int64_t k2base = L1 >= SC_CHUNK ? ((int64_t)c * SC_CHUNK) / L1 : (int64_t)c * CW;
    const int k1base = L1 >= SC_CHUNK ? (int)(((int64_t)c * SC_CHUNK) % L1) : 0;
    constexpr int PER = SC_CHUNK / SC_NT;
    double2 v[PER];
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const int e = threadIdx.x + i * SC_NT;
        const int k2o = e % CW, k1 = e / CW;
        v[i] = Wc[(int64_t)(k1base + k1) * L2 + k2base + k2o];
    }
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const int e = threadIdx.x + i * SC_NT;
        const int k2o = e % CW, k1 = e / CW;
        const int ix = sc_pad(k1 + K1C * k2o, log2K1C, PM);
        sR[ix] = v[i].x; sX[ix] = v[i].y;
    }
    __syncthreads();
    double loc[PER], val[PER]; double run = 0.0;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const int q = threadIdx.x * PER + i;
        val[i] = sR[sc_pad(fwd ? q : SC_CHUNK - 1 - q, log2K1C, PM)];
        run += val[i]; loc[i] = run;
    }
    double incl = group_scan_incl<SC_NT>(run, threadIdx.x, wsum);
    const double off = incl - run;
    if (fwd) {
        const double base = sc[c];
#pragma unroll
        for (int i = 0; i < PER; ++i) sR[sc_pad(threadIdx.x * PER + i, log2K1C, PM)] = base + off + loc[i];     // P_k
    } else {
        const double xl = sc[nch], above = sc[c];
#pragma unroll
        for (int i = 0; i < PER; ++i)                                // P_k = X_{N-1} - sum_{m > k} R_m
            sR[sc_pad(SC_CHUNK - 1 - (threadIdx.x * PER + i), log2K1C, PM)] = xl - (above + (off + loc[i] - val[i]));
    }
    __syncthreads();
    // natural order: X_{2k} at o[2k-1], P_k = X_{2k+1} at o[2k]; the chunk's 8192 outputs are contiguous from o[2 k0 - 1]
    const int64_t obase = 2 * (int64_t)c * SC_CHUNK - 1;
#pragma unroll
    for (int i = 0; i < 2 * PER; ++i) {
        const int j = threadIdx.x + i * SC_NT;
        const int ix = sc_pad(j >> 1, log2K1C, PM);
        const double val2 = (j & 1) ? sR[ix] : sX[ix];
        if (obase + j >= 0) o[obase + j] = val2;
    }
}

// ------------------------------------------------------------------------------------------------ host side
template <int Q1, int TL>
int launch_pa(lrp_ctx* ctx, int log2N, int cols, const double* in, int64_t ld_in, double2* W) {
    using C = PACfg<Q1, TL>;
    const int L2 = 1 << (log2N - 1 - Q1);
    LRP_PROF(ctx, K_DST_P1, 16.0 * ((int64_t)1 << log2N) * cols, 0);
    dst1_pa_kernel<Q1, TL><<<dim3(L2 / C::T2, cols), C::NT, C::SMEM, ctx->stream>>>(log2N, in, ld_in, W);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}
template <int Q2, int TL>
int launch_pb(lrp_ctx* ctx, int log2N, int cols, double2* W, double scale, double* xlast, int xstride, double* part) {
    using C = PBCfg<Q2, TL>;
    const int L1 = 1 << (log2N - 1 - Q2);
    LRP_PROF(ctx, K_DST_P2, 16.0 * ((int64_t)1 << log2N) * cols, 0);
    dst1_pb_kernel<Q2, TL><<<dim3(L1 / C::R2, cols), C::NT, C::SMEM, ctx->stream>>>(log2N, W, scale, xlast, xstride, part);
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
int dispatch_pb(int q2, int tl, lrp_ctx* ctx, int log2N, int cols, double2* W, double scale, double* xlast, int xstride,
                double* part) {
    if (tl == 12) { LRP_QL_SWITCH(q2, 12, launch_pb, ctx, log2N, cols, W, scale, xlast, xstride, part) }
    if (q2 == 12) return launch_pb<12, 13>(ctx, log2N, cols, W, scale, xlast, xstride, part);
    LRP_QL_SWITCH(q2, 13, launch_pb, ctx, log2N, cols, W, scale, xlast, xstride, part)
}

// split L = 2^q = L1 * L2 and the tile sizes (2^tl points per CTA) of the two sweeps.  L1 = 256 wherever a pair of
// rows of L2 still fits a CTA (sweep A then moves x and W in 128-byte runs and its sub-FFTs are one warp each).
struct Plan { int q1, q2, tla, tlb, nB, nch; };
int tile_rows(int tl, int q) { return 1 << (tl - q); }
Plan plan(int log2N) {
    const int q = log2N - 1;
    Plan p;
    p.q1 = q <= 14 ? 7 : 8;
    if (q - p.q1 > 12) p.q1 = q - 12;
    p.q2 = q - p.q1;
    p.tla = p.q1 >= 9 ? 13 : 12;
    p.tlb = p.q2 >= 12 ? 13 : 12;
    p.nB = (1 << p.q1) / tile_rows(p.tlb, p.q2);
    p.nch = (int)(((int64_t)1 << q) / SC_CHUNK);
    return p;
}

// columns per group (workspace bound: W of one group)
int group_cols(int64_t N, int batch) {
    int64_t per_col = N * 8;
    const int64_t budget_mb = 4096;
    int g = (int)((budget_mb << 20) / per_col);
    if (g < 1) g = 1;
    if (g > batch) g = batch;
    return g;
}

template <int Q, int TL>
int init_pair(lrp_ctx* ctx) {
    LRP_CUDA(ctx, cudaFuncSetAttribute(dst1_pa_kernel<Q, TL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PACfg<Q, TL>::SMEM));
    LRP_CUDA(ctx, cudaFuncSetAttribute(dst1_pb_kernel<Q, TL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PBCfg<Q, TL>::SMEM));
    return LRP_OK;
}

}  // namespace

int dst1_large_init(lrp_ctx* ctx) {
    LRP_TRY((init_pair<7, 12>(ctx))); LRP_TRY((init_pair<8, 12>(ctx))); LRP_TRY((init_pair<9, 12>(ctx)));
    LRP_TRY((init_pair<10, 12>(ctx))); LRP_TRY((init_pair<11, 12>(ctx)));
    LRP_TRY((init_pair<7, 13>(ctx))); LRP_TRY((init_pair<8, 13>(ctx))); LRP_TRY((init_pair<9, 13>(ctx)));
    LRP_TRY((init_pair<10, 13>(ctx))); LRP_TRY((init_pair<11, 13>(ctx))); LRP_TRY((init_pair<12, 13>(ctx)));
    LRP_CUDA(ctx, cudaFuncSetAttribute(dst1_scanapply_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * SC_ARR * (int)sizeof(double)));
    return LRP_OK;
}

size_t dst1_large_ws(int64_t N, int32_t batch) {
    const int g = group_cols(N, batch);
    const int64_t L = N / 2;
    const Plan p = plan(lrp_ilog2(N));
    return lrp_align_up((size_t)g * L * sizeof(double2)) + lrp_align_up((size_t)g * (p.nch + 1) * sizeof(double)) +
           lrp_align_up((size_t)g * p.nB * p.nch * sizeof(double));
}

int dst1_large(lrp_ctx* ctx, int log2N, int32_t batch, const double* d_in, int64_t ld_in,
               double* d_out, int64_t ld_out, double scale, void* ws, size_t ws_bytes) {
    const int64_t N = (int64_t)1 << log2N, L = N / 2;
    if (log2N > 25) return LRP_ERR_UNSUPPORTED_N;
    const Plan p = plan(log2N);
    const int g = group_cols(N, batch);
    lrp_arena ar(ws, ws_bytes);
    double2* W = ar.take<double2>((size_t)g * L);
    double* sums = ar.take<double>((size_t)g * (p.nch + 1));
    double* part = ar.take<double>((size_t)g * p.nB * p.nch);
    if (!ar.ok()) return LRP_ERR_WORKSPACE;
    constexpr int SC_SMEM = 2 * SC_ARR * (int)sizeof(double);
    for (int c0 = 0; c0 < batch; c0 += g) {
        const int cols = (batch - c0) < g ? (batch - c0) : g;
        double* o = d_out + (int64_t)c0 * ld_out;
        LRP_TRY(dispatch_pa(p.q1, p.tla, ctx, log2N, cols, d_in + (int64_t)c0 * ld_in, ld_in, W));
        LRP_TRY(dispatch_pb(p.q2, p.tlb, ctx, log2N, cols, W, scale, sums + p.nch, p.nch + 1, part));
        LRP_PROF(ctx, K_DST_CHUNKSUM, 8.0 * p.nB * p.nch * cols, 0);
        dst1_chunkreduce_kernel<<<dim3((p.nch + 127) / 128, cols), 128, 0, ctx->stream>>>(p.nch, p.nB, part, sums);
        LRP_LAUNCHED(ctx);
        LRP_PROF(ctx, K_DST_SCANSUMS, 0, 0);
        dst1_scansums_kernel<<<cols, 1024, 0, ctx->stream>>>(p.nch, sums);
        LRP_LAUNCHED(ctx);
        LRP_PROF(ctx, K_DST_FINISH, 16.0 * N * cols, 0);
        dst1_scanapply_kernel<<<dim3(p.nch, cols), SC_NT, SC_SMEM, ctx->stream>>>(log2N, p.q1, W, o, ld_out, sums);
        LRP_LAUNCHED(ctx);
    }
    return LRP_OK;
}
