// fft_smem.cuh -- shared-memory radix-8/4/2 Stockham FFT building blocks of the DST-I kernels (dst1.cu, dst1_large.cu).
#pragma once
#include "common.cuh"
#include <math.h>

namespace {

// bank swizzle of a shared-memory sequence index (a bijection on every aligned block of 16): stride-1, stride-8 and
// the 8-wide interleaved store patterns of the Stockham passes all become conflict-free for 8-byte accesses
__host__ __device__ constexpr int PADI(int i) { return i ^ ((i >> 3) & 15); }

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

// barrier over the GS threads of group g (of NG groups per CTA): the sub-FFTs of a CTA are independent, so a pass never
// needs to wait for the other groups.  One warp or less: __syncwarp; else a named barrier (ids 1..15) per group.
template <int GS, int NG>
__device__ __forceinline__ void group_bar(int g) {
    if constexpr (GS <= 32) __syncwarp();
    else if constexpr (NG == 1 || NG > 15) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(g + 1), "n"(GS) : "memory");
}

// One Stockham pass of radix R over a length-2^Q complex sequence held in (re, im) (padded with PADI),
// executed by the GS = 2^Q/8 threads of a group (gt = thread in group); every thread keeps its 8 complex
// values in registers across the barrier, so the pass is in place.  Twiddle exp(-2 pi i mm / L) = tw(tw_mul*mm).
template <int Q, int R, bool FIRST, int NG>
__device__ __forceinline__ void fft_pass(double* re, double* im, int gt, int g, int log2Ns,
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
    group_bar<GS, NG>(g);
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
    group_bar<GS, NG>(g);
}

// forward complex FFT of length 2^Q in shared memory, natural order in and out (Stockham autosort).
// g = index of the calling thread's group among the NG groups (of 2^Q/8 threads each) of the CTA.
template <int Q, int NG>
__device__ __forceinline__ void fft_smem(double* re, double* im, int gt, int g,
                                         const double2* lo, const double2* hi, int tw_mul) {
    constexpr int A = Q / 3, B = Q % 3;
    fft_pass<Q, 8, true, NG>(re, im, gt, g, 0, lo, hi, tw_mul);
#pragma unroll
    for (int p = 1; p < A; ++p) fft_pass<Q, 8, false, NG>(re, im, gt, g, 3 * p, lo, hi, tw_mul);
    if (B == 1) fft_pass<Q, 2, false, NG>(re, im, gt, g, 3 * A, lo, hi, tw_mul);
    if (B == 2) fft_pass<Q, 4, false, NG>(re, im, gt, g, 3 * A, lo, hi, tw_mul);
}

// Same transform with the first radix-8 pass fed from registers: v[r] = x[gt + r * 2^Q/8] (what a coalesced global load of
// the row delivers), so the sequence is never stored and re-read before the first butterfly.  The CTA-wide barrier
// after the first pass also publishes twiddle tables built since the last barrier.
template <int Q, int NG>
__device__ __forceinline__ void fft_smem_from_regs(double2 (&v)[8], double* re, double* im, int gt, int g,
                                                   const double2* lo, const double2* hi, int tw_mul) {
    constexpr int A = Q / 3, B = Q % 3;
    Bfly<8>::run(v);
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        int idx = PADI(gt * 8 + r);
        re[idx] = v[r].x; im[idx] = v[r].y;
    }
    __syncthreads();
#pragma unroll
    for (int p = 1; p < A; ++p) fft_pass<Q, 8, false, NG>(re, im, gt, g, 3 * p, lo, hi, tw_mul);
    if (B == 1) fft_pass<Q, 2, false, NG>(re, im, gt, g, 3 * A, lo, hi, tw_mul);
    if (B == 2) fft_pass<Q, 4, false, NG>(re, im, gt, g, 3 * A, lo, hi, tw_mul);
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

}  // namespace
