// tall_mma.cu -- the two dense contractions over tall matrices on the fp64 tensor pipe (DMMA, mma.sync m8n8k4 f64):
//   tall_gemm   : Out(n x m) = epilogue( A(n x k) B(k x m) )    fiber sampling (eq. (4)), factor
//                 rebuild U = Q Uc (Alg. 1 lines 9/14), Gram-Schmidt update P -= Q S
//   tall_gemm_t : S(k x m) = A(n x k)^T B(n x m)                projections / Gram blocks (reduction over n)
// fp64 has no tcgen05/TMEM path on sm_100a: the fp64 tensor pipe is the warp-level DMMA.  Its peak equals the DFMA
// peak, but one DMMA retires 256 FMAs for two operand registers per thread, which removes the shared-memory /
// issue-slot limit of a register-tiled DFMA kernel (profiles/r01a: 2.4-2.7 TFLOP/s).
#include "common.cuh"
#include "tall.cuh"
#include <math.h>

namespace {

// D(8x8) += A(8x4, row) * B(4x8, col).  lane: g = lane>>2, tg = lane&3.
//   a = A[g][tg],  b = B[tg][g],  (c0, c1) = C[g][2 tg + {0,1}]
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// d_i = lambda_{i+1} / h^2 = 4 N^2 sin^2(pi (i+1) / (2N))   (PAPER.md:200 as 4 sin^2(theta/2), reading Q1)
__device__ __forceinline__ double eig_d(int64_t i, double invN, double fourN2) {
    double s = sinpi(0.5 * (double)(i + 1) * invN);
    return fourN2 * s * s;
}

constexpr int MG_THREADS = 128;                      // 4 warps x 32 rows; column tiles of 8*NJ (NJ = 2 for m <= 16: fewer
                                                     // accumulator registers -> more CTAs per SM for the memory-bound shapes)

__host__ __device__ inline int mg_kp(int k) {         // padded k: multiple of 4 rounded up to (kp % 16 == 4)
    int k4 = (k + 3) & ~3;
    return k4 + (((4 - k4 % 16) + 16) % 16);
}

// Row mapping of a warp's 32 rows: fragment i (0..3) of lane group g holds row R0 + 16 (i>>1) + 2 g + (i&1), so that
// a thread owns row PAIRS and, when the operands are 16-byte aligned with even leading dimensions (VEC), moves them
// with 128-bit loads / stores (the output-row order of an MMA is bookkeeping only).
template <int NJ, bool VEC>
__global__ void __launch_bounds__(MG_THREADS, NJ == 2 ? 5 : (NJ <= 4 ? 4 : 3))
tall_gemm_mma_kernel(TallGemmArgs p) {
    constexpr int MG_CT = 8 * NJ;
    extern __shared__ __align__(16) double smem[];
    if (p.cond && *p.cond == 0) return;               // conditional launch (device-side decision, qr.cu): grid-uniform
    const int kp = mg_kp(p.k), k4 = (p.k + 3) & ~3;
    double* Bs = smem;                                // [MG_CT][kp]: Bs[c*kp + t] = B(t, c0 + c)
    double* dcol = smem + (size_t)MG_CT * kp;         // [MG_CT]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, tg = lane & 3;
    const double invN = 1.0 / (double)(p.n + 1);
    const double fourN2 = 4.0 * (double)(p.n + 1) * (double)(p.n + 1);
    const int64_t nslab = (p.n + MG_THREADS - 1) / MG_THREADS;
    for (int c0 = 0; c0 < p.m; c0 += MG_CT) {
        __syncthreads();
        for (int e = tid; e < MG_CT * k4; e += MG_THREADS) {
            int t = e % k4, c = e / k4;
            double v = 0.0;
            if (t < p.k && c0 + c < p.m) {
                if (p.mode == TG_SAMPLE) v = p.B[(int64_t)p.idx[c0 + c] + (int64_t)t * p.ldb] * p.scale_t[t];
                else v = p.B[(int64_t)t + (int64_t)(c0 + c) * p.ldb];
            }
            Bs[c * kp + t] = v;
        }
        if (p.mode == TG_SAMPLE)
            for (int c = tid; c < MG_CT; c += MG_THREADS) dcol[c] = (c0 + c < p.m) ? eig_d(p.idx[c0 + c], invN, fourN2) : 1.0;
        __syncthreads();
      for (int64_t slab = blockIdx.x; slab < nslab; slab += gridDim.x) {   // B staged once, the CTA streams its row slabs
        const int64_t R0 = slab * MG_THREADS + warp * 32;
        int64_t rows[4]; bool valid[4]; double drow[4], nrm[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            rows[i] = R0 + 16 * (i >> 1) + 2 * g + (i & 1); valid[i] = rows[i] < p.n;
            drow[i] = (p.mode == TG_SAMPLE && valid[i]) ? eig_d(rows[i], invN, fourN2) : 0.0;
            nrm[i] = 0.0;
        }
        double acc[4][NJ][2];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }
#pragma unroll 4
        for (int t0 = 0; t0 < k4; t0 += 4) {
            const int t = t0 + tg;
            double a[4], b[NJ];
            if (VEC) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    double2 v = make_double2(0.0, 0.0);
                    if (valid[2 * h] && t < p.k) v = *reinterpret_cast<const double2*>(p.A + rows[2 * h] + (int64_t)t * p.lda);
                    a[2 * h] = v.x; a[2 * h + 1] = v.y;
                }
            } else {
#pragma unroll
                for (int i = 0; i < 4; ++i) a[i] = (valid[i] && t < p.k) ? p.A[rows[i] + (int64_t)t * p.lda] : 0.0;
            }
#pragma unroll
            for (int j = 0; j < NJ; ++j) b[j] = Bs[(8 * j + g) * kp + t];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < NJ; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (!valid[2 * h]) continue;
            const bool pair = VEC && valid[2 * h + 1];
#pragma unroll
            for (int j = 0; j < NJ; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int cl = 8 * j + 2 * tg + e, col = c0 + cl;
                    if (col >= p.m) continue;
                    double v0 = acc[2 * h][j][e], v1 = acc[2 * h + 1][j][e];
                    if (p.mode == TG_SAMPLE) { v0 = v0 / (drow[2 * h] + dcol[cl]); v1 = v1 / (drow[2 * h + 1] + dcol[cl]); }
                    if (pair) {
                        if (p.mode == TG_SUBTRACT) {
                            double2 cin = *reinterpret_cast<const double2*>(p.Cin + rows[2 * h] + (int64_t)col * p.ldc);
                            v0 = cin.x - v0; v1 = cin.y - v1;
                        }
                        *reinterpret_cast<double2*>(p.Out + rows[2 * h] + (int64_t)col * p.ldo) = make_double2(v0, v1);
                        nrm[2 * h] = fma(v0, v0, nrm[2 * h]); nrm[2 * h + 1] = fma(v1, v1, nrm[2 * h + 1]);
                    } else {
                        if (p.mode == TG_SUBTRACT) v0 = p.Cin[rows[2 * h] + (int64_t)col * p.ldc] - v0;
                        p.Out[rows[2 * h] + (int64_t)col * p.ldo] = v0;
                        nrm[2 * h] = fma(v0, v0, nrm[2 * h]);
                        if (valid[2 * h + 1]) {
                            if (p.mode == TG_SUBTRACT) v1 = p.Cin[rows[2 * h + 1] + (int64_t)col * p.ldc] - v1;
                            p.Out[rows[2 * h + 1] + (int64_t)col * p.ldo] = v1;
                            nrm[2 * h + 1] = fma(v1, v1, nrm[2 * h + 1]);
                        }
                    }
                }
        }
        if (p.rownorm2) {                              // row norms accumulate over the column tiles
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                double s = nrm[i];
                s += __shfl_xor_sync(0xffffffffu, s, 1);
                s += __shfl_xor_sync(0xffffffffu, s, 2);
                if (tg == 0 && valid[i]) p.rownorm2[rows[i]] = (c0 == 0 ? 0.0 : p.rownorm2[rows[i]]) + s;
            }
        }
      }
    }
}

// ---- S = A^T B: 8 warps per CTA; the CTA owns ntc <= 8 tiles (16 x 16) of S and its row slab; the 8/ntc warps
//      that share a tile split the slab's rows and are summed through shared memory in a fixed order -------------
constexpr int MT_THREADS = 256;
constexpr int GT_GROUP = 16;                          // row slabs per first-level reduction group
constexpr int GT_MAXGRP = 64;                         // counters [0, 64): groups, [64]: the final level
struct GemmTOut { double* S; int64_t lds; int accumulate; double* Sadd; int64_t ldadd; double* gpartial; unsigned* counters; const int* cond; };

// ---- in-kernel reduction over the row slabs, two levels, fixed summation order (deterministic): the last CTA to
// finish in a group of GT_GROUP slabs sums the group's partials, the last group to finish sums the groups and writes
// S.  No second launch: a small dependent kernel queues behind whatever the other streams have in flight.  The
// counters return to zero, so they are initialised once per context.  Every thread of every CTA of the grid calls it
// (gridDim.x slabs, gridDim.y CTAs per slab) after its slab's partial entries are written.
__device__ __forceinline__ void slab_reduce_tail(double* partial, int k, int m, const GemmTOut& o, int* s_role) {
    const int km = k * m, nthr = blockDim.x;
    const int grp = blockIdx.x / GT_GROUP;
    const int g_lo = grp * GT_GROUP, g_hi = min(g_lo + GT_GROUP, (int)gridDim.x);
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned t = atomicAdd(&o.counters[grp], 1u);
        int role = 0;
        if (t == (unsigned)((g_hi - g_lo) * gridDim.y) - 1u) { o.counters[grp] = 0u; role = 1; }
        *s_role = role;
    }
    __syncthreads();
    if (*s_role == 0) return;
    __threadfence();
    double* gp = o.gpartial + (int64_t)grp * km;
    for (int e = threadIdx.x; e < km; e += nthr) {
        double v0 = 0.0, v1 = 0.0;
        int b = g_lo;
        for (; b + 1 < g_hi; b += 2) { v0 += __ldcg(partial + (int64_t)b * km + e); v1 += __ldcg(partial + (int64_t)(b + 1) * km + e); }
        if (b < g_hi) v0 += __ldcg(partial + (int64_t)b * km + e);
        gp[e] = v0 + v1;
    }
    __threadfence();
    __syncthreads();
    const int ngrp = (gridDim.x + GT_GROUP - 1) / GT_GROUP;
    if (threadIdx.x == 0) {
        const unsigned t = atomicAdd(&o.counters[GT_MAXGRP], 1u);
        int role = 1;
        if (t == (unsigned)ngrp - 1u) { o.counters[GT_MAXGRP] = 0u; role = 2; }
        *s_role = role;
    }
    __syncthreads();
    if (*s_role != 2) return;
    __threadfence();
    for (int e = threadIdx.x; e < km; e += nthr) {
        double v0 = 0.0, v1 = 0.0;
        int q = 0;
        for (; q + 1 < ngrp; q += 2) { v0 += __ldcg(o.gpartial + (int64_t)q * km + e); v1 += __ldcg(o.gpartial + (int64_t)(q + 1) * km + e); }
        if (q < ngrp) v0 += __ldcg(o.gpartial + (int64_t)q * km + e);
        const double v = v0 + v1;
        const int a = e % k, c = e / k;
        double* dst = o.S + a + (int64_t)c * o.lds;
        *dst = o.accumulate ? (*dst + v) : v;
        if (o.Sadd) o.Sadd[a + (int64_t)c * o.ldadd] += v;
    }
}

template <bool VEC>
__global__ void __launch_bounds__(MT_THREADS)
tall_gemm_t_mma_kernel(const double* __restrict__ A, int64_t lda, int k, const double* __restrict__ B, int64_t ldb, int m,
                       int64_t n, int64_t rows_per_cta, double* partial, int na, int nb, int ntc, GemmTOut o) {
    __shared__ double red[MT_THREADS / 32][8][32];
    __shared__ int s_role;
    if (o.cond && *o.cond == 0) return;                     // conditional launch: grid-uniform, counters untouched
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, g = lane >> 2, tg = lane & 3;
    const int nsub = (MT_THREADS / 32) / ntc;               // warps per tile
    const int tl = warp % ntc, sub = warp / ntc;
    const int tile = blockIdx.y * ntc + tl;
    const bool active = tile < na * nb && sub < nsub;
    const int a0 = 16 * (tile % na), b0 = 16 * (tile / na);
    const int64_t c_begin = (int64_t)blockIdx.x * rows_per_cta;
    int64_t c_end = c_begin + rows_per_cta; if (c_end > n) c_end = n;
    double acc[2][2][2] = {};
    if (active) {
        const int ca0 = a0 + g, ca1 = a0 + 8 + g, cb0 = b0 + g, cb1 = b0 + 8 + g;
        const double* pa0 = A + (int64_t)(ca0 < k ? ca0 : 0) * lda; const double* pa1 = A + (int64_t)(ca1 < k ? ca1 : 0) * lda;
        const double* pb0 = B + (int64_t)(cb0 < m ? cb0 : 0) * ldb; const double* pb1 = B + (int64_t)(cb1 < m ? cb1 : 0) * ldb;
        // the warps sharing a tile take interleaved 16-row chunks, so that at any time the CTA streams one contiguous
        // 16*nsub-row run of every column (DRAM row-buffer locality; blocked sub-slabs measured 28 % of HBM peak)
        for (int64_t rb = c_begin + 16 * sub; rb < c_end; rb += 16 * nsub) {   // warp-uniform (mma.sync needs the whole warp)
            const int64_t r = rb + tg;
            double x0[4], x1[4], y0[4], y1[4];
            if (VEC && rb + 16 <= c_end) {
                // 128-bit loads of row pairs: MMA step 2u takes rows rb + 8u + 2 tg, step 2u+1 the rows after them (the
                // order of the summed rows is free as long as both operands use the same one)
                const int64_t rv2 = rb + 2 * tg;
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    double2 a0 = *reinterpret_cast<const double2*>(pa0 + rv2 + 8 * u), a1 = *reinterpret_cast<const double2*>(pa1 + rv2 + 8 * u);
                    double2 b0 = *reinterpret_cast<const double2*>(pb0 + rv2 + 8 * u), b1 = *reinterpret_cast<const double2*>(pb1 + rv2 + 8 * u);
                    x0[2 * u] = a0.x; x0[2 * u + 1] = a0.y; x1[2 * u] = a1.x; x1[2 * u + 1] = a1.y;
                    y0[2 * u] = b0.x; y0[2 * u + 1] = b0.y; y1[2 * u] = b1.x; y1[2 * u + 1] = b1.y;
                }
            } else if (rb + 16 <= c_end) {
#pragma unroll
                for (int u = 0; u < 4; ++u) { x0[u] = pa0[r + 4 * u]; x1[u] = pa1[r + 4 * u]; y0[u] = pb0[r + 4 * u]; y1[u] = pb1[r + 4 * u]; }
            } else {
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const bool rv = r + 4 * u < c_end;
                    x0[u] = rv ? pa0[r + 4 * u] : 0.0; x1[u] = rv ? pa1[r + 4 * u] : 0.0;
                    y0[u] = rv ? pb0[r + 4 * u] : 0.0; y1[u] = rv ? pb1[r + 4 * u] : 0.0;
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                dmma(acc[0][0][0], acc[0][0][1], x0[u], y0[u]); dmma(acc[0][1][0], acc[0][1][1], x0[u], y1[u]);
                dmma(acc[1][0][0], acc[1][0][1], x1[u], y0[u]); dmma(acc[1][1][0], acc[1][1][1], x1[u], y1[u]);
            }
        }
    }
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) red[warp][(i * 2 + j) * 2 + e][lane] = acc[i][j][e];
    __syncthreads();
    if (sub == 0 && tile < na * nb) {
        double* P = partial + (int64_t)blockIdx.x * k * m;
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 2; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    double v = 0.0;
                    for (int s2 = 0; s2 < nsub; ++s2) v += red[tl + s2 * ntc][(i * 2 + j) * 2 + e][lane];
                    int a = a0 + 8 * i + g, b = b0 + 8 * j + 2 * tg + e;
                    if (a < k && b < m) P[a + (int64_t)b * k] = v;
                }
    }
    slab_reduce_tail(partial, k, m, o, &s_role);
}

// ---- G = E^T E with E = Cin - A B (n x m) formed on the fly and never written: the rho update of the stop test
//      (Alg. 4 line 24 in the factored form of DESIGN.md: E_U = U_{k-1} - U_k (U_k^T U_{k-1})).  One pass over A and Cin
//      instead of an update sweep (read A, Cin, write E) plus a Gram sweep (read E).  Per warp and 32-row slab: E in the
//      DMMA accumulators as in tall_gemm, through shared memory into fragment layout (the same registers serve as the
//      A and the B operand of E^T E), upper-triangular 8 x 8 tiles of G accumulated over the CTA's slabs; per-CTA
//      partials are reduced inside the kernel like those of tall_gemm_t.
constexpr int RG_THREADS = 128;
__host__ __device__ inline int rg_lde(int m8) { return m8 + (((4 - m8 % 16) + 16) % 16); }      // == 4 (mod 16): conflict-free fragments

template <int NJ>
__global__ void __launch_bounds__(RG_THREADS, NJ <= 5 ? 3 : 2)
tall_resid_gram_kernel(int64_t n, const double* __restrict__ A, int64_t lda, int k, const double* __restrict__ B, int64_t ldb,
                       const double* __restrict__ Cin, int64_t ldc, int m, double* partial, GemmTOut o) {
    constexpr int NT2 = NJ * (NJ + 1) / 2;
    extern __shared__ __align__(16) double smem[];
    __shared__ int s_role;
    const int kp = mg_kp(k), k4 = (k + 3) & ~3, lde = rg_lde(8 * NJ);
    double* Bs = smem;                                            // [8 NJ][kp]
    double* Es_all = smem + (size_t)8 * NJ * kp;                  // [4 warps][32][lde]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, tg = lane & 3;
    double* Es = Es_all + (size_t)warp * 32 * lde;
    for (int e = tid; e < 8 * NJ * k4; e += RG_THREADS) {
        const int t = e % k4, c = e / k4;
        Bs[c * kp + t] = (t < k && c < m) ? B[(int64_t)t + (int64_t)c * ldb] : 0.0;
    }
    __syncthreads();
    double gacc[NT2][2];
#pragma unroll
    for (int t = 0; t < NT2; ++t) { gacc[t][0] = 0.0; gacc[t][1] = 0.0; }
    const int64_t nslab = (n + RG_THREADS - 1) / RG_THREADS;
    for (int64_t slab = blockIdx.x; slab < nslab; slab += gridDim.x) {
        const int64_t R0 = slab * RG_THREADS + warp * 32;
        int64_t rows[4]; bool valid[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) { rows[i] = R0 + 16 * (i >> 1) + 2 * g + (i & 1); valid[i] = rows[i] < n; }
        double acc[4][NJ][2];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }
#pragma unroll 4
        for (int t0 = 0; t0 < k4; t0 += 4) {
            const int t = t0 + tg;
            double a[4], b[NJ];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                double2 v = make_double2(0.0, 0.0);
                if (valid[2 * h] && t < k) v = *reinterpret_cast<const double2*>(A + rows[2 * h] + (int64_t)t * lda);
                a[2 * h] = v.x; a[2 * h + 1] = valid[2 * h + 1] ? v.y : 0.0;
            }
#pragma unroll
            for (int j = 0; j < NJ; ++j) b[j] = Bs[(8 * j + g) * kp + t];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < NJ; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
        // E = Cin - A B into the warp's shared-memory tile (rows local 16 (i>>1) + 2 g + (i&1)); invalid rows / columns are zero
        __syncwarp();
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int j = 0; j < NJ; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int col = 8 * j + 2 * tg + e;
                    double2 cin = make_double2(0.0, 0.0);
                    if (valid[2 * h] && col < m) cin = *reinterpret_cast<const double2*>(Cin + rows[2 * h] + (int64_t)col * ldc);
                    const int rl = 16 * h + 2 * g;
                    Es[rl * lde + col] = (valid[2 * h] && col < m) ? cin.x - acc[2 * h][j][e] : 0.0;
                    Es[(rl + 1) * lde + col] = (valid[2 * h + 1] && col < m) ? cin.y - acc[2 * h + 1][j][e] : 0.0;
                }
        __syncwarp();
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            double f[NJ];
#pragma unroll
            for (int j = 0; j < NJ; ++j) f[j] = Es[(4 * ks + tg) * lde + 8 * j + g];
            int t = 0;
#pragma unroll
            for (int mt = 0; mt < NJ; ++mt)
#pragma unroll
                for (int nt = mt; nt < NJ; ++nt, ++t) dmma(gacc[t][0], gacc[t][1], f[mt], f[nt]);
        }
    }
    // CTA partial: warps summed in a fixed order through shared memory, both triangles written
    __syncthreads();
    double* red = Es_all;                                         // [4][NT2 * 2][32]
    {
#pragma unroll
        for (int t = 0; t < NT2; ++t) { red[((size_t)warp * NT2 * 2 + 2 * t) * 32 + lane] = gacc[t][0]; red[((size_t)warp * NT2 * 2 + 2 * t + 1) * 32 + lane] = gacc[t][1]; }
    }
    __syncthreads();
    if (warp == 0) {
        double* P = partial + (int64_t)blockIdx.x * m * m;
        int t = 0;
#pragma unroll
        for (int mt = 0; mt < NJ; ++mt)
#pragma unroll
            for (int nt = mt; nt < NJ; ++nt, ++t)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    double v = 0.0;
                    for (int w2 = 0; w2 < RG_THREADS / 32; ++w2) v += red[((size_t)w2 * NT2 * 2 + 2 * t + e) * 32 + lane];
                    const int a = 8 * mt + g, b = 8 * nt + 2 * tg + e;
                    if (a < m && b < m) {
                        if (mt != nt || a <= b) P[a + (int64_t)b * m] = v;
                        if (mt != nt || a < b) P[b + (int64_t)a * m] = v;
                    }
                }
    }
    slab_reduce_tail(partial, m, m, o, &s_role);
}

}  // namespace

// Dynamic shared-memory opt-in of every contraction kernel: once per context (lrp_create).
template <typename F> static int mma_optin(lrp_ctx* ctx, F fn) {
    cudaFuncAttributes fa;
    LRP_CUDA(ctx, cudaFuncGetAttributes(&fa, fn));
    const int v = ctx->smem_optin - (int)fa.sharedSizeBytes;
    if (v > 48 * 1024) LRP_CUDA(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, v));
    return LRP_OK;
}
int tall_mma_init(lrp_ctx* ctx) {
    LRP_TRY(mma_optin(ctx, tall_gemm_mma_kernel<2, true>)); LRP_TRY(mma_optin(ctx, tall_gemm_mma_kernel<2, false>));
    LRP_TRY(mma_optin(ctx, tall_gemm_mma_kernel<4, true>)); LRP_TRY(mma_optin(ctx, tall_gemm_mma_kernel<4, false>));
    LRP_TRY(mma_optin(ctx, tall_gemm_mma_kernel<5, true>)); LRP_TRY(mma_optin(ctx, tall_gemm_mma_kernel<5, false>));
    LRP_TRY(mma_optin(ctx, tall_gemm_mma_kernel<6, true>)); LRP_TRY(mma_optin(ctx, tall_gemm_mma_kernel<6, false>));
    LRP_TRY(mma_optin(ctx, tall_resid_gram_kernel<1>)); LRP_TRY(mma_optin(ctx, tall_resid_gram_kernel<2>));
    LRP_TRY(mma_optin(ctx, tall_resid_gram_kernel<3>)); LRP_TRY(mma_optin(ctx, tall_resid_gram_kernel<4>));
    LRP_TRY(mma_optin(ctx, tall_resid_gram_kernel<5>)); LRP_TRY(mma_optin(ctx, tall_resid_gram_kernel<6>));
    LRP_TRY(mma_optin(ctx, tall_resid_gram_kernel<7>)); LRP_TRY(mma_optin(ctx, tall_resid_gram_kernel<8>));
    return LRP_OK;
}

int tall_gemm(lrp_ctx* ctx, const TallGemmArgs& p) {
    if (p.n <= 0 || p.m <= 0) return LRP_OK;
    // column tiles of 8 nj: every tile pass re-reads A, so 33..48 columns (the rebuild U = Q Uc, the first sweep's
    // fibers) go in ONE pass of nj = 5 / 6 instead of two of nj = 4
    const int tiles = (p.m + 7) / 8;
    const int nj = p.m <= 16 ? 2 : (tiles == 5 ? 5 : (tiles == 6 ? 6 : 4));
    size_t smem = sizeof(double) * ((size_t)(8 * nj) * mg_kp(p.k > 0 ? p.k : 1) + 8 * nj);
    auto al16 = [](const void* q) { return ((uintptr_t)q & 15u) == 0; };
    const bool vec = (p.lda % 2 == 0) && (p.ldo % 2 == 0) && al16(p.A) && al16(p.Out) &&
                     (p.mode != TG_SUBTRACT || ((p.ldc % 2 == 0) && al16(p.Cin)));
    void (*kern)(TallGemmArgs) = nj == 2 ? (vec ? tall_gemm_mma_kernel<2, true> : tall_gemm_mma_kernel<2, false>)
                               : nj == 5 ? (vec ? tall_gemm_mma_kernel<5, true> : tall_gemm_mma_kernel<5, false>)
                               : nj == 6 ? (vec ? tall_gemm_mma_kernel<6, true> : tall_gemm_mma_kernel<6, false>)
                                         : (vec ? tall_gemm_mma_kernel<4, true> : tall_gemm_mma_kernel<4, false>);
    if (smem > (size_t)ctx->smem_optin) return LRP_ERR_BADARG;       // opt-in set once by tall_mma_init
    int64_t grid = (p.n + MG_THREADS - 1) / MG_THREADS;
    const int64_t resident = (int64_t)lrp_sm_count(ctx) * (nj == 2 ? 5 : (nj <= 4 ? 4 : 3));   // persistent over row slabs (B staged once per column tile per CTA):
    if (grid > resident) grid = resident;            // exactly one resident wave, so that the slabs are balanced
    if (p.cond) LRP_PROF(ctx, K_COND, 0, 0);             // device-side conditional launch: normally a no-op, no work accounted
    else LRP_PROF(ctx, p.mode == TG_SAMPLE ? K_GEMM_SAMPLE : (p.mode == TG_SUBTRACT ? K_GEMM_SUBTRACT : K_GEMM_PLAIN),
                  8.0 * p.n * (p.k + p.m + (p.mode == TG_SUBTRACT ? p.m : 0)), 2.0 * p.n * p.k * p.m);
    kern<<<(unsigned)grid, MG_THREADS, smem, ctx->stream>>>(p);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

static int tall_gemm_t_ntc(int k, int m) {       // tiles per CTA: 1, 2, 4 or 8 (the 8 warps split rows when fewer)
    int nt = ((k + 15) / 16) * ((m + 15) / 16);
    return nt >= 8 ? 8 : (nt >= 4 ? 4 : (nt >= 2 ? 2 : 1));
}
static int tall_gemm_t_nblk(const lrp_ctx* ctx, int64_t n, int k, int m) {
    (void)k; (void)m;
    int64_t want = (int64_t)lrp_sm_count(ctx) * 3;     // SMs x 3 resident CTAs (one wave); without a ctx (workspace sizing on the host) the upper bound LRP_SM_UPPER
    int64_t by_rows = (n + 511) / 512;
    int64_t nb = want < by_rows ? want : by_rows;
    return (int)(nb < 1 ? 1 : nb);
}

size_t tall_gemm_t_ws_doubles(const lrp_ctx* ctx, int64_t n, int k, int m) {
    (void)ctx;                                          // sized for the upper bound of the SM count: no device query
    return ((size_t)tall_gemm_t_nblk(nullptr, n, k, m) + GT_MAXGRP) * k * m;      // slab partials + group partials
}

int tall_gemm_t(lrp_ctx* ctx, int64_t n, const double* A, int64_t lda, int k, const double* B, int64_t ldb, int m,
                double* S, int64_t lds, int accumulate, double* partial_ws, double* Sadd, int64_t ldadd, const int* cond) {
    if (k <= 0 || m <= 0) return LRP_OK;
    int nblk = tall_gemm_t_nblk(ctx, n, k, m);
    const int nblk_max = tall_gemm_t_nblk(nullptr, n, k, m);
    const int ntc = tall_gemm_t_ntc(k, m);
    int64_t rows_per = (n + nblk - 1) / nblk;
    rows_per = (rows_per + 15) / 16 * 16;
    nblk = (int)((n + rows_per - 1) / rows_per);
    const int na = (k + 15) / 16, nb = (m + 15) / 16;
    dim3 grid(nblk, (na * nb + ntc - 1) / ntc);
    if ((nblk + GT_GROUP - 1) / GT_GROUP > GT_MAXGRP) return LRP_ERR_BADARG;
    GemmTOut o{};
    o.S = S; o.lds = lds; o.accumulate = accumulate; o.Sadd = Sadd; o.ldadd = ldadd; o.cond = cond;
    o.gpartial = partial_ws + (size_t)nblk_max * k * m;
    // one counter set per library stream: launches on a stream are ordered, the counters are back at zero when a launch ends
    const int slot = ctx->stream == ctx->aux ? 1 : (ctx->stream == ctx->aux2 ? 2 : 0);
    o.counters = ctx->d_counters + slot * (GT_MAXGRP + 1);
    if (cond) LRP_PROF(ctx, K_COND, 0, 0); else LRP_PROF(ctx, K_GEMM_T, 8.0 * n * (k + m), 2.0 * n * k * m);
    const bool vec = (lda % 2 == 0) && (ldb % 2 == 0) && (((uintptr_t)A | (uintptr_t)B) & 15u) == 0;
    if (vec) tall_gemm_t_mma_kernel<true><<<grid, MT_THREADS, 0, ctx->stream>>>(A, lda, k, B, ldb, m, n, rows_per, partial_ws, na, nb, ntc, o);
    else tall_gemm_t_mma_kernel<false><<<grid, MT_THREADS, 0, ctx->stream>>>(A, lda, k, B, ldb, m, n, rows_per, partial_ws, na, nb, ntc, o);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}

// G (m x m, ld ldg) = E^T E, E = Cin - A B (B: k x m device, ld ldb), without writing E.  Returns 1 when the shape or
// the alignment is outside the fused kernel's range (m > 64, odd leading dimensions): the caller then takes the
// update + Gram sweeps.  partial_ws: tall_gemm_t_ws_doubles(ctx, n, m, m) doubles.
int tall_resid_gram(lrp_ctx* ctx, int64_t n, const double* A, int64_t lda, int k, const double* B, int64_t ldb,
                    const double* Cin, int64_t ldc, int m, double* G, int64_t ldg, double* partial_ws) {
    if (k <= 0 || m <= 0) return 1;
    if (ctx->flags & LRP_FLAG_NO_FUSED_RHO) return 1;              // lrp_solve_opts.flags: force the two-sweep path
    const int NJ = (m + 7) / 8;
    const bool vec = (lda % 2 == 0) && (ldc % 2 == 0) && ((((uintptr_t)A) | ((uintptr_t)Cin)) & 15u) == 0;
    if (NJ > 8 || !vec) return 1;
    int nblk = tall_gemm_t_nblk(ctx, n, m, m);                     // same partial geometry as tall_gemm_t
    const int nblk_max = tall_gemm_t_nblk(nullptr, n, m, m);
    if (nblk > ctx->sm_count * (NJ <= 5 ? 3 : 2)) nblk = ctx->sm_count * (NJ <= 5 ? 3 : 2);   // one resident wave of the persistent CTAs
    const int64_t nslab = (n + RG_THREADS - 1) / RG_THREADS;
    if (nblk > nslab) nblk = (int)nslab;
    const size_t es = (size_t)4 * 32 * rg_lde(8 * NJ), rd = (size_t)4 * NJ * (NJ + 1) * 32;
    const size_t smem = sizeof(double) * ((size_t)8 * NJ * mg_kp(k) + (es > rd ? es : rd));
    if (smem > (size_t)ctx->smem_optin) return 1;
    GemmTOut o{};
    o.S = G; o.lds = ldg; o.accumulate = 0; o.Sadd = nullptr; o.ldadd = 0;
    o.gpartial = partial_ws + (size_t)nblk_max * m * m;
    const int slot = ctx->stream == ctx->aux ? 1 : (ctx->stream == ctx->aux2 ? 2 : 0);
    o.counters = ctx->d_counters + slot * (GT_MAXGRP + 1);
    void (*kern)(int64_t, const double*, int64_t, int, const double*, int64_t, const double*, int64_t, int, double*, GemmTOut) = nullptr;
    switch (NJ) {
        case 1: kern = tall_resid_gram_kernel<1>; break; case 2: kern = tall_resid_gram_kernel<2>; break;
        case 3: kern = tall_resid_gram_kernel<3>; break; case 4: kern = tall_resid_gram_kernel<4>; break;
        case 5: kern = tall_resid_gram_kernel<5>; break; case 6: kern = tall_resid_gram_kernel<6>; break;
        case 7: kern = tall_resid_gram_kernel<7>; break; default: kern = tall_resid_gram_kernel<8>; break;
    }
    LRP_PROF(ctx, K_RESID_GRAM, 8.0 * n * (k + m), 2.0 * n * m * (k + m));
    kern<<<nblk, RG_THREADS, smem, ctx->stream>>>(n, A, lda, k, B, ldb, Cin, ldc, m, partial_ws, o);
    LRP_LAUNCHED(ctx);
    return LRP_OK;
}
