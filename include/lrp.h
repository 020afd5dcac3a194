/* lrp.h -- C ABI of liblrp: the B200 (sm_100a) hot path of the Cross-DEIM low-rank Poisson solver
 * of arxiv/paper_2607_06021 (citations: `PAPER.md:<line>` + section / equation / algorithm).
 *
 * Problem (eq. (2), 194-196 eq. (3)): 5-point Dirichlet Poisson on an n x n interior grid,
 *     T W + W T^T = h^2 F,   T = tridiag(-1, 2, -1),   h = 1/(n+1),
 * with the right-hand side held as low-rank factors F = UF diag(SF) VF^T.  The factors are
 * taken to sine space by batched DST-I along each dimension, the spectral solution
 *     G(i,j) = (Uh diag(S) Vh^T)(i,j) / (d_i + d_j),  d_k = lambda_k / h^2 = 4 (n+1)^2 sin^2(pi k / (2(n+1)))
 * (eq. (4); lambda_k of PAPER.md:200 evaluated as 4 sin^2(theta/2), reading Q1) is
 * sampled only on index sets I, J chosen by leverage scores (Alg. 3), rebuilt into
 * factors by the stabilised cross approximation scross (Alg. 1), iterated by Cross-DEIM
 * (Alg. 4) and brought back by a final batched DST-I.
 *
 * Conventions
 *   - every `d_*` pointer is a DEVICE pointer to memory the CALLER owns; `h_*` pointers are HOST pointers.
 *   - fp64 throughout.  "tall" matrices are column-major with an explicit leading dimension ld >= n
 *     (each factor column contiguous).  Diagonal factors S are stored as vectors.
 *   - indices are 0-based int32_t (grid point i <-> 1-based frequency k = i + 1); sizes are int64_t/int32_t.
 *   - the library never allocates device memory for data: scratch comes from the workspace the caller
 *     hands to lrp_set_workspace (sized by the lrp_*_workspace_bytes functions).  Pointers must be
 *     8-byte aligned; the workspace must be 256-byte aligned.  (The ctx itself owns 780 bytes of device memory,
 *     the arrival counters of its in-kernel reductions, and 8 KB of pinned host memory.)
 *   - every call enqueues on the ctx's stream.  lrp_dst1_batched, lrp_sample_fibers are asynchronous;
 *     lrp_leverage_select, lrp_scross and lrp_cross_deim_solve synchronise the stream internally where
 *     their control flow needs device results (documented per function) and are complete on return
 *     only where stated.
 *   - return value: 0 = LRP_OK, negative = error, positive = warning (outputs valid).
 *     No exceptions, no globals, no environment variables, no CPU fallback: without a CUDA device every compute call fails.
 *   - n: n + 1 a power of two up to 2^25 (the fast paths), or any n with n + 1 <= 2^23 (Bluestein's chirp-z form of the
 *     DST-I, 8-16x the work; the paper's own grids n = 2^10..2^18, are of this kind).
 */
#ifndef LRP_H_
#define LRP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LRP_OK                  0
#define LRP_ERR_BADARG         -1   /* null / misaligned pointer, ld < n, set larger than the cap, duplicate or out-of-range index */
#define LRP_ERR_UNSUPPORTED_N  -2   /* n out of range (see above) */
#define LRP_ERR_WORKSPACE      -3   /* workspace missing or too small */
#define LRP_ERR_CUDA           -4   /* a CUDA call failed; see lrp_last_cuda_error */
#define LRP_ERR_STATIC_LIMIT   -5   /* lrp_topk_static: n or num_select beyond the fixed capacity of its built-in scratch */
#define LRP_WARN_NOCONV         1   /* Cross-DEIM reached max_sweeps (or r* > max_rank): outputs valid, tolerance not certified */

#define LRP_MAX_SWEEPS_INFO    32   /* per-sweep arrays in lrp_solve_info hold this many sweeps */

typedef struct lrp_ctx lrp_ctx;

/* Create a context bound to CUDA device `device` and to `cuda_stream` (a cudaStream_t; NULL = the
 * legacy default stream).  The stream is borrowed, not owned.  Fails with LRP_ERR_CUDA if there is no device. */
int lrp_create(lrp_ctx** out, int device, void* cuda_stream);
int lrp_destroy(lrp_ctx* ctx);
const char* lrp_strerror(int code);
/* cudaError_t (as int) of the last failing CUDA call seen by this ctx, 0 if none. */
int lrp_last_cuda_error(const lrp_ctx* ctx);
/* Number of kernel launches this ctx has enqueued since creation (bench.py's `gpu_launches`). */
int64_t lrp_launch_count(const lrp_ctx* ctx);

/* Per-kernel profile (used by bench.py's roofline): with profiling enabled every kernel launch is bracketed by CUDA
 * events on the ctx's stream (adds a few microseconds per launch: never enabled inside a timed region).
 * lrp_profile_get synchronises the stream and returns, for kernel class i < lrp_profile_count(): its name (static
 * string), launch count, summed event time in ms (0 unless profiling was on), and the summed ALGORITHMIC bytes and
 * flops of those launches.  lrp_profile_reset zeroes the counters. */
int lrp_profile_enable(lrp_ctx* ctx, int on);
/* on = 2 records the same events WITHOUT serialising the library's streams; lrp_profile_timeline then writes one
 * line per launch since the last reset (kernel class, start and end in ms after the first launch) to a CSV file: the
 * timeline of the real multi-stream run (per-class ms of overlapping kernels are then not additive). */
int lrp_profile_timeline(lrp_ctx* ctx, const char* path);
int lrp_profile_reset(lrp_ctx* ctx);
int lrp_profile_count(void);
int lrp_profile_get(lrp_ctx* ctx, int i, const char** name, int64_t* count, double* ms, double* bytes, double* flops);

/* Measured fp64 throughput of the device in TFLOP/s: plain DFMA and the fp64 tensor pipe (DMMA, mma.sync m8n8k4) from
 * register-only loops; a few milliseconds, synchronises.  bench.py uses the larger one as the peak of its fp64 ("alu")
 * rooflines (the fp64 peaks are to be measured on the box).  Not on the solve path. */
int lrp_fp64_peak(lrp_ctx* ctx, double* dfma_tflops, double* dmma_tflops);

/* Workspace sizes in bytes (host-side arithmetic only; safe to call without a GPU).
 *   lrp_workspace_bytes        : everything lrp_cross_deim_solve needs for rank-rF input, K_cap = 2 (max_rank + oversample)
 *                                (reading Q10); 0 when the arguments are invalid, e.g. rF + oversample + 1 > K_cap.
 *   lrp_dst1_workspace_bytes   : lrp_dst1_batched (0 for n + 1 = 2^p <= 16384, the single-pass shared-memory regime).
 *   lrp_leverage_workspace_bytes, lrp_scross_workspace_bytes : the standalone calls. */
size_t lrp_workspace_bytes(int64_t n, int32_t rF, int32_t max_rank, int32_t oversample);
size_t lrp_dst1_workspace_bytes(int64_t n, int32_t batch);
size_t lrp_leverage_workspace_bytes(int64_t n, int32_t k);
size_t lrp_scross_workspace_bytes(int64_t n, int32_t k, int32_t l);
/* Hand the ctx a device scratch buffer (caller-owned, must outlive the calls that use it). */
int lrp_set_workspace(lrp_ctx* ctx, void* d_ws, size_t bytes);

/* Batched DST-I:
 *     out(k, b) = scale * sum_{j=1..n} in(j, b) sin(j k pi / (n+1)),   k = 1..n,  b = 0..batch-1,
 * 1-based j,k stored 0-based.  scale = 1: unnormalised (applied twice = (n+1)/2 * identity);
 * scale = sqrt(2/(n+1)): the symmetric orthogonal Z of PAPER.md:198-200 (twice = identity).
 * in/out: tall n x batch, column b at d_in + b*ld_in.  d_in == d_out (same ld) is allowed; partial overlap is not.
 * Each column is transformed independently along its own (contiguous) dimension: no transpose.
 * Asynchronous.  Errors: BADARG, UNSUPPORTED_N, WORKSPACE (n > 16383 or n + 1 not a power of two: lrp_dst1_workspace_bytes), CUDA. */
int lrp_dst1_batched(lrp_ctx* ctx, int64_t n, int32_t batch,
                     const double* d_in, int64_t ld_in, double* d_out, int64_t ld_out, double scale);

/* Spectral fibers of G(i,j) = (Uh diag(S) Vh^T)(i,j) / (d_i + d_j)  (eq. (4); Alg. 1
 * line 3), O(r) per entry, never forming the n^2 matrix:
 *     d_C  (n x nJ, ld ldc): column c = G(:, J[c]);      d_Rt (n x nI, ld ldr): column c = G(I[c], :)^T.
 * Uh, Vh: tall n x r spectral factors; d_S: r values.  d_I / d_J: device index lists (0-based, in [0,n)).
 * Either output (with its index list) may be NULL.  Asynchronous.  Errors: BADARG, CUDA. */
int lrp_sample_fibers(lrp_ctx* ctx, int64_t n, int32_t r,
                      const double* d_Uh, int64_t ldu, const double* d_S, const double* d_Vh, int64_t ldv,
                      const int32_t* d_I, int32_t nI, const int32_t* d_J, int32_t nJ,
                      double* d_C, int64_t ldc, double* d_Rt, int64_t ldr);

/* Leverage-score selection (Alg. 3, deterministic top-k form, reading Q5):
 * thin QR A = Q R of the tall n x k block, scores[i] = ||Q(i,:)||^2 over the columns with
 * |R_cc| >= 1e-13 max|R_cc|, and d_idx_out = the num_select (<= n, <= 4096) largest, ordered by
 * (score descending, index ascending).  d_scores (n) may be NULL.  assume_orthonormal = 1 skips the QR
 * (A is used as Q).  A is not modified.  Complete on return (synchronises).  Errors: BADARG, WORKSPACE, CUDA. */
int lrp_leverage_select(lrp_ctx* ctx, int64_t n, int32_t k, const double* d_A, int64_t lda,
                        int32_t num_select, int assume_orthonormal,
                        int32_t* d_idx_out, double* d_scores);

/* Stabilised cross approximation, Algorithm 1 on already sampled fibers, square-grid case:
 * C = G(:,J) is n x k (k = #J), Rt = G(I,:)^T is n x l (l = #I).  Thin QR C = Q R_C, Rt = Z R_R; the tall
 * least-squares systems of lines 5-14 are solved by the SVD pseudo-inverse (relative cut 1e-13) folded to
 * the k x l core M (k <= l: M = Q(I,:)^+ R_R^T;  k > l: M = (Z(J,:)^+ R_C^T)^T); M = Uc diag(S) Vc^T;
 * numerical rank = #{S_c > 1e-14 S_1} (>= 1);  U = Q Uc, V = Z Vc.
 * Outputs: d_U (n x rank), d_S (min(k,l) values, the first *rank_out are the kept ones), d_V (n x rank),
 * d_rC (k) = |diag R_C|, d_rR (l) = |diag R_R| (Alg. 1 line 16), *h_rank_out, *h_smin_full_out (HOST
 * scalars; smin_full = smallest singular value of the untruncated core, reading Q11).
 * d_U / d_V must have room for min(k,l) columns.  C and Rt are read-only.  Complete on return.
 * Errors: BADARG (k or l < 1 or > 1024, ld < n), WORKSPACE, CUDA. */
int lrp_scross(lrp_ctx* ctx, int64_t n, const double* d_C, int64_t ldc, int32_t k,
               const double* d_Rt, int64_t ldr, int32_t l,
               const int32_t* d_I, const int32_t* d_J,
               double* d_U, int64_t ldu, double* d_S, double* d_V, int64_t ldv,
               double* d_rC, double* d_rR, int32_t* h_rank_out, double* h_smin_full_out);

typedef struct lrp_solve_opts {
    double  tol;               /* epsilon of Alg. 4 */
    int32_t max_rank;          /* r_max */
    int32_t oversample;        /* extra leverage indices per sweep (config 1: 8) */
    int32_t max_sweeps;        /* at most this many sweeps (reading Q16) */
    int32_t tol_mode;          /* 0: relative to ||S_k||_2 (default, reading Q15); 1: absolute, as printed in the paper */
    const int32_t* h_safeguard;/* HOST list of pre-drawn random indices (Alg. 4 lines 7-12): randomness is input data */
    int32_t n_safeguard;
    const double* d_U0;        /* optional warm start / initial guess for the selection (n x r0), may be NULL -> spectral RHS factors */
    const double* d_V0;
    int64_t ld0;
    int32_t r0;
    /* replay (test hook): take the index sets and prune masks of every sweep from these HOST arrays instead of
     * deciding them; replay_sweeps > 0 enables it.  Sets are concatenated sweep after sweep. */
    int32_t replay_sweeps;
    const int32_t* h_replay_nI;     /* [replay_sweeps] */
    const int32_t* h_replay_nJ;     /* [replay_sweeps] */
    const int32_t* h_replay_I;      /* concatenated I_k */
    const int32_t* h_replay_J;      /* concatenated J_k */
    const uint8_t* h_replay_keepI;  /* concatenated prune masks (1 = survives), may be NULL -> decide */
    const uint8_t* h_replay_keepJ;
    int32_t replay_final_rank;      /* > 0: use this final rank */
    int32_t flags;                  /* bit mask of LRP_FLAG_* below; 0 = default path */
    int32_t selection;              /* LRP_SELECT_TOPK (default), LRP_SELECT_BERNOULLI, LRP_SELECT_QDEIM, LRP_SELECT_DEIM */
    uint64_t ls_seed;               /* LRP_SELECT_BERNOULLI: seed of the counter-based uniforms */
    double  ls_c;                   /* LRP_SELECT_BERNOULLI: the constant c of Alg. 3 line 4; <= 0: cols + oversample */
} lrp_solve_opts;

/* lrp_solve_opts.selection: how the index sets are enriched each sweep (Alg. 4 line 5)
 *   TOPK      leverage scores, the (cols + oversample) largest (deterministic form of Alg. 3, reading Q5)
 *   BERNOULLI leverage scores as printed (Alg. 3 lines 4-5): keep i with probability
 *             min{1, c pi_i}, pi_i = l_i / cols; u_i from a counter-based generator keyed by (ls_seed, sweep, side, i)
 *   QDEIM     column-pivoted QR of U^T (Alg. 2 lines 7-10): cols indices
 *   DEIM      pivoted LU of U (Alg. 2 lines 3-6): cols indices */
#define LRP_SELECT_TOPK       0
#define LRP_SELECT_BERNOULLI  1
#define LRP_SELECT_QDEIM      2
#define LRP_SELECT_DEIM       3

/* lrp_solve_opts.flags: switch one of the driver's shortcuts off (comparison runs of the tests; results agree to rounding) */
#define LRP_FLAG_NO_QR_REUSE    1   /* factor every fiber block from scratch (reading R4 off) */
#define LRP_FLAG_NO_NESTED_RHO  2   /* rho always from the tall iterates (reading R5 off) */
#define LRP_FLAG_NO_FUSED_RHO   4   /* rho's residual Gram matrix by an update sweep + a Gram sweep instead of the fused kernel */
#define LRP_FLAG_NO_CHOLQR_LEVERAGE 8 /* leverage scores of the initial guess always through the Householder QR (reading R8 off) */
#define LRP_FLAG_NO_PRIORITY_STREAMS 16 /* TSQR tree levels on the job's own stream instead of a high-priority one (scheduling only) */

typedef struct lrp_solve_info {
    int32_t rank, sweeps, converged;
    double  rho, indicator, eta1, eta2, snorm, smin_full;
    int32_t nI[LRP_MAX_SWEEPS_INFO], nJ[LRP_MAX_SWEEPS_INFO], rank_per_sweep[LRP_MAX_SWEEPS_INFO];
    double  rho_per_sweep[LRP_MAX_SWEEPS_INFO], ind_per_sweep[LRP_MAX_SWEEPS_INFO];
    float   ms_dst_fwd, ms_select, ms_sample, ms_qr, ms_core, ms_rebuild, ms_stop, ms_dst_inv, ms_total;
    int64_t launches;
} lrp_solve_info;

/* Low-rank Poisson solve by Cross-DEIM (Alg. 4):
 * solves T W + W T^T = h^2 F with F = UF diag(SF) VF^T given in PHYSICAL space (columns need not be
 * orthonormal) and writes W ~= UW diag(SW) VW^T with rank info->rank <= max_rank.
 * d_UW, d_VW: tall with ld >= n and room for max_rank columns; d_SW: max_rank values.
 * Optional trace outputs (HOST, may be NULL): h_trace_I / h_trace_J receive the concatenated I_k / J_k (before
 * pruning) of every sweep (capacity LRP_MAX_SWEEPS_INFO * K_cap each), h_trace_keepI / h_trace_keepJ the
 * prune masks; the per-sweep counts are info->nI / nJ.
 * Optional spectral outputs (DEVICE, may be NULL): d_Uhat / d_Vhat (n x K_cap, ld = ld_hat) and d_Shat
 * (K_cap) receive the last spectral iterate before the final truncation (info->rank_per_sweep[sweeps-1] columns).
 * Between sweeps the fibers of surviving indices are not resampled: the leading columns of a fiber block that repeat
 * the previous block keep their Q and R factors, and when the previous index lists are prefixes of the current ones
 * rho (Alg. 4 line 24) is evaluated from the small core factors (readings R4, R5;
 * opts->flags LRP_FLAG_NO_QR_REUSE / LRP_FLAG_NO_NESTED_RHO switch either off for comparison).
 * Index lists are cut to K_cap = 2 (max_rank + oversample) entries (reading Q10); rF + oversample + 1 > K_cap (the first
 * selection would not fit) is LRP_ERR_BADARG.
 * Synchronous: complete on return.  Returns LRP_WARN_NOCONV (info->converged = 0, outputs valid) when the stop test never
 * passed within max_sweeps or when r* > max_rank (Alg. 4 line 31: the truncated result misses the tolerance). */
int lrp_cross_deim_solve(lrp_ctx* ctx, int64_t n, int32_t rF,
                         const double* d_UF, int64_t ldu, const double* d_SF, const double* d_VF, int64_t ldv,
                         const lrp_solve_opts* opts,
                         double* d_UW, int64_t lduw, double* d_SW, double* d_VW, int64_t ldvw,
                         lrp_solve_info* info,
                         int32_t* h_trace_I, int32_t* h_trace_J, uint8_t* h_trace_keepI, uint8_t* h_trace_keepJ,
                         double* d_Uhat, double* d_Shat, double* d_Vhat, int64_t ld_hat);

/* The same solve for a batch of `nprob` INDEPENDENT problems whose factors live in HOST memory (the end-to-end form:
 * section 3.2, applied to problem after problem; independent problems need no exchange).
 * Problem p: h_UF[p], h_VF[p] (n x rF, ld = ldu / ldv >= n, column-major), h_SF[p] (rF); results h_UW[p], h_VW[p]
 * (room for max_rank columns, ld = lduw / ldvw >= n; the leading info[p].rank columns are written), h_SW[p] (max_rank
 * values of room), info[p].  All problems share n, rF and *opts (opts->d_U0 / d_V0, if set, are DEVICE pointers as usual).
 * The call owns the copies.  A LANE solves its problems one after the other through two staging slots carved from the
 * workspace behind the solve's own, with the host->device copy of its next problem and the device->host copy of its
 * previous one on two library-owned copy streams while the current one is solved.  With a workspace of
 * lrp_solve_host_workspace_bytes(..., 2) and nprob >= 2 there are TWO lanes (even / odd problems; the second on a
 * library-owned context and stream, driven by a worker thread that lives for the call): two solves in flight fill the
 * SMs that one leaves idle.  With lrp_solve_host_workspace_bytes(..., 1) there is one lane.  Results do not depend on the
 * number of lanes.  The overlap needs PINNED (page-locked) host buffers; pageable ones give the same results with the
 * copies serialised.  Output pointers may repeat between problems p and q only if p - q is a multiple of 2 and the
 * earlier result is no longer needed (downloads of one lane are ordered).
 * Synchronous: every result is in host memory on return.  Returns the first error of a lane (negative; that lane's later
 * problems are then not run) or else the largest warning code over the batch (LRP_WARN_NOCONV: see info[p].converged). */
#define LRP_HOST_LANES_MAX 2
size_t lrp_solve_host_workspace_bytes(int64_t n, int32_t rF, int32_t max_rank, int32_t oversample, int32_t lanes);
int lrp_cross_deim_solve_host(lrp_ctx* ctx, int64_t n, int32_t rF, int32_t nprob,
                              const double* const* h_UF, int64_t ldu, const double* const* h_SF,
                              const double* const* h_VF, int64_t ldv,
                              const lrp_solve_opts* opts,
                              double* const* h_UW, int64_t lduw, double* const* h_SW,
                              double* const* h_VW, int64_t ldvw,
                              lrp_solve_info* info);

/* The same for problems whose factors are already on the DEVICE: d_UF, d_SF, d_VF, d_UW, d_SW, d_VW are HOST arrays of
 * nprob DEVICE pointers (layouts as in lrp_cross_deim_solve; outputs of different problems must not overlap).  With a
 * workspace of lrp_solve_batch_workspace_bytes(..., 2) and nprob >= 2 the even and the odd problems are solved by two
 * lanes at once, else one after the other; results do not depend on it.  Synchronous; return value as above. */
size_t lrp_solve_batch_workspace_bytes(int64_t n, int32_t rF, int32_t max_rank, int32_t oversample, int32_t lanes);
int lrp_cross_deim_solve_batch(lrp_ctx* ctx, int64_t n, int32_t rF, int32_t nprob,
                               const double* const* d_UF, int64_t ldu, const double* const* d_SF,
                               const double* const* d_VF, int64_t ldv,
                               const lrp_solve_opts* opts,
                               double* const* d_UW, int64_t lduw, double* const* d_SW,
                               double* const* d_VW, int64_t ldvw,
                               lrp_solve_info* info);

/* Generic function-handle Cross-DEIM (Alg. 4; "G(i,j) as a function handle") on the
 * paper's closed-form test matrices, eq. (6), PAPER.md:264-267 (0-based i, j; square n x n, any n >= K_cap):
 *     LRP_G_HILBERT:  H(i,j) = 1 / (1 + i + j)                        (rapid singular value decay)
 *     LRP_G_KMATRIX:  K(i,j) = (|x_i + y_j| / 2)^5,  x_i = -1 + 2 i/(n-1),  y_j = -1 + 2 j/(n-1)   (C^4, slow decay)
 * Same sweep loop, selection, scross, prune, stop test and final truncation as lrp_cross_deim_solve; only the fiber
 * sampler differs and there is no transform before or after.  The initial guess of Alg. 4 is
 * REQUIRED here: opts->d_U0, d_V0 (n x r0, any full-rank columns; used for the first selection only).
 * Outputs: d_U, d_V (n x max_rank, ld >= n), d_S (max_rank): G ~= U diag(S) V^T with rank info->rank.  Trace and
 * last-iterate outputs as for lrp_cross_deim_solve.  Workspace: lrp_matrix_workspace_bytes(n, r0, max_rank, oversample).
 * Synchronous.  Errors / warning as lrp_cross_deim_solve. */
#define LRP_G_POISSON  0
#define LRP_G_HILBERT  1
#define LRP_G_KMATRIX  2
size_t lrp_matrix_workspace_bytes(int64_t n, int32_t r0, int32_t max_rank, int32_t oversample);
int lrp_cross_deim_matrix(lrp_ctx* ctx, int32_t kind, int64_t n, const lrp_solve_opts* opts,
                          double* d_U, int64_t ldu, double* d_S, double* d_V, int64_t ldv,
                          lrp_solve_info* info,
                          int32_t* h_trace_I, int32_t* h_trace_J, uint8_t* h_trace_keepI, uint8_t* h_trace_keepJ,
                          double* d_Uhat, double* d_Shat, double* d_Vhat, int64_t ld_hat);
/* Fibers of a test matrix (the sampler behind lrp_cross_deim_matrix; Alg. 1 line 3):
 *     d_C (n x nJ): column c = G(:, J[c]);   d_Rt (n x nI): column c = G(I[c], :)^T.   Either may be NULL.  Asynchronous. */
int lrp_sample_matrix(lrp_ctx* ctx, int32_t kind, int64_t n, const int32_t* d_I, int32_t nI, const int32_t* d_J, int32_t nJ,
                      double* d_C, int64_t ldc, double* d_Rt, int64_t ldr);

/* Dense full-rank DST solver of section 3.1 (eq. (4)): W = Z ((Z F Z) ./ (d_i + d_j)) Z for a
 * dense n x n right-hand side F (column-major, ld >= n), O(n^2 log n) -- the baseline the low-rank method is measured
 * against, n <= 32768 (2 n^2 doubles of workspace + the transform's: lrp_dense_workspace_bytes).  d_W may alias d_F.
 * Asynchronous.  Errors: BADARG, UNSUPPORTED_N, WORKSPACE, CUDA. */
size_t lrp_dense_workspace_bytes(int64_t n);
int lrp_dense_poisson(lrp_ctx* ctx, int64_t n, const double* d_F, int64_t ldf, double* d_W, int64_t ldw);

/* Entries (U diag(S) V^T)(rows[t], cols[t]), t < count (X(i,j) = sum_k sigma_k u_k(i) v_k(j)):
 * the O(r) element access used to read a low-rank result without forming it.  All pointers device.  Asynchronous. */
int lrp_lowrank_entries(lrp_ctx* ctx, int64_t n, int32_t r, const double* d_U, int64_t ldu, const double* d_S,
                        const double* d_V, int64_t ldv, const int64_t* d_rows, const int64_t* d_cols,
                        int64_t count, double* d_out);

/* Allocation-free top-k (the index selection of Alg. 3 line 6, deterministic form, reading Q5) for
 * callers that cannot call cudaMalloc or own a workspace (CUDA graph capture, serving loops, harnesses that forbid it):
 *     d_idx_out[0..num_select) = the indices of the num_select largest d_scores[0..n), ordered by (score descending,
 *     index ascending) -- bit-identical to what lrp_leverage_select returns for the same scores.
 * No ctx and no workspace: the candidate buffers of the multi-level sort live in a 1.6 MB device array built into the
 * library (held by every GPU that loads it until the process exits).  Limits: n <= LRP_TOPK_STATIC_MAX_N,
 * num_select <= LRP_TOPK_STATIC_MAX_NUM, else LRP_ERR_STATIC_LIMIT.  The call allocates nothing and frees nothing.  The
 * FIRST call on a device looks up the array's device address (do it once outside a capture); the device that owns
 * `cuda_stream` (a cudaStream_t, NULL = legacy default stream) must be current.  d_scores (n doubles, 8-byte aligned) and
 * d_idx_out (num_select int32) are device pointers owned by the caller.  Asynchronous on `cuda_stream`.
 * All calls share the one array: calls that overlap on the GPU (different streams or host threads) race -- serialise them.
 * Errors: BADARG (null / misaligned pointer, n < 1, num_select < 0 or > n), STATIC_LIMIT, CUDA. */
#define LRP_TOPK_STATIC_MAX_N    4194304
#define LRP_TOPK_STATIC_MAX_NUM  256
int lrp_topk_static(void* cuda_stream, int64_t n, const double* d_scores, int32_t num_select, int32_t* d_idx_out);

#ifdef __cplusplus
}
#endif
#endif /* LRP_H_ */
