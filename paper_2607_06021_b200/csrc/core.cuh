// core.cuh -- one-CTA small dense kernels (core.cu) and index selection (select.cu)
#pragma once
#include "common.cuh"

struct CoreArgs {
    int k, l;                                   // k = #J (columns of C), l = #I (columns of Rt)
    const double* Q; int64_t ldq;               // n x k, orthonormal factor of C
    const double* Z; int64_t ldz;               // n x l, orthonormal factor of Rt
    const double* RC; int64_t ldrc;             // k x k
    const double* RR; int64_t ldrr;             // l x l
    const int32_t* I; const int32_t* J;         // device index lists
    double pinv_rcond, rank_rcond;
    double* Uc; double* S; double* Vc;          // k x p (ld k), p, l x p (ld l), p = min(k, l)
    double* rC; double* rR;                     // |diag R_C| (k), |diag R_R| (l)
    int32_t* scal_i; double* scal_d;            // [0] = numerical rank ; [0] = smin_full
    double* work; int32_t* iwork;               // core_work_doubles(k, l) doubles, max(k, l) ints
    int smem_doubles;                           // set by scross_core: dynamic shared memory available to the Jacobi sweeps
};
size_t core_work_doubles(int k, int l);
int scross_core(lrp_ctx* ctx, const CoreArgs& a);

struct EtaArgs {
    int r;
    const double* U; int64_t ldu; const int32_t* I; int nI;
    const double* V; int64_t ldv; const int32_t* J; int nJ;
    // optional factored form: U = QU CU (QU n x kU passed as U/ldu, CU kU x r), likewise V -- eta can then start from
    // the core's output, before the tall rebuild products exist
    const double* CU; int kU; int64_t ldcu; const double* CV; int kV; int64_t ldcv;
    double* eta;                                // [2] device: eta1, eta2
    double* work; size_t work_stride; int32_t* iwork; size_t iwork_stride;
    int smem_doubles;
};
size_t eta_work_doubles(int nmax, int r);
int eta_pair(lrp_ctx* ctx, const EtaArgs& a);

struct RhoArgs {
    int r, rp;                                  // ranks of the current and previous iterate
    const double* Sk; const double* Sp;
    const double* A; const double* B;           // r x rp (ld r): U_k^T U_{k-1}, V_k^T V_{k-1}
    const double* GU; const double* GV;         // rp x rp (ld rp): E_U^T E_U, E_V^T E_V
    double* out;                                // [2] device: rho, ||S_k||_2
    double* partial; unsigned* ticket;          // RHO_MAX_GRID per-CTA partial sums and the arrival counter of the reduction
};
constexpr int RHO_MAX_GRID = 64;
int rho_small(lrp_ctx* ctx, const RhoArgs& a);

// Nested case of the stop test: last sweep's index list is, up to `nrest` = kkp - k0 dropped trailing entries, a prefix
// of this sweep's, and the driver kept the Q columns of the common prefix (k0 columns), so
//   U_{k-1} = Q_k Y + P Uc_rest,   Y = [Uc_pref; 0] + T Uc_rest,   T = Q_k^T Q_rest,   P = Q_rest - Q_k T  (P _|_ Q_k),
// with Uc_pref / Uc_rest the first k0 / last nrest rows of Uc_{k-1} and Q_rest the dropped Q columns (set aside by the
// driver).  The operands of rho then come from small matrices:
//   A = U_k^T U_{k-1} = Uc_k^T Y,   E_U = Q_k M + P Uc_rest with M = Y - Uc_k A,   GU = M^T M + Uc_rest^T (P^T P) Uc_rest.
// nrest = 0 (nothing dropped): Y = [Uc_{k-1}; 0], no T, no P.  One CTA per side (side 0: U, side 1: V).
// scratch: 2 * kk * rp doubles per side.
struct RhoNestedSide {
    int kk, kkp, k0;                            // rows of Uc_k, rows of Uc_{k-1}, common prefix (k0 <= kkp, k0 <= kk)
    const double* Uc; int ldc;                  // kk x r
    const double* Ucp; int ldcp;                // kkp x rp
    const double* T;                            // kk x nrest (ld kk), unused when nrest = 0
    const double* Gp;                           // nrest x nrest (ld nrest) = P^T P
    double* A; double* G; double* scratch;      // r x rp (ld r), rp x rp (ld rp)
};
int rho_nested_prep(lrp_ctx* ctx, int r, int rp, const RhoNestedSide& u, const RhoNestedSide& v);

int leverage_colmask(lrp_ctx* ctx, int k, const double* R, int64_t ldr, double rcond, unsigned char* mask);

// top-`num` (<= 4096) of scores[0..n) ordered by (score desc, index asc) -> idx_out (device; -1 where fewer exist).
// ws: select_ws_bytes(ctx, n, num).  bern != nullptr: only the indices kept by the Bernoulli draw of Alg. 3 lines 4-5
// (u_i < min(1, c score_i / cols), u from the counter-based generator of select.cu) take part; *d_count (device) receives
// how many were kept.
struct SelectBernoulli { int cols; double c; unsigned long long seed; int sweep; int side; };
size_t select_ws_bytes(const lrp_ctx* ctx, int64_t n, int num);
int select_init(lrp_ctx* ctx);
int core_init(lrp_ctx* ctx);                     // one-time kernel attributes (lrp_create)
int select_topk(lrp_ctx* ctx, int64_t n, const double* scores, int num, int32_t* idx_out, void* ws,
                const SelectBernoulli* bern = nullptr, int* d_count = nullptr);

// (Q)DEIM index selection (Alg. 2; deim.cu): r indices in pivot order of the n x r matrix A (destroyed).
size_t deim_ws_bytes(int64_t n, int r);
int deim_select(lrp_ctx* ctx, int qdeim, int64_t n, int r, double* A, int64_t lda, int32_t* idx_out, void* ws);
