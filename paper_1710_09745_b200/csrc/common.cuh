// Internal declarations of libbkr (sm_100a).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/bkr.h"

#define BKR_NUM_SMS 148 /* B200: 2 dies x 74 SMs; grids are sized in multiples of this */
#define BKR_LINK_TILE 64 /* sites per link tile: one TMA bulk copy per (tile, hop) = 9 * 64 complex */

// Order of the 16 hops in the gather-form link stream and in the stencil's hop loop:
//   y-3, y-1, x+1, x-1, x+3, x-3, y+1, y+3, z-3, z-1, z+1, z+3, t-3, t-1, t+1, t+3.
// For a tile of consecutive x-rows (y0 .. y0+3) consecutive hops then read overlapping sets of input rows
// (y0-3..y0, y0-1..y0+2, y0..y0+3 four times, y0+1..y0+4, y0+3..y0+6), so every L1 reuse has distance one hop -- the
// only distance at which the per-hop footprint of N x 48 bytes per site survives in L1 (ncu: with the order x, y+1, y-1,
// y+3, y-3 the L1 hit rate was 24 % against 34 % possible).  Encoded as bit fields indexed by the hop number h.
#define BKR_HOP_MU_BITS 0xffaa5005u /* 2 bits per hop: direction mu */
#define BKR_HOP_LONG_BITS 0x99b1u /* 1 bit per hop: 1 = long link (three sites) */
#define BKR_HOP_BACK_BITS 0x332bu /* 1 bit per hop: 1 = backward */
#define BKR_HOP_MU(h) ((BKR_HOP_MU_BITS >> (2 * (h))) & 3u)
#define BKR_HOP_LONG(h) ((BKR_HOP_LONG_BITS >> (h)) & 1u)
#define BKR_HOP_BACK(h) ((BKR_HOP_BACK_BITS >> (h)) & 1u)

struct Geom {
    int X[4];     // extents x,y,z,t (all even, >= 4)
    int V, Vh;    // sites, sites per parity (48^3 x 96 = 10.6 M fits an int)
};

template <typename Real> struct CxT;
template <> struct CxT<double> { typedef double2 type; };
template <> struct CxT<float> { typedef float2 type; };

// Flags the solver kernels share (device memory).  Every loop kernel returns at once when done != 0,
// so the host can enqueue iterations in batches without synchronising.
struct SolverFlags {
    int done;          // 1: converged or broken down -> loop kernels become no-ops
    int breakdown;     // 1: non-positive / non-finite Cholesky pivot
    int illcond;       // with breakdown: every entry was finite -- the block is (nearly) rank deficient, not broken: the host
                       // restarts from X with the two-pass QR (solver.cu, PAPER.md:184-186 refs [43, 44])
    int iters;         // completed iterations (Alg. 1 l.9 applications of M)
    int want_update;   // mixed precision: reliable update requested (Alg. 3)
    double relres_max; // max_i ||C[:,i]|| / ||b_i||  after the last l.12
    double relres_last_update;
    // deferred X update: xpend = 1 while W = beta C of the last l.9 has not been applied to X yet;
    // xidle = !xpend (a kernel gate is "skip when the flag is non-zero", so the flush needs the negation)
    int xpend, xidle;
};

struct bkr_ctx {
    Geom g;
    int device;
    cudaStream_t stream;
    int last_cuda;
    long long launches;
    // gather-form links Wt[parity][tile][hop][el][lane] (layout.cu), fp64 and optional fp32 copy
    double2 *links64;
    float2 *links32;
    // tile processing order of the stencil (L2 blocking, dslash.cu): device table + the blocking it was built for
    int *tile_order;
    int tile_order_key;
    // segment table of the window stencil (dslash_win.cu): (first tile, end tile, strip first, strip last)
    int4 *win_segs;
    int win_nseg, win_key;
    // strip table of the row-window stencil (dslash_row.cu): first tile of each (z, t) strip in processing order
    int *row_strips;
    int row_nstrip, row_key;
    int dslash_force; // bkr_set_dslash_variant: -1 automatic, 0 plain, 1 window, 2 row window
    int l2_budget_mb, row_unit_tiles, row_vec_policy; // bkr_set_option (0 = built-in default)
    int ablation;       // BKR_OPT_ABLATION bit mask (bkr.h): 0 = the full method
    int tune[BKR_TUNE_COUNT]; // BKR_OPT_TUNE + k (bkr.h): launch parameters, 0 = default
    SolverFlags *api_flags; // device flags for the API-level fused update
    int dslash_nblock;  // rhs count of the whole block while launch_dslash works through it in chunks (L2 blocking uses it)
    int dslash_variant; // last stencil kernel used: 0 plain, 1 window, -1 none yet
    // scratch for apply_M (odd-parity temporary), grown on demand, per precision
    void *tmp_odd[2];
    size_t tmp_odd_bytes[2];
    // two-stage reduction scratch: [num_ctas][N*N] complex fp64
    double2 *partials;
    size_t partials_bytes;
    // small-matrix scratch for the API-level gram / cholesky calls
    double2 *small;
    double2 *panel; // dense (N/2) x (N/2) copies of coefficient sub-matrices for the panel launches of blocks > 32 rhs
    // solver workspace (allocated on first solve for a given N / precision, reused)
    struct Workspace *ws;
    // device staging blocks of the host-buffer entry points (kept between calls)
    double2 *stage[2];
    size_t stage_bytes;
};

#define BKR_CUDA(ctx, call)                                   \
    do {                                                      \
        cudaError_t e_ = (call);                              \
        if (e_ != cudaSuccess) {                              \
            (ctx)->last_cuda = (int)e_;                       \
            return e_ == cudaErrorMemoryAllocation ? BKR_ENOMEM : BKR_ECUDA; \
        }                                                     \
    } while (0)

// every ABI entry makes the context's device current (a context may live on any device of the process)
#define BKR_ENTER(ctx)                                                          \
    do {                                                                        \
        if (cudaSetDevice((ctx)->device) != cudaSuccess) return BKR_ECUDA;      \
    } while (0)

#define BKR_TRY(call)                 \
    do {                              \
        int rc_ = (call);             \
        if (rc_ != BKR_OK) return rc_; \
    } while (0)

static inline int bkr_check_launch(bkr_ctx *ctx)
{
    cudaError_t e = cudaGetLastError();
    ctx->launches++;
    if (e != cudaSuccess) {
        ctx->last_cuda = (int)e;
        return BKR_ECUDA;
    }
    return BKR_OK;
}

static inline size_t field_elems(const Geom &g, int N) { return (size_t)g.Vh * 3 * (size_t)N; }
static inline int link_tiles(const Geom &g) { return (g.Vh + BKR_LINK_TILE - 1) / BKR_LINK_TILE; }
static inline size_t link_elems(const Geom &g) { return (size_t)2 * link_tiles(g) * 16 * 9 * BKR_LINK_TILE; }

// ---- layout.cu
int launch_pack_links(bkr_ctx *ctx, const double2 *fat, const double2 *lng, double2 *out64, float2 *out32);
int launch_pack(bkr_ctx *ctx, int N, int prec, const double2 *canonical, void *native);
int launch_unpack(bkr_ctx *ctx, int N, int prec, const void *native, double2 *canonical);
int launch_convert(bkr_ctx *ctx, size_t n_complex, int src_prec, const void *src, int dst_prec, void *dst,
                   const int *done);

// ---- dslash.cu :  out = D in   or (xpay) out = a * xp - D in
int launch_dslash(bkr_ctx *ctx, int out_parity, int N, int prec, const void *in, void *out, const void *xp,
                  double a, const int *done);

// ---- dslash_win.cu : same operation, shared-memory window version; returns 1 when not applicable
int launch_dslash_win(bkr_ctx *ctx, int out_parity, int N, int prec, const void *in, void *out, const void *xp,
                      double a, const int *done);

// ---- dslash_row.cu : same operation, row-window version for 9..32 fp64 rhs; returns 1 when not applicable
int launch_dslash_row(bkr_ctx *ctx, int out_parity, int N, int prec, const void *in, void *out, const void *xp,
                      double a, const int *done);

// Second stage of the Gram reduction for one matrix element, by 16 lanes of a warp (lane bits 1..4 = g): the sum of
// pp[q * stride], q = 0 .. np - 1, where lane g adds q = g, g + 16, g + 32, ... (all its loads in flight at once) and a
// butterfly over the 16 lanes adds the 16 sums -- a fixed order, so every caller (small_kernel, gram_finish_kernel,
// bkr_gram_static) gets bit-identical results from the same partials (P12).  Whole warps must call it; act = this lane's
// element exists.  Lane bit 0 distinguishes two elements handled by one warp.
__device__ __forceinline__ double2 sum_partials_16(const double2 *pp, size_t stride, int np, int g, bool act)
{
    double2 acc = make_double2(0.0, 0.0);
    for (int q0 = g; q0 < np; q0 += 160) {
        double2 v[10];
#pragma unroll
        for (int c = 0; c < 10; c++) {
            const int q = q0 + 16 * c;
            v[c] = (act && q < np) ? pp[(size_t)q * stride] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int c = 0; c < 10; c++) {
            acc.x += v[c].x;
            acc.y += v[c].y;
        }
    }
#pragma unroll
    for (int m = 2; m <= 16; m <<= 1) {
        acc.x += __shfl_xor_sync(0xffffffffu, acc.x, m);
        acc.y += __shfl_xor_sync(0xffffffffu, acc.y, m);
    }
    return acc;
}

// ---- blas.cu
// stage 1 of K = X^dag Y: per-CTA partial sums into ctx->partials; returns the number of partials.
int launch_gram_partials(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian,
                         int *num_partials, const int *done);
// both stages with the partials in a file-scope device array of mblas.cu (no allocation; N <= BKR_STATIC_MAX_N)
int launch_gram_static(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, double2 *K);
// stage 2 alone (API path): K = fixed-order sum of the partials, mirrored if hermitian.  ldk: row stride of K (0 = N).
int launch_gram_finish(bkr_ctx *ctx, int N, int num_partials, int hermitian, double2 *K, int ldk = 0);
// Blocks of 34..64 rhs (N even): the whole Gram matrix K (N x N, row stride N) from the panels X_I^dag Y_J of N / 2 columns
// each -- three launches if hermitian (the lower triangle mirrored), else four; every block is read twice (PAPER.md:262-270:
// the paper's recursive tiling, one level, on the host).
int launch_gram_panels(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, double2 *K, const int *done);
// Z = C + W a   (C may be NULL = 0; Z may alias C; Z must not alias W).  a: N x N complex fp64 (device).
// precZ is the precision of Z and C, precW of W; arithmetic in precZ.
// tri: 0 = general a, 1 = a upper triangular, 2 = a lower triangular (entries on the other side are not read).
int launch_block_update(bkr_ctx *ctx, int N, int precZ, int precW, const double2 *a, const void *C,
                        const void *W, void *Z, const int *done, int tri = 0);
// Fused update at the top of an iteration (the X update of Alg. 1 l.10 deferred into the next iteration's
// l.8; Alg. 2 l.4 of the previous iteration folded in as well), one pass over Q, P, X:
//   if (!flags->done)  Q = Q Sinv (in place; Sinv upper triangular),  Pn = Q + P Sdag (S^dag lower triangular; zero
//                      fragments skipped; Pn must not alias P)
//   if (flags->xpend)  X += P Wm   (X fp64, in place).      prec = precision of P, Q, Pn.
int launch_pqx_update(bkr_ctx *ctx, int N, int prec, const double2 *Sinv, const double2 *Sdag, const double2 *Wm, void *Q,
                      const void *P, void *Pn, double2 *X, const SolverFlags *flags);
// Alg. 1 l.11 + Alg. 2 l.2 fused: Z = C + W a and stage 1 of H = Z^dag Z (Hermitian) in one pass; all blocks precision prec.
int launch_update_gram(bkr_ctx *ctx, int N, int prec, const double2 *a, const void *C, const void *W, void *Z, int *num_partials,
                       const int *done);
// per-column reductions (two-stage, deterministic), results in out[j], j < N (device fp64):
//   mode 0: sum_k |x_kj|^2        mode 1: Re sum_k conj(x_kj) y_kj      mode 2: sum_k |x_kj - y_kj|^2
int launch_col_reduce(bkr_ctx *ctx, int N, int prec, int mode, const void *X, const void *Y, double *out,
                      const int *done);
// Z = alpha * X + beta * Y elementwise with per-call real scalars (Y may be NULL); all precision prec.
int launch_axpby(bkr_ctx *ctx, size_t n_complex, int prec, double alpha, const void *X, double beta,
                 const void *Y, void *Z, const int *done);
// batched CG updates with per-column real coefficients coef[j] (device fp64):
//   mode 0: X += coef * P ; R -= coef * Q        mode 1: P = R + coef * P
int launch_cg_update(bkr_ctx *ctx, int N, int prec, int mode, const double *coef, void *X, const void *P,
                     void *R, const void *Q, const int *done);

// ---- small.cu : one-CTA kernels for the N x N algebra, see small.cu for the modes
struct SmallArgs {
    int N;
    int mode;
    int num_partials;        // > 0: input matrix = fixed-order sum of ctx partials; 0: read `in`
    const double2 *partials; // [num_partials][N*N]
    const double2 *in;       // N x N (upper triangle used)
    double2 *C, *Cprev, *Cinv; // residual factor (Alg. 1 l.4, l.12), its previous value, its inverse
    double2 *negbeta, *W;    // -beta and W = beta C  (Alg. 1 l.9, l.10)
    double2 *Sinv, *Sdag;    // S^-1 and S^dagger (Alg. 1 l.11 / l.8)
    double2 *out0, *out1;    // API path outputs
    const double *bnorm2;    // ||b_i||^2
    double tol, delta;
    SolverFlags *flags;
    int *status;             // API path
    int mixed;
    double pivot_tol;        // breakdown when a pivot d <= pivot_tol * h_jj (0: the mode's default)
    double2 *scratch;        // N x N in global memory (set by launch_small): the fourth work matrix when N > 56
};
enum { SMALL_CHOL = 0, SMALL_HPDINV = 1, SMALL_BETA = 2, SMALL_QR = 3, SMALL_INIT = 4, SMALL_RELUPD = 5, SMALL_RQ1 = 6, SMALL_RQ2 = 7 };
int launch_small(bkr_ctx *ctx, const SmallArgs &args);
// CG scalar kernel: per-rhs alpha / beta / convergence bookkeeping
struct CgScalars {
    double rho[BKR_MAX_N], pAp[BKR_MAX_N], rho_new[BKR_MAX_N], bb[BKR_MAX_N];
    double alpha[BKR_MAX_N], beta[BKR_MAX_N];
    int iters[BKR_MAX_N], conv[BKR_MAX_N];
};
int launch_cg_scalar(bkr_ctx *ctx, int N, int step, double tol, CgScalars *s, SolverFlags *flags);

// ---- microbench.cu
int run_microbench(bkr_ctx *ctx, int kind, int reps, double *result);
// ---- probes.cu (kinds 10..29: result[0] = SM cycles, [1] = work units per SM, [2] = second work count)
int run_probe(bkr_ctx *ctx, int kind, double *result);

// ---- solver.cu
int solver_block(bkr_ctx *ctx, double mass, int N, const double2 *B, double2 *X, double tol, int maxiter,
                 int inner_prec, double delta, double *true_relres, bkr_stats *stats);
int solver_cg(bkr_ctx *ctx, double mass, int N, const double2 *B, double2 *X, double tol, int maxiter,
              int batched, int *iters, double *true_relres, bkr_stats *stats);
int solver_bench_iterations(bkr_ctx *ctx, double mass, int N, int prec, const double2 *B, int iters,
                            long long *launches);
int solver_read_flags(bkr_ctx *ctx, int out[4]);
void solver_free_workspace(bkr_ctx *ctx);
void solver_invalidate(bkr_ctx *ctx); // links changed: cached bench state is stale
int ensure_partials(bkr_ctx *ctx, size_t bytes);
int ensure_tmp_odd(bkr_ctx *ctx, int N, int prec);
