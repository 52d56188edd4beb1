/*
 * bkr.h -- C ABI of libbkr: block-Krylov (blockCGrQ) solver for the even-odd preconditioned
 * improved-staggered normal operator M = 4 m^2 - D_eo D_oe on one NVIDIA B200 (sm_100a).
 *
 * The calls follow the paper's statement of the problem (arXiv:1710.09745; citations are
 * "PAPER.md:<line>" of the paper text): one matrix M fixed by the gauge links and the mass,
 * many right-hand sides, "solve M x = b" (eq. 1), BLOCKCGRQ(X, B) taking an
 * initial X and the block B (Algorithm 1), relative-residual tolerances
 * (PAPER.md:322), and the three kernel families the paper optimises: the multi-rhs stencil
 * (PAPER.md:218-232), streaming multi-BLAS (eq. 3) and reduction multi-BLAS
 * (eq. 4).
 *
 * Conventions
 *  - Every call returns an int status (BKR_OK = 0, negative = error); nothing throws or exits.
 *  - Unless a parameter says HOST, pointers are DEVICE pointers owned by the caller (e.g. PyTorch
 *    allocations); the library never frees or keeps them beyond the call (bkr_load_links copies).
 *  - Work is enqueued on the CUDA stream given to bkr_create.  Kernel-level calls (pack, dslash,
 *    apply_M, gram, block_axpy, small-matrix calls) are asynchronous; the solve calls synchronise
 *    that stream before returning because they report iteration counts.
 *  - complex = (re, im) pairs.  "canonical" arrays are fp64; "native" arrays are fp64 or fp32.
 *  - All lattice extents must be even and >= 4 (at extent 4, x+3 wraps onto x-1: legal).
 *  - 1 <= N <= BKR_MAX_N right-hand sides; anything else -> BKR_EINVAL.
 *
 * Layouts
 *  canonical links   U[mu][s][a][b]      mu = 0..3 (x,y,z,t); s = x + X(y + Y(z + Z t)); 3x3 row-major.
 *                                        Staggered phases, boundary signs and coefficients are already
 *                                        multiplied in; backward hops use U(x - h mu)^dagger (eq. 2).
 *  canonical vector  v[rhs][e][a]        e = s div 2 = even-odd index of a site of the field's parity,
 *                                        a = colour 0..2; a parity field has Vh = XYZT/2 sites.
 *  native block      v[rhs][a][e]        the L x N "composite field" of PAPER.md:176, 212-216: N vectors of
 *                                        L = 3 Vh complex stored one after the other (component j is the
 *                                        contiguous view at offset j*L); inside a vector, row k = a*Vh + e
 *                                        (colour planes, SoA over sites).  bkr_field_bytes() bytes, 16-byte
 *                                        aligned base.
 *  small matrices    a[i][j]             N x N complex fp64, row-major, device memory.
 */
#ifndef BKR_H
#define BKR_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BKR_MAX_N 64 /* blocks of more than 32 rhs must have an even N (they are worked on as two panels of N / 2) */

typedef struct bkr_ctx bkr_ctx; /* opaque: device copies of the links, workspaces, stream */

enum { BKR_F64 = 0, BKR_F32 = 1 };

enum {
    BKR_OK = 0,
    BKR_EINVAL = -1,     /* bad argument (dims, N, precision, null pointer, aliasing)             */
    BKR_ENOLINKS = -2,   /* operator call before bkr_load_links (or fp32 links not requested)      */
    BKR_ENOMEM = -3,     /* device or host allocation failed                                       */
    BKR_ECUDA = -4,      /* a CUDA call failed; bkr_last_cuda_error() gives the cudaError_t        */
    BKR_EBREAKDOWN = -5, /* the block lost rank for good (two-pass QR included) or a Gram matrix is non-finite
                          * (PAPER.md:109); X = best so far */
    BKR_ENOCONV = -6,    /* maxiter reached; X holds the last iterate, stats are filled             */
    BKR_ETOOBIG = -7     /* size beyond the fixed capacity of a no-allocation entry point (bkr_gram_static) */
};

typedef struct {
    int iters;              /* applications of M to the block inside the loop (Alg. 1 l.9)  */
    int reliable_updates;   /* Algorithm 3 invocations (0 for a pure fp64 solve)            */
    int status;             /* same value the call returned                                  */
    int restarts;           /* times the loop was re-entered because the true residual missed tol */
    double seconds;         /* wall time of the solve loop on the stream (CUDA events)      */
    double true_relres_max; /* max_i ||b_i - M x_i|| / ||b_i||, recomputed in fp64          */
    double iter_relres_max; /* max_i ||C[:,i]|| / ||b_i|| the loop stopped on */
    long long gpu_launches; /* kernels launched by this call                                  */
    int reorthonormalisations; /* two-pass QRs of an ill-conditioned residual block (refs [43, 44]) */
} bkr_stats;

/* Create a context for an X*Y*Z*T lattice on CUDA device `device`; `cuda_stream` is a cudaStream_t
 * (NULL = the legacy default stream).  */
int bkr_create(bkr_ctx **out, const int dims[4], int device, void *cuda_stream);
int bkr_destroy(bkr_ctx *ctx);

/* Copy the caller's canonical fat (one-hop) and long (three-hop) links into the library's device
 * layout (eq. 2; "reordering the ... link fields to achieve memory
 * coalescing").  also_f32 != 0 additionally keeps an fp32 copy for the inner operator of the
 * mixed-precision solver.  The caller may free its buffers on return. */
int bkr_load_links(bkr_ctx *ctx, const void *fat, const void *lng, int also_f32);

/* Bytes of one native block of N rhs on one parity in precision prec (0 on bad arguments). */
size_t bkr_field_bytes(const bkr_ctx *ctx, int N, int prec);

/* canonical fp64 [rhs][e][a]  <->  native [rhs][a][e] in precision prec. */
int bkr_pack(bkr_ctx *ctx, int N, int prec, const void *canonical, void *native);
int bkr_unpack(bkr_ctx *ctx, int N, int prec, const void *native, void *canonical);

/* Multi-rhs stencil: out = D_{out_parity, 1-out_parity} in for all N rhs, each link
 * matrix loaded once per site and reused for the N vectors.  in/out native, in != out.
 * out_parity 1: odd <- even (D_oe); 0: even <- odd (D_eo). */
int bkr_dslash(bkr_ctx *ctx, int out_parity, int N, int prec, const void *in, void *out);

/* The stencil with its "xpay" epilogue, the second half of M (the 1158 flop per site include the 12
 * of this axpy): out = a * xp - D_{out_parity, 1-out_parity} in.  xp, out: native blocks on parity out_parity; in on the
 * other parity; out must alias neither. */
int bkr_dslash_xpay(bkr_ctx *ctx, int out_parity, int N, int prec, double a, const void *xp, const void *in, void *out);

/* out = 4 m^2 in - D_eo (D_oe in) on even sites ("Schur decomposed"); in/out native. */
int bkr_apply_M(bkr_ctx *ctx, double mass, int N, int prec, const void *in, void *out);

/* Reduction multi-BLAS (eq. 4): K = X^dag Y, k_ij = sum_k conj(x_ki) y_kj, one pass over
 * the blocks, fp64 accumulation, deterministic two-stage reduction.  hermitian != 0: only i <= j is
 * computed and the rest mirrored with a real diagonal.  X, Y native; K N*N complex fp64. */
int bkr_gram(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, void *K);

/* The same reduction for callers that must not reach cudaMalloc (code under CUDA stream capture, tight serving loops,
 * harnesses that forbid allocation): bkr_gram keeps its per-CTA partial sums in a buffer it allocates on first use,
 * this entry point keeps them in a fixed device array inside the library -- 148 x 32 x 32 complex fp64 = 2.3 MB, held by
 * every GPU that loads the library until the process exits -- and calls no cudaMalloc, cudaFree or allocating library
 * routine, on the first call or later.  Arguments, layouts and result as bkr_gram with the FP64 tensor products (bit-identical
 * to its default path); N <= BKR_STATIC_MAX_N, else BKR_ETOOBIG and nothing is launched.  The array is shared by every
 * context and stream of a device: calls that overlap on the GPU race on it, so callers serialise them (one stream, or
 * events).  Nothing in it needs clearing between calls (stage 1 writes every entry stage 2 reads). */
#define BKR_STATIC_MAX_N 32
int bkr_gram_static(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, void *K);

/* Streaming multi-BLAS (eq. 3): Y <- Y + X a, y_kj += sum_i x_ki a_ij, every vector
 * streamed once.  a: N*N complex fp64; X, Y native, X != Y. */
int bkr_block_axpy(bkr_ctx *ctx, int N, int prec, const void *a, const void *X, void *Y);

/* The general form the solver uses (eq. 3; "templated on ... Y precision >= X precision", PAPER.md:260;
 * triangular coefficient matrices in Algorithm 1 l.8 and Algorithm 2 l.4):   Z <- C + W a.
 * Z, C: native blocks of precision precZ (C may be NULL = 0; Z may alias C); W: native block of precision precW, W != Z;
 * arithmetic and accumulation in fp64, rounded to precZ on store.  tri: 0 = general a, 1 = a upper triangular, 2 = a lower
 * triangular: the entries on the zero side are NOT read (they may hold anything). */
int bkr_block_update(bkr_ctx *ctx, int N, int precZ, int precW, int tri, const void *a, const void *C, const void *W, void *Z);

/* The two fused, as the solver uses them for Algorithm 1 l.11 + Algorithm 2 l.2 (aliased
 * Hermitian reduction PAPER.md:289):  Y <- Y + X a  and  K = Y^dag Y  of the updated Y, in one pass over X and Y.
 * K is the Gram matrix of Y as stored (for fp32 blocks: of the fp32-rounded result), accumulated in fp64, Hermitian
 * with a real diagonal, bit-reproducible.  a, K: N*N complex fp64 (device); X, Y native, X != Y. */
int bkr_block_axpy_gram(bkr_ctx *ctx, int N, int prec, const void *a, const void *X, void *Y, void *K);

/* The fused update the solver runs at the top of an iteration (Algorithm 2 l.4 of the previous iteration, Algorithm 1
 * l.8, and the deferred l.10 of the previous iteration), one pass over Q, P, X:
 *     if do_qp:  Q <- Q Sinv (in place);  Pn <- Q + P Sdag        Sinv UPPER triangular, Sdag LOWER triangular:
 *     if do_x :  X <- X + P Wm (in place)                          entries on the other side are NOT read
 * Sinv, Sdag, Wm: N*N complex fp64 (device).  Q, P, Pn: native blocks of precision prec, Pn != P; X: native fp64 block
 * (also when prec is fp32).  N <= 24 is what the solver uses it for; any 1 <= N <= 32 is accepted. */
int bkr_block_qpx_update(bkr_ctx *ctx, int N, int prec, const void *Sinv, const void *Sdag, const void *Wm, void *Q,
                         const void *P, void *Pn, void *X, int do_qp, int do_x);

/* Small dense algebra on the device, one kernel launch (Algorithm 2 l.3):
 * bkr_cholesky_upper: H = R^dag R, R upper triangular with real positive diagonal; Rinv = R^-1.
 * bkr_hpd_inverse   : Ginv = G^-1 for Hermitian positive-definite G (via Cholesky).
 * Inputs use the upper triangle only.  status (device int, may be NULL) receives BKR_OK/BKR_EBREAKDOWN. */
int bkr_cholesky_upper(bkr_ctx *ctx, int N, const void *H, void *R, void *Rinv, int *status);
int bkr_hpd_inverse(bkr_ctx *ctx, int N, const void *G, void *Ginv, int *status);

/* blockCGrQ (Algorithm 1) for M X = B, N rhs on even sites.
 * B, X: canonical fp64 device arrays; X holds the initial guess on entry and the solution on return.
 * Stops when max_i ||r_i|| / ||b_i|| <= tol (iterated residual from C), then recomputes the
 * true residual in fp64 and, if it misses tol, re-enters the loop from X (counted in stats->restarts).
 * inner_prec = BKR_F64: pure fp64.  BKR_F32: P, Q, MP and the inner operator in fp32 with block reliable
 * updates (Algorithm 3) whenever the max relative residual dropped by `delta`.
 * true_relres: HOST array of N doubles (may be NULL).  stats: HOST (may be NULL). */
int bkr_solve_block(bkr_ctx *ctx, double mass, int N, const void *B, void *X, double tol, int maxiter,
                    int inner_prec, double delta, double *true_relres, bkr_stats *stats);

/* The paper's baseline: CG on each rhs.  batched = 0: N sequential single-rhs solves;
 * batched = 1: one CG loop sharing the multi-rhs stencil with per-rhs scalars ("pseudo-block",
 * PAPER.md:77).  iters: HOST array of N ints (may be NULL). */
int bkr_solve_cg(bkr_ctx *ctx, double mass, int N, const void *B, void *X, double tol, int maxiter,
                 int batched, int *iters, double *true_relres, bkr_stats *stats);

/* Workload driver of the paper's model test (192 rhs solved in blocks of N = 8 .. 64, sloppy
 * sweep to 5e-6 and fine sweep to 2e-9 as in the Truncated Solver Method): nrhs right-hand sides, nrhs a multiple of
 * N, solved block by block with bkr_solve_block.  Sweep 0 solves every block to tol_sloppy from the X given on entry
 * (skipped when tol_sloppy <= 0); sweep 1 solves it to tol_fine starting from the result of sweep 0.
 * B, X: DEVICE, canonical fp64, (nrhs, Vh, 3); block b is rhs [b N, (b + 1) N).
 * true_relres: HOST array of nrhs doubles, after the last sweep (may be NULL).
 * stats: HOST array of 2 * (nrhs / N) entries, stats[2 b + sweep] (may be NULL; a skipped sweep is zeroed).
 * Returns the first non-zero status of a block solve (later blocks are still solved), else BKR_OK. */
int bkr_solve_many(bkr_ctx *ctx, double mass, int nrhs, int N, const void *B, void *X, double tol_sloppy, double tol_fine,
                   int maxiter, int inner_prec, double delta, double *true_relres, bkr_stats *stats);

/* End-to-end variants: B and X are HOST arrays (canonical fp64); the host->device copy of B and X0 and
 * the device->host copy of X run inside the call. */
int bkr_solve_block_host(bkr_ctx *ctx, double mass, int N, const void *B_host, void *X_host, double tol,
                         int maxiter, int inner_prec, double delta, double *true_relres, bkr_stats *stats);
int bkr_solve_cg_host(bkr_ctx *ctx, double mass, int N, const void *B_host, void *X_host, double tol,
                      int maxiter, int batched, int *iters, double *true_relres, bkr_stats *stats);

/* One full blockCGrQ iteration (Alg. 1 l.8-12) on synthetic state, for benchmarking the hot path
 * without a solve: initialises Q, P, C from B (canonical fp64) on the first call for this N/prec and
 * then enqueues `iters` iterations (no convergence test, no host sync).  Returns kernels launched
 * in *launches (HOST, may be NULL). */
int bkr_bench_iterations(bkr_ctx *ctx, double mass, int N, int prec, const void *B, int iters,
                         long long *launches);

/* Device-side loop state after bkr_bench_iterations (or a solve), read back with a stream synchronisation:
 * state[0] = iterations completed since the last (re)initialisation, state[1] = done flag (1: the loop kernels have
 * become no-ops), state[2] = Cholesky breakdown, state[3] = an X update is still deferred.  state: HOST, 4 ints.
 * bench.py uses it to prove that every timed iteration did its full work.  BKR_EINVAL before the first solve. */
int bkr_solver_state(bkr_ctx *ctx, int *state);

/* Which stencil kernel the most recent Dslash launch of this context used (bkr_dslash, bkr_apply_M or inside a solver):
 * 0 = plain multi-rhs kernel (register tiling + link ring), 2 = row-window kernel, 1 = shared-memory window kernel with
 * cluster-multicast links (same operation; chosen per lattice/N/precision),
 * -1 = none yet.  Diagnostic only. */
int bkr_dslash_variant(const bkr_ctx *ctx);

/* Force the stencil kernel of later calls (tests and measurements; every variant computes the same operation):
 * -1 = automatic choice (default), 0 = plain kernel, 1 = window kernel, 2 = row-window kernel (16 rhs per CTA, z/t
 * neighbours by register loads; fp64, X = 32).  A forced variant that cannot run the lattice / N falls back to the
 * plain kernel; bkr_dslash_variant() tells which one ran. */
int bkr_set_dslash_variant(bkr_ctx *ctx, int variant);

/* Launch-policy knobs (the paper's autotuner picks such parameters on first call; here they have measured
 * defaults and this call overrides them for sweeps).  value 0 restores the default.
 *   BKR_OPT_L2_BUDGET_MB    L2 working-set budget (MB) that sizes the z blocks of the stencil's sweep order
 *   BKR_OPT_ROW_UNIT_TILES  64-site tiles per work unit of the row-window stencil (1, 2, 4, 8 ...)
 *   BKR_OPT_ROW_VEC_POLICY  L2 eviction priority of its z/t neighbour loads: 0 evict_normal, 1 evict_last
 *   BKR_OPT_ABLATION        bit mask of BKR_ABL_*: parts of the method switched off for the comparison of the paper's
 *                           Fig. 4 (no block / block BLAS / block BLAS + block Dslash).  Results are
 *                           the same up to rounding; only the kernels that produce them change.  0 = the full method.
 *   BKR_OPT_TUNE + k        stencil launch parameter k of BKR_TUNE_* below (ring depths, segment length, thread
 *                           shape); every setting computes the same result. */
enum { BKR_OPT_L2_BUDGET_MB = 0, BKR_OPT_ROW_UNIT_TILES = 1, BKR_OPT_ROW_VEC_POLICY = 2, BKR_OPT_ABLATION = 3, BKR_OPT_TUNE = 16 };
enum {
    BKR_TUNE_WIN_STAGES = 0,      /* window stencil: hop-stage ring depth, 2-8 (default: the deepest that fits)          */
    BKR_TUNE_DSLASH_CHUNK = 1,    /* 1 = never split a block into chunks of 16 / 8 rhs; 2 = always split blocks > 16 rhs   */
    BKR_TUNE_WIN_SEGLEN = 2,      /* 64-site tiles per segment (default 8)                                                */
    BKR_TUNE_WIN_SLIM = 3,        /* 2 = keep spare window slots instead of releasing the lower halo early                */
    BKR_TUNE_F32_MATH = 4,        /* multi-BLAS on fp32 blocks: 0 = FP64 tensor products, exact (default); 1 = split-TF32   */
                                  /* everywhere it exists (faster per call, ~3e-7 errors: more solver iterations);          */
                                  /* 2 = split-TF32 updates only; 3 = split-TF32 reductions only                            */
    BKR_TUNE_FUSE_QPX_MAX_N = 5,  /* largest block for which the solver uses the fused Q / P / X update (default 32 = the limit)   */
    BKR_TUNE_FUSE_GRAM_MAX_N = 6, /* largest block for which it fuses the Q' update with its Gram matrix (default 16, <= 32)   */
    BKR_TUNE_COUNT = 16
};
enum {
    BKR_ABL_UNFUSED_UPDATES = 1, /* Q, P, X updates as separate kernels, X updated right after Alg. 1 l.9 (no deferral)   */
    BKR_ABL_UNFUSED_GRAM = 2,    /* Q' = Q - MP beta and its Gram matrix as two kernels                                  */
    BKR_ABL_VECTOR_BLAS = 4,     /* block updates / Gram matrices as N^2 single-vector caxpys / dot products */
    BKR_ABL_VECTOR_DSLASH = 8,   /* the stencil one rhs at a time: links re-read for every rhs         */
    BKR_ABL_NO_GRAPH = 16        /* batches of iterations as individual launches instead of one CUDA graph               */
};
int bkr_set_option(bkr_ctx *ctx, int option, int value);

/* Measured on-chip peaks for the rooflines (not on the hot path).  kind: 0 fp64 FMA, 1 fp32 FMA,
 * 2 fp64 tensor MMA (m8n8k4), 3 L2 -> SM bandwidth by 16-byte loads, 4 the same by TMA bulk copies, 5 shared-memory read
 * bandwidth.  Runs `reps` launches on the context's stream, synchronises, and writes result[0] = ms per launch,
 * result[1] = flop (kinds 0-2) or bytes (kinds 3-5) per launch.  Kinds 10-29 are the on-chip probes of csrc/probes.cu
 * (register-file / shared-memory / TMA sharing, the stencil's dry loop): result[0] = SM cycles, result[1] = work units per
 * SM, result[2] = a second work count or 0.  result: HOST array of 4 doubles. */
int bkr_microbench(bkr_ctx *ctx, int kind, int reps, double *result);

int bkr_last_cuda_error(const bkr_ctx *ctx);
const char *bkr_strerror(int status);
const char *bkr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BKR_H */
