// C ABI of libbkr (include/bkr.h): argument checking and dispatch only; all arithmetic is in the kernels.
#include "common.cuh"

#include <new>
#include <stdlib.h>
#include <string.h>

static bool valid_n(int N) { return N >= 1 && N <= BKR_MAX_N && (N <= 32 || N % 2 == 0); }
// fused-kernel entry points keep the 32-rhs limit of their kernels
static bool valid_n32(int N) { return N >= 1 && N <= 32; }
static bool valid_prec(int p) { return p == BKR_F64 || p == BKR_F32; }

extern "C" {

int bkr_create(bkr_ctx **out, const int dims[4], int device, void *cuda_stream)
{
    if (!out || !dims) return BKR_EINVAL;
    *out = nullptr;
    long long V = 1;
    for (int mu = 0; mu < 4; mu++) {
        if (dims[mu] < 4 || (dims[mu] & 1)) return BKR_EINVAL;
        V *= dims[mu];
    }
    if (V > (1LL << 30)) return BKR_EINVAL; // site indices are 32-bit; element offsets are 64-bit
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return BKR_ECUDA;
    if (cudaSetDevice(device) != cudaSuccess) return BKR_ECUDA;
    bkr_ctx *ctx = (bkr_ctx *)calloc(1, sizeof(bkr_ctx));
    if (!ctx) return BKR_ENOMEM;
    for (int mu = 0; mu < 4; mu++) ctx->g.X[mu] = dims[mu];
    ctx->g.V = (int)V;
    ctx->g.Vh = (int)(V / 2);
    ctx->device = device;
    ctx->dslash_variant = -1;
    ctx->dslash_force = -1;
    ctx->stream = (cudaStream_t)cuda_stream;
    if (cudaMalloc((void **)&ctx->small, (size_t)5 * BKR_MAX_N * BKR_MAX_N * sizeof(double2)) != cudaSuccess) {
        free(ctx);
        return BKR_ENOMEM;
    }
    *out = ctx;
    return BKR_OK;
}

int bkr_destroy(bkr_ctx *ctx)
{
    if (!ctx) return BKR_EINVAL;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    solver_free_workspace(ctx);
    cudaFree(ctx->links64);
    cudaFree(ctx->links32);
    cudaFree(ctx->tile_order);
    cudaFree(ctx->win_segs);
    cudaFree(ctx->row_strips);
    cudaFree(ctx->api_flags);
    cudaFree(ctx->tmp_odd[0]);
    cudaFree(ctx->tmp_odd[1]);
    cudaFree(ctx->partials);
    cudaFree(ctx->small);
    cudaFree(ctx->panel);
    cudaFree(ctx->stage[0]);
    cudaFree(ctx->stage[1]);
    free(ctx);
    return BKR_OK;
}

int bkr_load_links(bkr_ctx *ctx, const void *fat, const void *lng, int also_f32)
{
    if (!ctx || !fat || !lng) return BKR_EINVAL;
    BKR_ENTER(ctx);
    size_t n = link_elems(ctx->g);
    if (!ctx->links64) BKR_CUDA(ctx, cudaMalloc((void **)&ctx->links64, n * sizeof(double2)));
    if (also_f32 && !ctx->links32) BKR_CUDA(ctx, cudaMalloc((void **)&ctx->links32, n * sizeof(float2)));
    if (!also_f32 && ctx->links32) { // an fp32 copy of the previous links must not survive a reload without one
        BKR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->links32);
        ctx->links32 = nullptr;
    }
    solver_invalidate(ctx);
    return launch_pack_links(ctx, (const double2 *)fat, (const double2 *)lng, ctx->links64,
                             also_f32 ? ctx->links32 : nullptr);
}

size_t bkr_field_bytes(const bkr_ctx *ctx, int N, int prec)
{
    if (!ctx || !valid_n(N) || !valid_prec(prec)) return 0;
    return field_elems(ctx->g, N) * (prec == BKR_F64 ? sizeof(double2) : sizeof(float2));
}

int bkr_pack(bkr_ctx *ctx, int N, int prec, const void *canonical, void *native)
{
    if (!ctx || !valid_n(N) || !valid_prec(prec) || !canonical || !native || canonical == native) return BKR_EINVAL;
    BKR_ENTER(ctx);
    return launch_pack(ctx, N, prec, (const double2 *)canonical, native);
}

int bkr_unpack(bkr_ctx *ctx, int N, int prec, const void *native, void *canonical)
{
    if (!ctx || !valid_n(N) || !valid_prec(prec) || !canonical || !native || canonical == native) return BKR_EINVAL;
    BKR_ENTER(ctx);
    return launch_unpack(ctx, N, prec, native, (double2 *)canonical);
}

int bkr_dslash(bkr_ctx *ctx, int out_parity, int N, int prec, const void *in, void *out)
{
    if (!ctx || !valid_n(N) || !valid_prec(prec) || !in || !out || in == out) return BKR_EINVAL;
    BKR_ENTER(ctx);
    if (out_parity != 0 && out_parity != 1) return BKR_EINVAL;
    return launch_dslash(ctx, out_parity, N, prec, in, out, nullptr, 0.0, nullptr);
}

int bkr_dslash_xpay(bkr_ctx *ctx, int out_parity, int N, int prec, double a, const void *xp, const void *in, void *out)
{
    if (!ctx || !valid_n(N) || !valid_prec(prec) || !in || !out || !xp || in == out || xp == out) return BKR_EINVAL;
    if (out_parity != 0 && out_parity != 1) return BKR_EINVAL;
    BKR_ENTER(ctx);
    return launch_dslash(ctx, out_parity, N, prec, in, out, xp, a, nullptr);
}

int bkr_apply_M(bkr_ctx *ctx, double mass, int N, int prec, const void *in, void *out)
{
    if (!ctx || !valid_n(N) || !valid_prec(prec) || !in || !out || in == out) return BKR_EINVAL;
    BKR_ENTER(ctx);
    if (!(prec == BKR_F64 ? (void *)ctx->links64 : (void *)ctx->links32)) return BKR_ENOLINKS;
    BKR_TRY(ensure_tmp_odd(ctx, N, prec));
    BKR_TRY(launch_dslash(ctx, 1, N, prec, in, ctx->tmp_odd[prec], nullptr, 0.0, nullptr));
    return launch_dslash(ctx, 0, N, prec, ctx->tmp_odd[prec], out, in, 4.0 * mass * mass, nullptr);
}

int bkr_gram(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, void *K)
{
    if (!ctx || !valid_n(N) || !valid_prec(prec) || !X || !Y || !K) return BKR_EINVAL;
    BKR_ENTER(ctx);
    int np = 0;
    if (N > 32) return launch_gram_panels(ctx, N, prec, X, Y, hermitian ? 1 : 0, (double2 *)K, nullptr);
    BKR_TRY(launch_gram_partials(ctx, N, prec, X, Y, hermitian ? 1 : 0, &np, nullptr));
    return launch_gram_finish(ctx, N, np, hermitian ? 1 : 0, (double2 *)K);
}

int bkr_gram_static(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, void *K)
{
    if (!ctx || N < 1 || !valid_prec(prec) || !X || !Y || !K) return BKR_EINVAL;
    if (N > BKR_STATIC_MAX_N) return BKR_ETOOBIG;
    BKR_ENTER(ctx);
    return launch_gram_static(ctx, N, prec, X, Y, hermitian ? 1 : 0, (double2 *)K);
}

int bkr_block_axpy(bkr_ctx *ctx, int N, int prec, const void *a, const void *X, void *Y)
{
    if (!ctx || !valid_n(N) || !valid_prec(prec) || !a || !X || !Y || X == Y) return BKR_EINVAL;
    BKR_ENTER(ctx);
    return launch_block_update(ctx, N, prec, prec, (const double2 *)a, Y, X, Y, nullptr);
}

int bkr_block_update(bkr_ctx *ctx, int N, int precZ, int precW, int tri, const void *a, const void *C, const void *W, void *Z)
{
    if (!ctx || !valid_n(N) || !valid_prec(precZ) || !valid_prec(precW) || tri < 0 || tri > 2 || !a || !W || !Z || W == Z) return BKR_EINVAL;
    BKR_ENTER(ctx);
    return launch_block_update(ctx, N, precZ, precW, (const double2 *)a, C, W, Z, nullptr, tri);
}

int bkr_block_axpy_gram(bkr_ctx *ctx, int N, int prec, const void *a, const void *X, void *Y, void *K)
{
    if (!ctx || !valid_n32(N) || !valid_prec(prec) || !a || !X || !Y || !K || X == Y) return BKR_EINVAL;
    BKR_ENTER(ctx);
    int np = 0;
    BKR_TRY(launch_update_gram(ctx, N, prec, (const double2 *)a, Y, X, Y, &np, nullptr));
    return launch_gram_finish(ctx, N, np, 1, (double2 *)K);
}

int bkr_block_qpx_update(bkr_ctx *ctx, int N, int prec, const void *Sinv, const void *Sdag, const void *Wm, void *Q,
                         const void *P, void *Pn, void *X, int do_qp, int do_x)
{
    if (!ctx || !valid_n32(N) || !valid_prec(prec) || !Sinv || !Sdag || !Wm || !Q || !P || !Pn || !X || P == Pn) return BKR_EINVAL;
    BKR_ENTER(ctx);
    if (!ctx->api_flags) BKR_CUDA(ctx, cudaMalloc((void **)&ctx->api_flags, sizeof(SolverFlags)));
    SolverFlags f;
    memset(&f, 0, sizeof(f));
    f.done = do_qp ? 0 : 1;
    f.xpend = do_x ? 1 : 0;
    f.xidle = do_x ? 0 : 1;
    // small synchronous copy from the stack: ordered before the kernel by the stream synchronisation
    BKR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    BKR_CUDA(ctx, cudaMemcpy(ctx->api_flags, &f, sizeof(f), cudaMemcpyHostToDevice));
    return launch_pqx_update(ctx, N, prec, (const double2 *)Sinv, (const double2 *)Sdag, (const double2 *)Wm, Q, P, Pn,
                             (double2 *)X, ctx->api_flags);
}

int bkr_cholesky_upper(bkr_ctx *ctx, int N, const void *H, void *R, void *Rinv, int *status)
{
    if (!ctx || N < 1 || N > BKR_MAX_N || !H || !R) return BKR_EINVAL;
    BKR_ENTER(ctx);
    SmallArgs a;
    memset(&a, 0, sizeof(a));
    a.N = N;
    a.mode = SMALL_CHOL;
    a.in = (const double2 *)H;
    a.out0 = (double2 *)R;
    a.out1 = (double2 *)Rinv;
    a.status = status;
    return launch_small(ctx, a);
}

int bkr_hpd_inverse(bkr_ctx *ctx, int N, const void *G, void *Ginv, int *status)
{
    if (!ctx || N < 1 || N > BKR_MAX_N || !G || !Ginv) return BKR_EINVAL;
    BKR_ENTER(ctx);
    SmallArgs a;
    memset(&a, 0, sizeof(a));
    a.N = N;
    a.mode = SMALL_HPDINV;
    a.in = (const double2 *)G;
    a.out0 = (double2 *)Ginv;
    a.status = status;
    return launch_small(ctx, a);
}

static bool valid_solve(bkr_ctx *ctx, int N, const void *B, void *X, double tol, int maxiter)
{
    return ctx && valid_n(N) && B && X && B != X && tol > 0.0 && maxiter >= 0;
}

int bkr_solve_block(bkr_ctx *ctx, double mass, int N, const void *B, void *X, double tol, int maxiter, int inner_prec,
                    double delta, double *true_relres, bkr_stats *stats)
{
    if (!valid_solve(ctx, N, B, X, tol, maxiter) || !valid_prec(inner_prec)) return BKR_EINVAL;
    BKR_ENTER(ctx);
    if (inner_prec == BKR_F32 && !(delta > 0.0 && delta < 1.0)) return BKR_EINVAL;
    if (!ctx->links64 || (inner_prec == BKR_F32 && !ctx->links32)) return BKR_ENOLINKS;
    int rc = solver_block(ctx, mass, N, (const double2 *)B, (double2 *)X, tol, maxiter, inner_prec, delta, true_relres,
                          stats);
    if (stats) stats->status = rc;
    return rc;
}

int bkr_solve_many(bkr_ctx *ctx, double mass, int nrhs, int N, const void *B, void *X, double tol_sloppy, double tol_fine,
                   int maxiter, int inner_prec, double delta, double *true_relres, bkr_stats *stats)
{
    if (!valid_solve(ctx, N, B, X, tol_fine, maxiter) || !valid_prec(inner_prec) || nrhs < N || nrhs % N != 0) return BKR_EINVAL;
    BKR_ENTER(ctx);
    if (inner_prec == BKR_F32 && !(delta > 0.0 && delta < 1.0)) return BKR_EINVAL;
    if (!ctx->links64 || (inner_prec == BKR_F32 && !ctx->links32)) return BKR_ENOLINKS;
    const size_t blk = (size_t)N * ctx->g.Vh * 3; // complex numbers per block
    int first = BKR_OK;
    for (int b = 0; b < nrhs / N; b++) {
        const double2 *Bb = (const double2 *)B + (size_t)b * blk;
        double2 *Xb = (double2 *)X + (size_t)b * blk;
        for (int sweep = 0; sweep < 2; sweep++) {
            bkr_stats *st = stats ? stats + 2 * b + sweep : nullptr;
            if (sweep == 0 && !(tol_sloppy > 0.0)) {
                if (st) memset(st, 0, sizeof(*st));
                continue;
            }
            const int rc = solver_block(ctx, mass, N, Bb, Xb, sweep == 0 ? tol_sloppy : tol_fine, maxiter, inner_prec, delta,
                                        true_relres ? true_relres + (size_t)b * N : nullptr, st);
            if (st) st->status = rc;
            if (rc != BKR_OK && first == BKR_OK) first = rc;
            if (rc == BKR_ECUDA || rc == BKR_ENOMEM) return rc;
        }
    }
    return first;
}

int bkr_solve_cg(bkr_ctx *ctx, double mass, int N, const void *B, void *X, double tol, int maxiter, int batched,
                 int *iters, double *true_relres, bkr_stats *stats)
{
    if (!valid_solve(ctx, N, B, X, tol, maxiter)) return BKR_EINVAL;
    BKR_ENTER(ctx);
    if (!ctx->links64) return BKR_ENOLINKS;
    int rc = solver_cg(ctx, mass, N, (const double2 *)B, (double2 *)X, tol, maxiter, batched ? 1 : 0, iters,
                       true_relres, stats);
    if (stats) stats->status = rc;
    return rc;
}

// host-buffer variants: staging through two device blocks the context keeps between calls (no allocation in the timed
// end-to-end region after the first call for a given N)
static int with_host_buffers(bkr_ctx *ctx, int N, const void *B_host, void *X_host, double2 **dB, double2 **dX)
{
    const size_t bytes = field_elems(ctx->g, N) * sizeof(double2);
    if (ctx->stage_bytes < bytes) {
        cudaFree(ctx->stage[0]);
        cudaFree(ctx->stage[1]);
        ctx->stage[0] = ctx->stage[1] = nullptr;
        ctx->stage_bytes = 0;
        BKR_CUDA(ctx, cudaMalloc((void **)&ctx->stage[0], bytes));
        if (cudaMalloc((void **)&ctx->stage[1], bytes) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(ctx->stage[0]);
            ctx->stage[0] = nullptr;
            return BKR_ENOMEM;
        }
        ctx->stage_bytes = bytes;
    }
    *dB = ctx->stage[0];
    *dX = ctx->stage[1];
    BKR_CUDA(ctx, cudaMemcpyAsync(*dB, B_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    BKR_CUDA(ctx, cudaMemcpyAsync(*dX, X_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    return BKR_OK;
}

static int finish_host_buffers(bkr_ctx *ctx, int N, void *X_host, double2 *dX, int rc)
{
    const size_t bytes = field_elems(ctx->g, N) * sizeof(double2);
    cudaError_t e = cudaMemcpyAsync(X_host, dX, bytes, cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) {
        ctx->last_cuda = (int)e;
        return BKR_ECUDA;
    }
    return rc;
}

int bkr_solve_block_host(bkr_ctx *ctx, double mass, int N, const void *B_host, void *X_host, double tol, int maxiter,
                         int inner_prec, double delta, double *true_relres, bkr_stats *stats)
{
    if (!valid_solve(ctx, N, B_host, X_host, tol, maxiter)) return BKR_EINVAL;
    BKR_ENTER(ctx);
    double2 *dB, *dX;
    BKR_TRY(with_host_buffers(ctx, N, B_host, X_host, &dB, &dX));
    int rc = bkr_solve_block(ctx, mass, N, dB, dX, tol, maxiter, inner_prec, delta, true_relres, stats);
    return finish_host_buffers(ctx, N, X_host, dX, rc);
}

int bkr_solve_cg_host(bkr_ctx *ctx, double mass, int N, const void *B_host, void *X_host, double tol, int maxiter,
                      int batched, int *iters, double *true_relres, bkr_stats *stats)
{
    if (!valid_solve(ctx, N, B_host, X_host, tol, maxiter)) return BKR_EINVAL;
    BKR_ENTER(ctx);
    double2 *dB, *dX;
    BKR_TRY(with_host_buffers(ctx, N, B_host, X_host, &dB, &dX));
    int rc = bkr_solve_cg(ctx, mass, N, dB, dX, tol, maxiter, batched, iters, true_relres, stats);
    return finish_host_buffers(ctx, N, X_host, dX, rc);
}

int bkr_bench_iterations(bkr_ctx *ctx, double mass, int N, int prec, const void *B, int iters, long long *launches)
{
    if (!ctx || !valid_n(N) || !valid_prec(prec) || !B || iters < 0) return BKR_EINVAL;
    BKR_ENTER(ctx);
    if (!ctx->links64 || (prec == BKR_F32 && !ctx->links32)) return BKR_ENOLINKS;
    return solver_bench_iterations(ctx, mass, N, prec, (const double2 *)B, iters, launches);
}

int bkr_solver_state(bkr_ctx *ctx, int *state)
{
    if (!ctx || !state) return BKR_EINVAL;
    BKR_ENTER(ctx);
    return solver_read_flags(ctx, state);
}

int bkr_microbench(bkr_ctx *ctx, int kind, int reps, double *result)
{
    if (!ctx) return BKR_EINVAL;
    BKR_ENTER(ctx);
    return run_microbench(ctx, kind, reps, result);
}

int bkr_last_cuda_error(const bkr_ctx *ctx) { return ctx ? ctx->last_cuda : 0; }

const char *bkr_strerror(int status)
{
    switch (status) {
    case BKR_OK: return "ok";
    case BKR_EINVAL: return "invalid argument";
    case BKR_ENOLINKS: return "links not loaded (or no fp32 copy requested)";
    case BKR_ENOMEM: return "out of memory";
    case BKR_ECUDA: return "CUDA error (see bkr_last_cuda_error)";
    case BKR_EBREAKDOWN: return "Cholesky breakdown: block lost rank or non-finite Gram matrix";
    case BKR_ENOCONV: return "maxiter reached without convergence";
    case BKR_ETOOBIG: return "size beyond the fixed capacity of this no-allocation entry point (N <= 32 for bkr_gram_static)";
    default: return "unknown status";
    }
}

int bkr_dslash_variant(const bkr_ctx *ctx) { return ctx ? ctx->dslash_variant : -1; }

int bkr_set_option(bkr_ctx *ctx, int option, int value)
{
    if (!ctx || value < 0) return BKR_EINVAL;
    switch (option) {
    case BKR_OPT_L2_BUDGET_MB: ctx->l2_budget_mb = value; break;
    case BKR_OPT_ROW_UNIT_TILES: ctx->row_unit_tiles = value; break;
    case BKR_OPT_ROW_VEC_POLICY: ctx->row_vec_policy = value; break;
    case BKR_OPT_ABLATION: ctx->ablation = value & 31; break;
    default:
        if (option < BKR_OPT_TUNE || option >= BKR_OPT_TUNE + BKR_TUNE_COUNT) return BKR_EINVAL;
        ctx->tune[option - BKR_OPT_TUNE] = value;
    }
    // blocking tables are rebuilt on the next stencil call
    ctx->tile_order_key = ctx->win_key = ctx->row_key = -1;
    return BKR_OK;
}

int bkr_set_dslash_variant(bkr_ctx *ctx, int variant)
{
    if (!ctx || variant < -1 || variant > 2) return BKR_EINVAL;
    ctx->dslash_force = variant;
    return BKR_OK;
}

const char *bkr_version(void) { return "libbkr 0.1 (sm_100a)"; }

} // extern "C"
