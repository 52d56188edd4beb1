// Second stage of the Gram reduction and the per-column kernels of the CG baseline on native blocks
// v[j][k].  The block kernels (reduction and streaming multi-BLAS) are in mblas.cu.
#include "common.cuh"

int ensure_partials(bkr_ctx *ctx, size_t bytes)
{
    if (ctx->partials_bytes >= bytes) return BKR_OK;
    if (ctx->partials) cudaFree(ctx->partials);
    ctx->partials = nullptr;
    ctx->partials_bytes = 0;
    BKR_CUDA(ctx, cudaMalloc((void **)&ctx->partials, bytes));
    ctx->partials_bytes = bytes;
    return BKR_OK;
}

// ------------------------------------------------------------------------------------------ Gram, stage 2
// Two matrix elements per warp, 16 lanes each (sum_partials_16): one thread per element walking its 148 partials one after the
// other took 34 us per call at N = 16, 12 % of a two-block reduction on the API path.
static const int GRAM_FINISH_THREADS = 128;
static inline unsigned gram_finish_blocks(int N) { return (unsigned)(((size_t)N * N * 16 + GRAM_FINISH_THREADS - 1) / GRAM_FINISH_THREADS); }

__global__ void __launch_bounds__(GRAM_FINISH_THREADS)
gram_finish_kernel(int N, int num_partials, int hermitian, const double2 *__restrict__ partials, double2 *__restrict__ K, int ldk,
                   const int *done)
{
    if (done && *done) return;
    const int w = (blockIdx.x * GRAM_FINISH_THREADS + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 1, o = 2 * w + (lane & 1);
    const bool act = o < N * N;
    const int i = act ? o / N : 0, j = act ? o % N : 0;
    const bool lower = hermitian && i > j;
    const int src = lower ? j * N + i : i * N + j;
    double2 s = sum_partials_16(partials + src, (size_t)N * N, num_partials, g, act);
    if (act && g == 0) {
        if (lower) s.y = -s.y;
        if (hermitian && i == j) s.y = 0.0;
        K[i * ldk + j] = s;
    }
}

int launch_gram_finish(bkr_ctx *ctx, int N, int num_partials, int hermitian, double2 *K, int ldk)
{
    gram_finish_kernel<<<gram_finish_blocks(N), GRAM_FINISH_THREADS, 0, ctx->stream>>>(N, num_partials, hermitian, ctx->partials, K, ldk ? ldk : N,
                                                                     nullptr);
    return bkr_check_launch(ctx);
}

// lower triangle of an N x N matrix from its upper one: K_ij = conj(K_ji), i > j
__global__ void mirror_lower_kernel(int N, double2 *K, const int *done)
{
    if (done && *done) return;
    const int o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= N * N) return;
    const int i = o / N, j = o % N;
    if (i > j) {
        const double2 v = K[j * N + i];
        K[o] = make_double2(v.x, -v.y);
    }
}

int launch_gram_panels(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, double2 *K, const int *done)
{
    const int p = N / 2;
    const size_t col = (size_t)3 * ctx->g.Vh * (prec == BKR_F64 ? sizeof(double2) : sizeof(float2));
    for (int I = 0; I < 2; I++)
        for (int J = 0; J < 2; J++) {
            if (hermitian && I > J) continue;
            int np = 0;
            const char *xi = (const char *)X + (size_t)I * p * col, *yj = (const char *)Y + (size_t)J * p * col;
            BKR_TRY(launch_gram_partials(ctx, p, prec, xi, yj, (hermitian && I == J) ? 1 : 0, &np, done));
            gram_finish_kernel<<<gram_finish_blocks(p), GRAM_FINISH_THREADS, 0, ctx->stream>>>(p, np, (hermitian && I == J) ? 1 : 0, ctx->partials,
                                                                             K + (size_t)I * p * N + (size_t)J * p, N, done);
            BKR_TRY(bkr_check_launch(ctx));
        }
    if (hermitian) {
        mirror_lower_kernel<<<(N * N + 127) / 128, 128, 0, ctx->stream>>>(N, K, done);
        BKR_TRY(bkr_check_launch(ctx));
    }
    return BKR_OK;
}

// ------------------------------------------------------------------------------------------ per-column kernels
// The CG baseline works on single vectors: column j of a native block is the contiguous range
// [j L, (j+1) L).  blockIdx.y = column.  Reductions: per-thread serial sums over a grid-stride loop, fixed-order
// tree in shared memory, one partial per CTA, fixed-order final sum (col_finish_kernel): deterministic.
static const int COL_THREADS = 256;

template <typename Real>
__global__ void __launch_bounds__(COL_THREADS)
col_reduce_kernel(size_t L, int mode, const typename CxT<Real>::type *__restrict__ X,
                  const typename CxT<Real>::type *__restrict__ Y, double *__restrict__ partials, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    __shared__ double red[COL_THREADS];
    if (done && *done) return;
    const int j = blockIdx.y;
    const Cx *x = X + (size_t)j * L;
    const Cx *y = Y ? Y + (size_t)j * L : nullptr;
    double s0 = 0.0, s1 = 0.0;
    const size_t stride = (size_t)gridDim.x * COL_THREADS;
    for (size_t k = (size_t)blockIdx.x * COL_THREADS + threadIdx.x; k < L; k += stride) {
        const Cx xv = x[k];
        const double xr = xv.x, xi = xv.y;
        if (mode == 0) {
            s0 = fma(xr, xr, s0);
            s1 = fma(xi, xi, s1);
        } else {
            const Cx yv = y[k];
            const double yr = yv.x, yi = yv.y;
            if (mode == 1) {
                s0 = fma(xr, yr, s0);
                s1 = fma(xi, yi, s1);
            } else {
                const double dr = xr - yr, di = xi - yi;
                s0 = fma(dr, dr, s0);
                s1 = fma(di, di, s1);
            }
        }
    }
    red[threadIdx.x] = s0 + s1;
    __syncthreads();
    for (int w = COL_THREADS / 2; w > 0; w >>= 1) {
        if (threadIdx.x < w) red[threadIdx.x] += red[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) partials[(size_t)j * gridDim.x + blockIdx.x] = red[0];
}

__global__ void col_finish_kernel(int N, int num_partials, const double *__restrict__ partials, double *__restrict__ out,
                                  const int *done)
{
    if (done && *done) return;
    int j = threadIdx.x;
    if (j >= N) return;
    double s = 0.0;
    for (int p = 0; p < num_partials; p++) s += partials[(size_t)j * num_partials + p];
    out[j] = s;
}

int launch_col_reduce(bkr_ctx *ctx, int N, int prec, int mode, const void *X, const void *Y, double *out, const int *done)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    size_t nb = (L + COL_THREADS * 4 - 1) / (COL_THREADS * 4);
    const size_t cap = (size_t)BKR_NUM_SMS * 8 / N + 1;
    unsigned gx = (unsigned)(nb < cap ? nb : cap);
    BKR_TRY(ensure_partials(ctx, (size_t)2 * BKR_NUM_SMS * BKR_MAX_N * BKR_MAX_N * sizeof(double2)));
    double *part = (double *)ctx->partials;
    dim3 grid(gx, N);
    if (prec == BKR_F64)
        col_reduce_kernel<double><<<grid, COL_THREADS, 0, ctx->stream>>>(L, mode, (const double2 *)X, (const double2 *)Y, part, done);
    else
        col_reduce_kernel<float><<<grid, COL_THREADS, 0, ctx->stream>>>(L, mode, (const float2 *)X, (const float2 *)Y, part, done);
    BKR_TRY(bkr_check_launch(ctx));
    col_finish_kernel<<<1, BKR_MAX_N, 0, ctx->stream>>>(N, (int)gx, part, out, done);
    return bkr_check_launch(ctx);
}

template <typename Real>
__global__ void axpby_kernel(size_t n, Real alpha, const typename CxT<Real>::type *__restrict__ X, Real beta,
                             const typename CxT<Real>::type *Y, typename CxT<Real>::type *Z, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    if (done && *done) return;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t stride = (size_t)gridDim.x * blockDim.x;
    for (; i < n; i += stride) {
        Cx x = X[i], o;
        o.x = alpha * x.x;
        o.y = alpha * x.y;
        if (Y) {
            Cx y = Y[i];
            o.x = fma(beta, y.x, o.x);
            o.y = fma(beta, y.y, o.y);
        }
        Z[i] = o;
    }
}

int launch_axpby(bkr_ctx *ctx, size_t n, int prec, double alpha, const void *X, double beta, const void *Y, void *Z,
                 const int *done)
{
    size_t nb = (n + 255) / 256;
    unsigned grid = (unsigned)(nb < (size_t)BKR_NUM_SMS * 16 ? nb : (size_t)BKR_NUM_SMS * 16);
    if (prec == BKR_F64)
        axpby_kernel<double><<<grid, 256, 0, ctx->stream>>>(n, alpha, (const double2 *)X, beta, (const double2 *)Y, (double2 *)Z, done);
    else
        axpby_kernel<float><<<grid, 256, 0, ctx->stream>>>(n, (float)alpha, (const float2 *)X, (float)beta, (const float2 *)Y, (float2 *)Z, done);
    return bkr_check_launch(ctx);
}

// batched CG updates with per-column real coefficients (the "pseudo-block" baseline); blockIdx.y = column
template <typename Real>
__global__ void __launch_bounds__(256)
cg_update_kernel(size_t L, int mode, const double *__restrict__ coef, typename CxT<Real>::type *X,
                 typename CxT<Real>::type *P, typename CxT<Real>::type *R, const typename CxT<Real>::type *Q,
                 const int *done)
{
    typedef typename CxT<Real>::type Cx;
    if (done && *done) return;
    const int j = blockIdx.y;
    const Real cf = (Real)coef[j];
    const size_t base = (size_t)j * L;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < L; k += stride) {
        const size_t o = base + k;
        if (mode == 0) {
            Cx x = X[o], p = P[o], r = R[o], q = Q[o];
            x.x = fma(cf, p.x, x.x);
            x.y = fma(cf, p.y, x.y);
            r.x = fma(-cf, q.x, r.x);
            r.y = fma(-cf, q.y, r.y);
            X[o] = x;
            R[o] = r;
        } else {
            Cx p = P[o], r = R[o];
            p.x = fma(cf, p.x, r.x);
            p.y = fma(cf, p.y, r.y);
            P[o] = p;
        }
    }
}

int launch_cg_update(bkr_ctx *ctx, int N, int prec, int mode, const double *coef, void *X, const void *P, void *R,
                     const void *Q, const int *done)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    size_t nb = (L + 255) / 256;
    const size_t cap = (size_t)BKR_NUM_SMS * 16 / N + 1;
    dim3 grid((unsigned)(nb < cap ? nb : cap), N);
    if (prec == BKR_F64)
        cg_update_kernel<double><<<grid, 256, 0, ctx->stream>>>(L, mode, coef, (double2 *)X, (double2 *)P, (double2 *)R, (const double2 *)Q, done);
    else
        cg_update_kernel<float><<<grid, 256, 0, ctx->stream>>>(L, mode, coef, (float2 *)X, (float2 *)P, (float2 *)R, (const float2 *)Q, done);
    return bkr_check_launch(ctx);
}
