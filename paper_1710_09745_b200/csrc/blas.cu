// Multi-BLAS on native blocks (row-major L x N, row k = 3 e + a):
//   reduction multi-BLAS  K = X^dag Y          PAPER.md:272-299 (eq. 4)
//   streaming multi-BLAS  Z = C + W a          PAPER.md:245-270 (eq. 3; Alg. 1 l.8, l.10, l.11, Alg. 2 l.4)
// plus the per-column kernels of the CG baseline.  Both block kernels stream every vector
// element once, so memory traffic is linear in N.  Reductions accumulate in fp64 whatever the
// storage precision and finish in a fixed order (no floating-point atomics): results are bit-reproducible.
#include "common.cuh"

static const int GRAM_THREADS = 256;
static const int GRAM_TI = 4; // register tile of the N x N output per thread: TI x TI

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

// ------------------------------------------------------------------------------------------ Gram, stage 1
// Thread (tile, ks): tile = (ti, tj) of the output, ks = slice of the rows.  Tiles vary fastest over the lanes,
// so the lanes of a warp read the same one or two rows: 4 distinct 64-byte pieces of X and of Y per row,
// broadcast to the lanes that share them.  Each thread keeps TI x TI complex fp64 accumulators.
template <typename Real, bool HERM>
__global__ void __launch_bounds__(GRAM_THREADS)
gram_kernel(size_t L, int N, const typename CxT<Real>::type *__restrict__ X,
            const typename CxT<Real>::type *__restrict__ Y, double2 *__restrict__ partials, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int TI = GRAM_TI;
    extern __shared__ double2 red[]; // [active threads][TI*TI]
    if (done && *done) return;
    const int NT = (N + TI - 1) / TI;
    const int ntiles = HERM ? NT * (NT + 1) / 2 : NT * NT;
    const int KS = GRAM_THREADS / ntiles;
    const int tile = threadIdx.x % ntiles, ks = threadIdx.x / ntiles;
    int ti, tj;
    if (HERM) { // enumerate ti <= tj
        int t = tile;
        ti = 0;
        while (t >= NT - ti) {
            t -= NT - ti;
            ti++;
        }
        tj = ti + t;
    } else {
        ti = tile / NT;
        tj = tile % NT;
    }
    double2 acc[TI][TI];
#pragma unroll
    for (int a = 0; a < TI; a++)
#pragma unroll
        for (int b = 0; b < TI; b++) acc[a][b] = make_double2(0.0, 0.0);

    // contiguous chunk of rows per CTA
    size_t rows_per_cta = (L + gridDim.x - 1) / gridDim.x;
    size_t r0 = (size_t)blockIdx.x * rows_per_cta;
    size_t r1 = r0 + rows_per_cta < L ? r0 + rows_per_cta : L;
    if (ks < KS) {
        for (size_t k = r0 + ks; k < r1; k += KS) {
            double2 x[TI], y[TI];
#pragma unroll
            for (int a = 0; a < TI; a++) {
                int i = ti * TI + a, j = tj * TI + a;
                Cx xv = i < N ? __ldg(X + k * N + i) : Cx{0, 0};
                Cx yv = j < N ? __ldg(Y + k * N + j) : Cx{0, 0};
                x[a] = make_double2((double)xv.x, (double)xv.y);
                y[a] = make_double2((double)yv.x, (double)yv.y);
            }
#pragma unroll
            for (int a = 0; a < TI; a++)
#pragma unroll
                for (int b = 0; b < TI; b++) { // conj(x_a) * y_b
                    acc[a][b].x = fma(x[a].x, y[b].x, acc[a][b].x);
                    acc[a][b].x = fma(x[a].y, y[b].y, acc[a][b].x);
                    acc[a][b].y = fma(x[a].x, y[b].y, acc[a][b].y);
                    acc[a][b].y = fma(-x[a].y, y[b].x, acc[a][b].y);
                }
        }
    }
    // block reduction over the row slices, fixed order
#pragma unroll
    for (int a = 0; a < TI; a++)
#pragma unroll
        for (int b = 0; b < TI; b++) red[(size_t)threadIdx.x * (TI * TI) + a * TI + b] = acc[a][b];
    __syncthreads();
    // warp-shuffle-free fixed-order tree: element q of tile t summed over ks by one thread per (t, q)
    for (int o = threadIdx.x; o < ntiles * TI * TI; o += GRAM_THREADS) {
        int t = o / (TI * TI), q = o % (TI * TI);
        double2 s = make_double2(0.0, 0.0);
        for (int k2 = 0; k2 < KS; k2++) {
            double2 v = red[(size_t)(k2 * ntiles + t) * (TI * TI) + q];
            s.x += v.x;
            s.y += v.y;
        }
        // scatter to the N x N partial of this CTA
        int tti, ttj;
        if (HERM) {
            int tt = t;
            tti = 0;
            while (tt >= NT - tti) {
                tt -= NT - tti;
                tti++;
            }
            ttj = tti + tt;
        } else {
            tti = t / NT;
            ttj = t % NT;
        }
        int i = tti * TI + q / TI, j = ttj * TI + q % TI;
        if (i < N && j < N) partials[(size_t)blockIdx.x * N * N + i * N + j] = s;
    }
}

int launch_gram_partials(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, int *num_partials,
                         const int *done)
{
    size_t L = (size_t)ctx->g.Vh * 3;
    int grid = BKR_NUM_SMS * 2;
    if ((size_t)grid * 64 > L) grid = (int)((L + 63) / 64);
    BKR_TRY(ensure_partials(ctx, (size_t)BKR_NUM_SMS * 2 * BKR_MAX_N * BKR_MAX_N * sizeof(double2)));
    size_t smem = (size_t)GRAM_THREADS * GRAM_TI * GRAM_TI * sizeof(double2);
#define GRAM_GO(Real, H)                                                                                              \
    do {                                                                                                              \
        static bool attr_set = false;                                                                                 \
        if (!attr_set) {                                                                                              \
            cudaFuncSetAttribute(gram_kernel<Real, H>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);       \
            attr_set = true;                                                                                          \
        }                                                                                                             \
        gram_kernel<Real, H><<<grid, GRAM_THREADS, smem, ctx->stream>>>(L, N, (const CxT<Real>::type *)X,             \
                                                                        (const CxT<Real>::type *)Y, ctx->partials, done); \
    } while (0)
    if (prec == BKR_F64) {
        if (hermitian) GRAM_GO(double, true); else GRAM_GO(double, false);
    } else {
        if (hermitian) GRAM_GO(float, true); else GRAM_GO(float, false);
    }
#undef GRAM_GO
    *num_partials = grid;
    return bkr_check_launch(ctx);
}

// ------------------------------------------------------------------------------------------ Gram, stage 2
__global__ void gram_finish_kernel(int N, int num_partials, int hermitian, const double2 *__restrict__ partials,
                                   double2 *__restrict__ K)
{
    int o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= N * N) return;
    int i = o / N, j = o % N;
    bool lower = hermitian && i > j;
    int src = lower ? j * N + i : o;
    double2 s = make_double2(0.0, 0.0);
    for (int p = 0; p < num_partials; p++) {
        double2 v = partials[(size_t)p * N * N + src];
        s.x += v.x;
        s.y += v.y;
    }
    if (lower) s.y = -s.y;
    if (hermitian && i == j) s.y = 0.0;
    K[o] = s;
}

int launch_gram_finish(bkr_ctx *ctx, int N, int num_partials, int hermitian, double2 *K)
{
    gram_finish_kernel<<<(N * N + 127) / 128, 128, 0, ctx->stream>>>(N, num_partials, hermitian, ctx->partials, K);
    return bkr_check_launch(ctx);
}

// ------------------------------------------------------------------------------------------ streaming update
// Z = C + W a.  blockDim = (N, R): thread (j, r) owns column j of a (in registers) and walks over rows
// k = r, r + R*gridDim, ...; the N threads of a row read w_k0..w_k,N-1 with warp-broadcast loads.
template <typename A, typename B> struct WiderT { typedef double type; };
template <> struct WiderT<float, float> { typedef float type; };

template <typename RealZ, typename RealW, int NMAX>
__global__ void __launch_bounds__(256)
update_kernel(size_t L, int N, const double2 *__restrict__ a, const typename CxT<RealZ>::type *C,
              const typename CxT<RealW>::type *__restrict__ W, typename CxT<RealZ>::type *Z, const int *done)
{
    typedef typename CxT<RealZ>::type CxZ;
    typedef typename CxT<RealW>::type CxW;
    if (done && *done) return;
    typedef typename WiderT<RealZ, RealW>::type Acc; // arithmetic in the wider of the two precisions
    const int j = threadIdx.x;
    Acc ar[NMAX], ai[NMAX];
#pragma unroll
    for (int i = 0; i < NMAX; i++) {
        double2 v = i < N ? a[i * N + j] : make_double2(0.0, 0.0);
        ar[i] = (Acc)v.x;
        ai[i] = (Acc)v.y;
    }
    size_t row_stride = (size_t)gridDim.x * blockDim.y;
    for (size_t k = (size_t)blockIdx.x * blockDim.y + threadIdx.y; k < L; k += row_stride) {
        Acc sx = 0, sy = 0;
        if (C) {
            CxZ c = C[k * N + j];
            sx = c.x;
            sy = c.y;
        }
        const CxW *w = W + k * N;
#pragma unroll
        for (int i = 0; i < NMAX; i++) {
            if (i < N) {
                CxW wv = __ldg(w + i);
                Acc wx = (Acc)wv.x, wy = (Acc)wv.y;
                sx = fma(wx, ar[i], sx);
                sx = fma(-wy, ai[i], sx);
                sy = fma(wx, ai[i], sy);
                sy = fma(wy, ar[i], sy);
            }
        }
        CxZ o;
        o.x = (RealZ)sx;
        o.y = (RealZ)sy;
        Z[k * N + j] = o;
    }
}

template <typename RealZ, typename RealW>
static int launch_update_t(bkr_ctx *ctx, int N, const double2 *a, const void *C, const void *W, void *Z, const int *done)
{
    typedef typename CxT<RealZ>::type CxZ;
    typedef typename CxT<RealW>::type CxW;
    size_t L = (size_t)ctx->g.Vh * 3;
    int R = 256 / N;
    dim3 block(N, R);
    size_t nb = (L + R - 1) / R;
    unsigned grid = (unsigned)(nb < (size_t)BKR_NUM_SMS * 8 ? nb : (size_t)BKR_NUM_SMS * 8);
#define UPD_GO(NMAX) update_kernel<RealZ, RealW, NMAX><<<grid, block, 0, ctx->stream>>>(L, N, a, (const CxZ *)C, (const CxW *)W, (CxZ *)Z, done)
    if (N <= 4) UPD_GO(4);
    else if (N <= 8) UPD_GO(8);
    else if (N <= 16) UPD_GO(16);
    else if (N <= 24) UPD_GO(24);
    else UPD_GO(32);
#undef UPD_GO
    return bkr_check_launch(ctx);
}

int launch_block_update(bkr_ctx *ctx, int N, int precZ, int precW, const double2 *a, const void *C, const void *W, void *Z,
                        const int *done)
{
    if (precZ == BKR_F64 && precW == BKR_F64) return launch_update_t<double, double>(ctx, N, a, C, W, Z, done);
    if (precZ == BKR_F64 && precW == BKR_F32) return launch_update_t<double, float>(ctx, N, a, C, W, Z, done);
    if (precZ == BKR_F32 && precW == BKR_F32) return launch_update_t<float, float>(ctx, N, a, C, W, Z, done);
    // fp32 <- fp64: only Qhat = R C^-1 of the reliable update (Alg. 3 l.5), computed in fp64, rounded on store
    return launch_update_t<float, double>(ctx, N, a, C, W, Z, done);
}

// ------------------------------------------------------------------------------------------ per-column kernels
// blockDim = (N, R).  Deterministic: per-thread serial sums, fixed-order sum over the R rows of a CTA in
// shared memory, per-CTA partials, fixed-order final sum by col_finish_kernel.
template <typename Real>
__global__ void __launch_bounds__(256)
col_reduce_kernel(size_t L, int N, int mode, const typename CxT<Real>::type *__restrict__ X,
                  const typename CxT<Real>::type *__restrict__ Y, double *__restrict__ partials, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    __shared__ double red[256];
    if (done && *done) return;
    const int j = threadIdx.x;
    double s = 0.0;
    size_t row_stride = (size_t)gridDim.x * blockDim.y;
    for (size_t k = (size_t)blockIdx.x * blockDim.y + threadIdx.y; k < L; k += row_stride) {
        Cx x = X[k * N + j];
        double xr = x.x, xi = x.y;
        if (mode == 0) {
            s = fma(xr, xr, s);
            s = fma(xi, xi, s);
        } else {
            Cx y = Y[k * N + j];
            double yr = y.x, yi = y.y;
            if (mode == 1) {
                s = fma(xr, yr, s);
                s = fma(xi, yi, s);
            } else {
                double dr = xr - yr, di = xi - yi;
                s = fma(dr, dr, s);
                s = fma(di, di, s);
            }
        }
    }
    red[threadIdx.y * N + j] = s;
    __syncthreads();
    if (threadIdx.y == 0) {
        double t = 0.0;
        for (int r = 0; r < (int)blockDim.y; r++) t += red[r * N + j];
        partials[(size_t)blockIdx.x * N + j] = t;
    }
}

__global__ void col_finish_kernel(int N, int num_partials, const double *__restrict__ partials, double *__restrict__ out,
                                  const int *done)
{
    if (done && *done) return;
    int j = threadIdx.x;
    if (j >= N) return;
    double s = 0.0;
    for (int p = 0; p < num_partials; p++) s += partials[(size_t)p * N + j];
    out[j] = s;
}

int launch_col_reduce(bkr_ctx *ctx, int N, int prec, int mode, const void *X, const void *Y, double *out, const int *done)
{
    size_t L = (size_t)ctx->g.Vh * 3;
    int R = 256 / N;
    dim3 block(N, R);
    size_t nb = (L + R - 1) / R;
    unsigned grid = (unsigned)(nb < (size_t)BKR_NUM_SMS * 4 ? nb : (size_t)BKR_NUM_SMS * 4);
    BKR_TRY(ensure_partials(ctx, (size_t)BKR_NUM_SMS * 2 * BKR_MAX_N * BKR_MAX_N * sizeof(double2)));
    double *part = (double *)ctx->partials;
    if (prec == BKR_F64)
        col_reduce_kernel<double><<<grid, block, 0, ctx->stream>>>(L, N, mode, (const double2 *)X, (const double2 *)Y, part, done);
    else
        col_reduce_kernel<float><<<grid, block, 0, ctx->stream>>>(L, N, mode, (const float2 *)X, (const float2 *)Y, part, done);
    BKR_TRY(bkr_check_launch(ctx));
    col_finish_kernel<<<1, 32, 0, ctx->stream>>>(N, (int)grid, part, out, done);
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

// batched CG updates with per-column real coefficients (the "pseudo-block" baseline)
template <typename Real>
__global__ void __launch_bounds__(256)
cg_update_kernel(size_t L, int N, int mode, const double *__restrict__ coef, typename CxT<Real>::type *X,
                 const typename CxT<Real>::type *P, typename CxT<Real>::type *R, const typename CxT<Real>::type *Q,
                 const int *done)
{
    typedef typename CxT<Real>::type Cx;
    if (done && *done) return;
    const int j = threadIdx.x;
    const Real cf = (Real)coef[j];
    size_t row_stride = (size_t)gridDim.x * blockDim.y;
    for (size_t k = (size_t)blockIdx.x * blockDim.y + threadIdx.y; k < L; k += row_stride) {
        size_t o = k * N + j;
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
            const_cast<Cx *>(P)[o] = p;
        }
    }
}

int launch_cg_update(bkr_ctx *ctx, int N, int prec, int mode, const double *coef, void *X, const void *P, void *R,
                     const void *Q, const int *done)
{
    size_t L = (size_t)ctx->g.Vh * 3;
    int Rr = 256 / N;
    dim3 block(N, Rr);
    size_t nb = (L + Rr - 1) / Rr;
    unsigned grid = (unsigned)(nb < (size_t)BKR_NUM_SMS * 8 ? nb : (size_t)BKR_NUM_SMS * 8);
    if (prec == BKR_F64)
        cg_update_kernel<double><<<grid, block, 0, ctx->stream>>>(L, N, mode, coef, (double2 *)X, (const double2 *)P, (double2 *)R, (const double2 *)Q, done);
    else
        cg_update_kernel<float><<<grid, block, 0, ctx->stream>>>(L, N, mode, coef, (float2 *)X, (const float2 *)P, (float2 *)R, (const float2 *)Q, done);
    return bkr_check_launch(ctx);
}
