// Multi-BLAS on native blocks v[j][k] (N vectors of L = 3 Vh complex, row index k contiguous):
//   reduction multi-BLAS  K = X^dag Y          PAPER.md:272-299 (eq. 4)
//   streaming multi-BLAS  Z = C + W a          PAPER.md:245-270 (eq. 3; Alg. 1 l.8, l.10, l.11, Alg. 2 l.4)
// plus the per-column kernels of the CG baseline.  Both block kernels stream every vector element
// once, so memory traffic is linear in N.
//
// Arithmetic.  Both are tall-skinny complex GEMMs (inner or outer dimension N <= 32).
// On B200 the FP64 tensor path (DMMA m8n8k4) runs on the same pipe and at the same peak as DFMA (measured:
// 36.8 vs 36.7 TFLOP/s, no overlap), so it raises no ceiling; it is used because one DMMA replaces 8 DFMAs per
// lane and needs 2 operand registers for 8 FMAs, which removes the load/issue pressure that made the plain-FMA
// kernels latency bound.  A complex product is 4 real DMMAs.  All accumulation is fp64 whatever the storage
// precision.  Reductions finish in a fixed order (no floating-point atomics): results are bit-reproducible.
#include "common.cuh"

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1])
        : "d"(a), "d"(b));
}

template <typename Cx> __device__ __forceinline__ double2 ld_cx(const Cx *p)
{
    const Cx v = __ldg(p);
    return make_double2((double)v.x, (double)v.y);
}
template <typename Cx> __device__ __forceinline__ double2 ld_cx_stream(const Cx *p)
{
    const Cx v = __ldcs(p);
    return make_double2((double)v.x, (double)v.y);
}

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
// G = X^dag Y on 8 x 8 tiles of the N x N output.  A warp owns 8-row units of the blocks; per 4 rows and tile
// pair (ti, tj):  A[m][q] = X[8 ti + m][k + q] (8 x 4),  B[q][n] = Y[8 tj + n][k + q] (4 x 8), lane = 4 m + q
// loads one complex of X (and of Y unless X == Y) with one 16-byte load, and
//   Re G += Xr Yr + Xi Yi     Im G += Xr Yi - Xi Yr      (the two Im terms are kept apart, subtracted at the end).
// HERM: only pairs ti <= tj.  Otherwise blockIdx.y picks TIB i-tiles, all j-tiles.
static const int GRAM_WARPS = 8;
static const int GRAM_GRID = 2 * BKR_NUM_SMS;

template <typename Real, int NT, bool HERM, bool ALIAS, int TIB>
__global__ void __launch_bounds__(GRAM_WARPS * 32, NT <= 2 ? 2 : 1)
gram_kernel(size_t L, int N, const typename CxT<Real>::type *__restrict__ X,
            const typename CxT<Real>::type *__restrict__ Y, double2 *__restrict__ partials, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int NXT = HERM ? NT : TIB;                    // i-tiles this CTA touches
    constexpr int NP = HERM ? NT * (NT + 1) / 2 : TIB * NT; // tile pairs this CTA accumulates
    __shared__ double2 red[BKR_MAX_N * BKR_MAX_N];
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int m = lane >> 2, q = lane & 3;
    const int ti0 = HERM ? 0 : blockIdx.y * TIB;

    const Cx *px[NXT], *py[NT];
#pragma unroll
    for (int t = 0; t < NXT; t++) {
        const int i = 8 * (ti0 + t) + m;
        px[t] = i < N ? X + (size_t)i * L + q : nullptr;
    }
#pragma unroll
    for (int t = 0; t < NT; t++) {
        const int j = 8 * t + m;
        py[t] = j < N ? Y + (size_t)j * L + q : nullptr;
    }

    double acc[NP][3][2];
#pragma unroll
    for (int p = 0; p < NP; p++)
#pragma unroll
        for (int c = 0; c < 3; c++) acc[p][c][0] = acc[p][c][1] = 0.0;

    // a unit = NS 4-row steps (8 rows for N <= 16, 4 rows above: fewer fragment registers next to more accumulators)
    constexpr int NS = NT <= 2 ? 2 : 1;
    const size_t units = L / (4 * NS); // L is a multiple of 8 for even extents >= 4
    const size_t u0 = units * blockIdx.x / gridDim.x, u1 = units * (blockIdx.x + 1) / gridDim.x;

    double2 xc[NS][NXT], yc[NS][ALIAS ? 1 : NT]; // current fragments
    double2 xn[NS][NXT], yn[NS][ALIAS ? 1 : NT]; // prefetched
    auto load = [&](double2(&xf)[NS][NXT], double2(&yf)[NS][ALIAS ? 1 : NT], size_t u) {
        const size_t k = u * 4 * NS;
#pragma unroll
        for (int s = 0; s < NS; s++) {
#pragma unroll
            for (int t = 0; t < NXT; t++) xf[s][t] = px[t] ? ld_cx(px[t] + k + 4 * s) : make_double2(0.0, 0.0);
            if (!ALIAS) {
#pragma unroll
                for (int t = 0; t < NT; t++) yf[s][t] = py[t] ? ld_cx(py[t] + k + 4 * s) : make_double2(0.0, 0.0);
            }
        }
    };
    size_t u = u0 + warp;
    if (u < u1) load(xc, yc, u);
    for (; u < u1; u += GRAM_WARPS) {
        const bool more = u + GRAM_WARPS < u1;
        if (more) load(xn, yn, u + GRAM_WARPS);
#pragma unroll
        for (int s = 0; s < NS; s++) {
            int p = 0;
#pragma unroll
            for (int ti = 0; ti < NXT; ti++) {
#pragma unroll
                for (int tj = HERM ? ti : 0; tj < NT; tj++, p++) {
                    const double2 a = xc[s][ti];
                    const double2 b = ALIAS ? xc[s][tj] : yc[s][tj];
                    dmma(acc[p][0], a.x, b.x);
                    dmma(acc[p][0], a.y, b.y);
                    dmma(acc[p][1], a.x, b.y);
                    dmma(acc[p][2], a.y, b.x);
                }
            }
        }
        if (more) {
#pragma unroll
            for (int s = 0; s < NS; s++) {
#pragma unroll
                for (int t = 0; t < NXT; t++) xc[s][t] = xn[s][t];
                if (!ALIAS) {
#pragma unroll
                    for (int t = 0; t < NT; t++) yc[s][t] = yn[s][t];
                }
            }
        }
    }

    // fixed-order reduction over the warps of the CTA, then one partial per CTA
    for (int o = threadIdx.x; o < N * N; o += blockDim.x) red[o] = make_double2(0.0, 0.0);
    __syncthreads();
    for (int w = 0; w < GRAM_WARPS; w++) {
        if (warp == w) {
            int p = 0;
#pragma unroll
            for (int ti = 0; ti < NXT; ti++) {
#pragma unroll
                for (int tj = HERM ? ti : 0; tj < NT; tj++, p++) {
#pragma unroll
                    for (int r = 0; r < 2; r++) {
                        const int i = 8 * (ti0 + ti) + m, j = 8 * tj + 2 * q + r;
                        if (i < N && j < N) {
                            double2 v = red[i * N + j];
                            v.x += acc[p][0][r];
                            v.y += acc[p][1][r] - acc[p][2][r];
                            red[i * N + j] = v;
                        }
                    }
                }
            }
        }
        __syncthreads();
    }
    const int row0 = 8 * ti0, row1 = HERM ? N : min(N, 8 * (ti0 + TIB));
    for (int o = row0 * N + threadIdx.x; o < row1 * N; o += blockDim.x)
        partials[(size_t)blockIdx.x * N * N + o] = red[o];
}

template <typename Real, int NT>
static void gram_go(bkr_ctx *ctx, size_t L, int N, const void *X, const void *Y, int hermitian, int grid, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int TIB = NT > 2 ? 2 : NT;
    const Cx *x = (const Cx *)X, *y = (const Cx *)Y;
    if (hermitian) {
        if (X == Y)
            gram_kernel<Real, NT, true, true, NT><<<grid, GRAM_WARPS * 32, 0, ctx->stream>>>(L, N, x, y, ctx->partials, done);
        else
            gram_kernel<Real, NT, true, false, NT><<<grid, GRAM_WARPS * 32, 0, ctx->stream>>>(L, N, x, y, ctx->partials, done);
    } else {
        dim3 g2(grid, (NT + TIB - 1) / TIB);
        gram_kernel<Real, NT, false, false, TIB><<<g2, GRAM_WARPS * 32, 0, ctx->stream>>>(L, N, x, y, ctx->partials, done);
    }
}

int launch_gram_partials(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, int *num_partials,
                         const int *done)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    int grid = GRAM_GRID;
    if (N > 16) grid = BKR_NUM_SMS; // one CTA per SM above two tiles (launch bounds of gram_kernel)
    if ((size_t)grid * GRAM_WARPS > L / 8) grid = (int)((L / 8 + GRAM_WARPS - 1) / GRAM_WARPS);
    BKR_TRY(ensure_partials(ctx, (size_t)GRAM_GRID * BKR_MAX_N * BKR_MAX_N * sizeof(double2)));
    const int NT = (N + 7) / 8;
#define GRAM_NT(Real)                                                                 \
    switch (NT) {                                                                     \
    case 1: gram_go<Real, 1>(ctx, L, N, X, Y, hermitian, grid, done); break;          \
    case 2: gram_go<Real, 2>(ctx, L, N, X, Y, hermitian, grid, done); break;          \
    case 3: gram_go<Real, 3>(ctx, L, N, X, Y, hermitian, grid, done); break;          \
    default: gram_go<Real, 4>(ctx, L, N, X, Y, hermitian, grid, done); break;         \
    }
    if (prec == BKR_F64) {
        GRAM_NT(double)
    } else {
        GRAM_NT(float)
    }
#undef GRAM_NT
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
// Z = C + W a  as  D(8 rows x 8 j) += A(8 rows x 4 i) B(4 i x 8 j):  A[m][q] = W[4 is + q][k + m] (one 16-byte load
// per lane gives Re and Im), B[q][n] = a[4 is + q][8 tj + n] from shared memory in fragment order (one
// conflict-free 8-byte load per lane), and
//   Re Z += Wr ar - Wi ai      Im Z += Wr ai + Wi ar.
// A warp owns MT = 2 row tiles (16 rows) per iteration: 2 NIS loads of W, 16 NIS NTJ DMMAs, then C is read and Z
// written as 16-byte pieces, 8 consecutive rows of 4 vectors per instruction.
static const int UPD_WARPS = 8;
static const int UPD_MT = 2;

template <typename Cx> __device__ __forceinline__ void st_cx(Cx *p, double re, double im);
template <> __device__ __forceinline__ void st_cx<double2>(double2 *p, double re, double im) { *p = make_double2(re, im); }
template <> __device__ __forceinline__ void st_cx<float2>(float2 *p, double re, double im)
{
    *p = make_float2((float)re, (float)im);
}

template <typename RealZ, typename RealW, int NTJ, int NIS, bool HASC>
__global__ void __launch_bounds__(UPD_WARPS * 32, 2)
update_kernel(size_t L, int N, const double2 *__restrict__ a, const typename CxT<RealZ>::type *C,
              const typename CxT<RealW>::type *__restrict__ W, typename CxT<RealZ>::type *Z, const int *done)
{
    typedef typename CxT<RealZ>::type CxZ;
    typedef typename CxT<RealW>::type CxW;
    __shared__ double bre[NIS * NTJ * 32], bim[NIS * NTJ * 32], bnim[NIS * NTJ * 32];
    if (done && *done) return;
    for (int idx = threadIdx.x; idx < NIS * NTJ * 32; idx += blockDim.x) {
        const int ln = idx & 31, f = idx >> 5;
        const int is = f / NTJ, tj = f % NTJ;
        const int i = 4 * is + (ln & 3), j = 8 * tj + (ln >> 2);
        const double2 v = (i < N && j < N) ? a[i * N + j] : make_double2(0.0, 0.0);
        bre[idx] = v.x;
        bim[idx] = v.y;
        bnim[idx] = -v.y;
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int m = lane >> 2, q = lane & 3;
    const size_t units = L / 8;
    const size_t gw = (size_t)blockIdx.x * UPD_WARPS + warp, GW = (size_t)gridDim.x * UPD_WARPS;

    for (size_t u = UPD_MT * gw; u < units; u += UPD_MT * GW) {
        double2 wf[UPD_MT][NIS];
#pragma unroll
        for (int mt = 0; mt < UPD_MT; mt++) {
            const bool rowok = u + mt < units;
            const size_t k = (u + mt) * 8 + m;
#pragma unroll
            for (int is = 0; is < NIS; is++) {
                const int i = 4 * is + q;
                wf[mt][is] = (rowok && i < N) ? ld_cx_stream(W + (size_t)i * L + k) : make_double2(0.0, 0.0);
            }
        }
        double zre[UPD_MT][NTJ][2], zim[UPD_MT][NTJ][2];
#pragma unroll
        for (int mt = 0; mt < UPD_MT; mt++)
#pragma unroll
            for (int tj = 0; tj < NTJ; tj++) zre[mt][tj][0] = zre[mt][tj][1] = zim[mt][tj][0] = zim[mt][tj][1] = 0.0;
#pragma unroll
        for (int is = 0; is < NIS; is++) {
#pragma unroll
            for (int tj = 0; tj < NTJ; tj++) {
                const int f = (is * NTJ + tj) * 32 + lane;
                const double ar = bre[f], ai = bim[f], nai = bnim[f];
#pragma unroll
                for (int mt = 0; mt < UPD_MT; mt++) {
                    dmma(zre[mt][tj], wf[mt][is].x, ar);
                    dmma(zre[mt][tj], wf[mt][is].y, nai);
                    dmma(zim[mt][tj], wf[mt][is].x, ai);
                    dmma(zim[mt][tj], wf[mt][is].y, ar);
                }
            }
        }
#pragma unroll
        for (int mt = 0; mt < UPD_MT; mt++) {
            if (u + mt < units) {
                const size_t k = (u + mt) * 8 + m;
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++) {
#pragma unroll
                    for (int r = 0; r < 2; r++) {
                        const int j = 8 * tj + 2 * q + r;
                        if (j < N) {
                            double re = zre[mt][tj][r], im = zim[mt][tj][r];
                            if (HASC) {
                                const double2 c = ld_cx_stream(C + (size_t)j * L + k);
                                re += c.x;
                                im += c.y;
                            }
                            st_cx<CxZ>(Z + (size_t)j * L + k, re, im);
                        }
                    }
                }
            }
        }
    }
}

template <typename RealZ, typename RealW, int NTJ, int NIS>
static void update_go(bkr_ctx *ctx, size_t L, int N, const double2 *a, const void *C, const void *W, void *Z, const int *done)
{
    typedef typename CxT<RealZ>::type CxZ;
    typedef typename CxT<RealW>::type CxW;
    size_t iters = (L / 8 + UPD_MT * UPD_WARPS - 1) / (UPD_MT * UPD_WARPS);
    unsigned grid = (unsigned)(iters < (size_t)BKR_NUM_SMS * 2 ? iters : (size_t)BKR_NUM_SMS * 2);
    if (C)
        update_kernel<RealZ, RealW, NTJ, NIS, true><<<grid, UPD_WARPS * 32, 0, ctx->stream>>>(L, N, a, (const CxZ *)C, (const CxW *)W, (CxZ *)Z, done);
    else
        update_kernel<RealZ, RealW, NTJ, NIS, false><<<grid, UPD_WARPS * 32, 0, ctx->stream>>>(L, N, a, nullptr, (const CxW *)W, (CxZ *)Z, done);
}

template <typename RealZ, typename RealW>
static int launch_update_t(bkr_ctx *ctx, int N, const double2 *a, const void *C, const void *W, void *Z, const int *done)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    const int NIS = (N + 3) / 4;
#define UPD_GO(NTJ_, NIS_) update_go<RealZ, RealW, NTJ_, NIS_>(ctx, L, N, a, C, W, Z, done); break
    switch (NIS) {
    case 1: UPD_GO(1, 1);
    case 2: UPD_GO(1, 2);
    case 3: UPD_GO(2, 3);
    case 4: UPD_GO(2, 4);
    case 5: UPD_GO(3, 5);
    case 6: UPD_GO(3, 6);
    case 7: UPD_GO(4, 7);
    default: UPD_GO(4, 8);
    }
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
    BKR_TRY(ensure_partials(ctx, (size_t)GRAM_GRID * BKR_MAX_N * BKR_MAX_N * sizeof(double2)));
    double *part = (double *)ctx->partials;
    dim3 grid(gx, N);
    if (prec == BKR_F64)
        col_reduce_kernel<double><<<grid, COL_THREADS, 0, ctx->stream>>>(L, mode, (const double2 *)X, (const double2 *)Y, part, done);
    else
        col_reduce_kernel<float><<<grid, COL_THREADS, 0, ctx->stream>>>(L, mode, (const float2 *)X, (const float2 *)Y, part, done);
    BKR_TRY(bkr_check_launch(ctx));
    col_finish_kernel<<<1, 32, 0, ctx->stream>>>(N, (int)gx, part, out, done);
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
