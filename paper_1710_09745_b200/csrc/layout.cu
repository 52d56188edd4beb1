// Field and link layouts ("reordering the vector and link fields to achieve memory
// coalescing"; PAPER.md:212-216 composite fields).  See DESIGN.md section 5.
//
//   native block  v[e][a][j]     : L x N row-major, the N rhs of a (site, colour) row contiguous, so that a
//                                  neighbour gather in the stencil is one contiguous 6*N*w-byte read and the
//                                  block BLAS sees plain row-major tall-skinny matrices.
//   native links  L[d][el][e]    : d = (type*4 + mu)*2 + parity, el = 3*row + col; complex SoA over sites, so
//                                  the lanes of a warp that work on different sites read contiguous 16 B
//                                  (fp64) / 8 B (fp32) pieces and lanes on the same site broadcast.
#include "common.cuh"

__global__ void pack_links_kernel(Geom g, const double2 *__restrict__ fat, const double2 *__restrict__ lng,
                                  double2 *__restrict__ out64, float2 *__restrict__ out32)
{
    // one thread per (type, mu, site, el)
    size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t total = (size_t)2 * 4 * g.V * 9;
    if (tid >= total) return;
    int el = (int)(tid % 9);
    size_t r = tid / 9;
    int s = (int)(r % g.V);
    r /= g.V;
    int mu = (int)(r % 4);
    int type = (int)(r / 4);
    int x = s % g.X[0];
    int q = s / g.X[0];
    int y = q % g.X[1];
    q /= g.X[1];
    int z = q % g.X[2];
    int t = q / g.X[2];
    int parity = (x + y + z + t) & 1;
    int e = s >> 1;
    const double2 *src = (type == 0 ? fat : lng) + ((size_t)mu * g.V + s) * 9 + el;
    double2 u = *src;
    size_t o = ((size_t)(((type * 4 + mu) * 2 + parity) * 9 + el)) * g.Vh + e;
    out64[o] = u;
    if (out32) out32[o] = make_float2((float)u.x, (float)u.y);
}

int launch_pack_links(bkr_ctx *ctx, const double2 *fat, const double2 *lng, double2 *out64, float2 *out32)
{
    size_t total = (size_t)2 * 4 * ctx->g.V * 9;
    unsigned blocks = (unsigned)((total + 255) / 256);
    pack_links_kernel<<<blocks, 256, 0, ctx->stream>>>(ctx->g, fat, lng, out64, out32);
    return bkr_check_launch(ctx);
}

// canonical [j][e][a] fp64  <->  native [e][a][j].  A 32 x 32 shared-memory transpose over (row k, rhs j)
// keeps both sides coalesced.
template <typename Real, bool PACK>
__global__ void transpose_kernel(size_t L, int N, const double2 *__restrict__ canon_in, double2 *__restrict__ canon_out,
                                 const typename CxT<Real>::type *__restrict__ nat_in,
                                 typename CxT<Real>::type *__restrict__ nat_out)
{
    typedef typename CxT<Real>::type Cx;
    __shared__ double2 tile[32][33];
    size_t k0 = (size_t)blockIdx.x * 32;
    int tx = threadIdx.x, ty = threadIdx.y; // 32 x 8
    if (PACK) {
        for (int j = ty; j < N; j += 8) {
            size_t k = k0 + tx;
            if (k < L) tile[j][tx] = canon_in[(size_t)j * L + k];
        }
        __syncthreads();
        for (int kk = ty; kk < 32; kk += 8) {
            size_t k = k0 + kk;
            if (k < L && tx < N) {
                double2 v = tile[tx][kk];
                Cx o;
                o.x = (Real)v.x;
                o.y = (Real)v.y;
                nat_out[k * N + tx] = o;
            }
        }
    } else {
        for (int kk = ty; kk < 32; kk += 8) {
            size_t k = k0 + kk;
            if (k < L && tx < N) {
                Cx v = nat_in[k * N + tx];
                tile[tx][kk] = make_double2((double)v.x, (double)v.y);
            }
        }
        __syncthreads();
        for (int j = ty; j < N; j += 8) {
            size_t k = k0 + tx;
            if (k < L) canon_out[(size_t)j * L + k] = tile[j][tx];
        }
    }
}

int launch_pack(bkr_ctx *ctx, int N, int prec, const double2 *canonical, void *native)
{
    size_t L = (size_t)ctx->g.Vh * 3;
    dim3 block(32, 8);
    unsigned blocks = (unsigned)((L + 31) / 32);
    if (prec == BKR_F64)
        transpose_kernel<double, true><<<blocks, block, 0, ctx->stream>>>(L, N, canonical, nullptr, nullptr, (double2 *)native);
    else
        transpose_kernel<float, true><<<blocks, block, 0, ctx->stream>>>(L, N, canonical, nullptr, nullptr, (float2 *)native);
    return bkr_check_launch(ctx);
}

int launch_unpack(bkr_ctx *ctx, int N, int prec, const void *native, double2 *canonical)
{
    size_t L = (size_t)ctx->g.Vh * 3;
    dim3 block(32, 8);
    unsigned blocks = (unsigned)((L + 31) / 32);
    if (prec == BKR_F64)
        transpose_kernel<double, false><<<blocks, block, 0, ctx->stream>>>(L, N, nullptr, canonical, (const double2 *)native, nullptr);
    else
        transpose_kernel<float, false><<<blocks, block, 0, ctx->stream>>>(L, N, nullptr, canonical, (const float2 *)native, nullptr);
    return bkr_check_launch(ctx);
}

// precision conversion of a native block (mixed-precision solver: Q-hat is stored in fp32)
template <typename Src, typename Dst>
__global__ void convert_kernel(size_t n, const Src *__restrict__ src, Dst *__restrict__ dst, const int *done)
{
    if (done && *done) return;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t stride = (size_t)gridDim.x * blockDim.x;
    for (; i < n; i += stride) {
        Src v = src[i];
        Dst o;
        o.x = v.x;
        o.y = v.y;
        dst[i] = o;
    }
}

int launch_convert(bkr_ctx *ctx, size_t n, int sp, const void *src, int dp, void *dst, const int *done)
{
    unsigned blocks = (unsigned)((n + 255) / 256);
    if (blocks > BKR_NUM_SMS * 16) blocks = BKR_NUM_SMS * 16;
    if (sp == BKR_F64 && dp == BKR_F32)
        convert_kernel<double2, float2><<<blocks, 256, 0, ctx->stream>>>(n, (const double2 *)src, (float2 *)dst, done);
    else if (sp == BKR_F32 && dp == BKR_F64)
        convert_kernel<float2, double2><<<blocks, 256, 0, ctx->stream>>>(n, (const float2 *)src, (double2 *)dst, done);
    else if (sp == BKR_F64)
        convert_kernel<double2, double2><<<blocks, 256, 0, ctx->stream>>>(n, (const double2 *)src, (double2 *)dst, done);
    else
        convert_kernel<float2, float2><<<blocks, 256, 0, ctx->stream>>>(n, (const float2 *)src, (float2 *)dst, done);
    return bkr_check_launch(ctx);
}
