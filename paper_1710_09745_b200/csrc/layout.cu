// Field and link layouts ("reordering the vector and link fields to achieve memory
// coalescing"; PAPER.md:212-216 composite fields).  See DESIGN.md section 5.
//
//   native block  v[j][a][e]     : N vectors of L = 3 Vh complex each, stored one after the other ("composite
//                                  field" whose components are contiguous views); inside a
//                                  vector the three colour planes are SoA over the even-odd site index, so a
//                                  warp of 32 consecutive sites (stencil) or rows (block BLAS) reads 512
//                                  contiguous bytes per instruction in fp64.
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

// canonical [j][e][a] fp64  <->  native [j][a][e]: a 3 x Vh transpose per rhs.  One thread per (e, j); the
// native side is coalesced (32 consecutive sites of one plane per warp instruction), the canonical side reads or
// writes 48 contiguous bytes per thread.  Not on the hot path (boundary of the solve calls only).
template <typename Real, bool PACK>
__global__ void transpose_kernel(size_t Vh, int N, const double2 *__restrict__ canon_in, double2 *__restrict__ canon_out,
                                 const typename CxT<Real>::type *__restrict__ nat_in,
                                 typename CxT<Real>::type *__restrict__ nat_out)
{
    typedef typename CxT<Real>::type Cx;
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y;
    if (e >= Vh) return;
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const size_t ic = ((size_t)j * Vh + e) * 3 + a, in = ((size_t)j * 3 + a) * Vh + e;
        if (PACK) {
            const double2 v = canon_in[ic];
            Cx o;
            o.x = (Real)v.x;
            o.y = (Real)v.y;
            nat_out[in] = o;
        } else {
            const Cx v = nat_in[in];
            canon_out[ic] = make_double2((double)v.x, (double)v.y);
        }
    }
}

int launch_pack(bkr_ctx *ctx, int N, int prec, const double2 *canonical, void *native)
{
    size_t Vh = (size_t)ctx->g.Vh;
    dim3 grid((unsigned)((Vh + 255) / 256), N);
    if (prec == BKR_F64)
        transpose_kernel<double, true><<<grid, 256, 0, ctx->stream>>>(Vh, N, canonical, nullptr, nullptr, (double2 *)native);
    else
        transpose_kernel<float, true><<<grid, 256, 0, ctx->stream>>>(Vh, N, canonical, nullptr, nullptr, (float2 *)native);
    return bkr_check_launch(ctx);
}

int launch_unpack(bkr_ctx *ctx, int N, int prec, const void *native, double2 *canonical)
{
    size_t Vh = (size_t)ctx->g.Vh;
    dim3 grid((unsigned)((Vh + 255) / 256), N);
    if (prec == BKR_F64)
        transpose_kernel<double, false><<<grid, 256, 0, ctx->stream>>>(Vh, N, nullptr, canonical, (const double2 *)native, nullptr);
    else
        transpose_kernel<float, false><<<grid, 256, 0, ctx->stream>>>(Vh, N, nullptr, canonical, (const float2 *)native, nullptr);
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
