// Field and link layouts ("reordering the vector and link fields to achieve memory
// coalescing"; PAPER.md:212-216 composite fields).  See DESIGN.md section 5.
//
//   native block  v[j][a][e]     : N vectors of L = 3 Vh complex each, stored one after the other ("composite
//                                  field" whose components are contiguous views); inside a
//                                  vector the three colour planes are SoA over the even-odd site index, so a
//                                  warp of 32 consecutive sites (stencil) or rows (block BLAS) reads 512
//                                  contiguous bytes per instruction in fp64.
//   native links  Wt[p][tile][h][el][lane] : gather form, tile-major (see pack_links_kernel below).
#include "common.cuh"

// Gather-form links.  For the output site x of parity p (even-odd index e) and hop h = 0..15 in the order of
// common.cuh (BKR_HOP_*: direction mu, type 0 fat / 1 long = hop length 1 / 3, dir 0 forward / 1 backward) the
// stencil needs the matrix
//     W_h(x) = U_mu(x)                (forward)         W_h(x) = - U_mu(x - hop mu)^dagger   (backward)
// so that (D in)(x) = sum_h W_h(x) in(nbr_h(x))  (eq. 2).  Storing W per output site makes the
// whole link stream of a tile of BKR_LINK_TILE consecutive sites ONE contiguous chunk
//     Wt[p][tile][h][el][lane],   el = 3*row + col,  lane = e % BKR_LINK_TILE,
// which the stencil kernel streams with 1-D TMA bulk copies, one per hop.  Bytes read per call are unchanged
// (16 matrices per output site); storage is twice the canonical links (each U appears as a forward and as a
// backward copy).
__global__ void pack_links_kernel(Geom g, int ntiles, const double2 *__restrict__ fat, const double2 *__restrict__ lng,
                                  double2 *__restrict__ out64, float2 *__restrict__ out32)
{
    // one thread per (parity, e, h)
    const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t padded = (size_t)ntiles * BKR_LINK_TILE;
    if (tid >= 2 * padded * 16) return;
    const int h = (int)(tid % 16);
    const size_t r = tid / 16;
    const int e = (int)(r % padded);
    const int parity = (int)(r / padded);
    const int mu = BKR_HOP_MU(h), type = BKR_HOP_LONG(h), dir = BKR_HOP_BACK(h);
    const size_t base = ((((size_t)parity * ntiles + e / BKR_LINK_TILE) * 16 + h) * 9) * BKR_LINK_TILE + e % BKR_LINK_TILE;
    double2 w[9];
    if (e < g.Vh) {
        int s = 2 * e;
        int c[4];
        const int x0 = s % g.X[0];
        int q = s / g.X[0];
        c[1] = q % g.X[1];
        q /= g.X[1];
        c[2] = q % g.X[2];
        c[3] = q / g.X[2];
        c[0] = x0 + ((c[1] + c[2] + c[3] + parity) & 1);
        s = s - x0 + c[0];
        const int stride[4] = {1, g.X[0], g.X[0] * g.X[1], g.X[0] * g.X[1] * g.X[2]};
        const double2 *src = (type == 0 ? fat : lng) + (size_t)mu * g.V * 9;
        if (dir == 0) {
            for (int el = 0; el < 9; el++) w[el] = src[(size_t)s * 9 + el];
        } else {
            const int hop = type ? 3 : 1;
            int cb = c[mu] - hop;
            if (cb < 0) cb += g.X[mu];
            const int sb = s + (cb - c[mu]) * stride[mu];
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++) {
                    const double2 u = src[(size_t)sb * 9 + b * 3 + a];
                    w[a * 3 + b] = make_double2(-u.x, u.y); // -conj(U_ba)
                }
        }
    } else {
        for (int el = 0; el < 9; el++) w[el] = make_double2(0.0, 0.0);
    }
    for (int el = 0; el < 9; el++) {
        const size_t o = base + (size_t)el * BKR_LINK_TILE;
        if (out64) out64[o] = w[el];
        if (out32) out32[o] = make_float2((float)w[el].x, (float)w[el].y);
    }
}

int launch_pack_links(bkr_ctx *ctx, const double2 *fat, const double2 *lng, double2 *out64, float2 *out32)
{
    const int ntiles = link_tiles(ctx->g);
    size_t total = (size_t)2 * ntiles * BKR_LINK_TILE * 16;
    unsigned blocks = (unsigned)((total + 255) / 256);
    pack_links_kernel<<<blocks, 256, 0, ctx->stream>>>(ctx->g, ntiles, fat, lng, out64, out32);
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
