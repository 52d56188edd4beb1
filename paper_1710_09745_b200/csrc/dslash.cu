// Multi-rhs improved-staggered stencil ("Dslash"), PAPER.md:95-101 (eq. 2) and PAPER.md:218-232.
//
//   out(x) = sum_mu [ F_mu(x) in(x+mu) - F_mu(x-mu)^dag in(x-mu) + K_mu(x) in(x+3mu) - K_mu(x-3mu)^dag in(x-3mu) ]
//   optional epilogue  out = a * xp - out   (second half of M = 4 m^2 - D_eo D_oe)
//
// Mapping.  One thread = one output site x T right-hand sides (register tile, the
// paper's "register tiling" PAPER.md:232); threadIdx.y = rhs group g (rhs g*T .. g*T+T-1), so the G = ceil(N/T)
// warps that work on the same 32 sites sit in one CTA and the second..G-th read of a link hits L1 (the paper's
// "cache tiling").  With the SoA layouts v[j][a][e] and L[d][el][e] every load instruction of a
// warp reads 32 consecutive sites of one plane: 512 contiguous bytes in fp64.  Each link matrix is held in
// registers (18 reals) and reused for the T vectors; links are read with evict-first hints (used once per call),
// results are written with streaming stores, neighbour vectors use the default policy so that the x/y reuse is
// served by L1 and the z/t reuse by L2.
//
// Per site and rhs: 16 x 36 = 576 FMAs (1152 flop; the paper counts 1146).  At N = 16 in fp64 the
// three per-SM budgets are within 25 % of each other (HBM 166 clk/site, FP64 pipe 144, L1->register 132), see
// DESIGN.md section 7.
#include "common.cuh"

template <typename Real> struct LdSt;
template <> struct LdSt<double> {
    static __device__ __forceinline__ double2 link(const double2 *p) { return __ldcs(p); }
    static __device__ __forceinline__ double2 vec(const double2 *p) { return __ldg(p); }
    static __device__ __forceinline__ void out(double2 *p, double2 v) { __stcs(p, v); }
};
template <> struct LdSt<float> {
    static __device__ __forceinline__ float2 link(const float2 *p) { return __ldcs(p); }
    static __device__ __forceinline__ float2 vec(const float2 *p) { return __ldg(p); }
    static __device__ __forceinline__ void out(float2 *p, float2 v) { __stcs(p, v); }
};

// acc[i] (+)= U v_i  (DAG = false)   or   acc[i] -= U^dag v_i  (DAG = true), i < T.
// Column by column: for input colour b only U[.][b] (or, daggered, U[b][.]) and one complex per rhs are live, so the
// register tile is 6 T accumulators + 6 link reals + the loads in flight.
template <typename Real, int T, bool EXACT, bool DAG>
__device__ __forceinline__ void hop(Real (&acc)[T][6], const typename CxT<Real>::type *__restrict__ U, size_t Vh,
                                    const typename CxT<Real>::type *__restrict__ vin, int nvalid)
{
    typedef typename CxT<Real>::type Cx;
#pragma unroll
    for (int b = 0; b < 3; b++) {
        Cx u[3]; // forward: column b of U;  backward: row b of U (conjugated below)
#pragma unroll
        for (int a = 0; a < 3; a++) u[a] = LdSt<Real>::link(U + (DAG ? b * 3 + a : a * 3 + b) * Vh);
#pragma unroll
        for (int i = 0; i < T; i++) {
            if (EXACT || i < nvalid) {
                const Cx v = LdSt<Real>::vec(vin + (size_t)(i * 3 + b) * Vh);
#pragma unroll
                for (int a = 0; a < 3; a++) {
                    if (!DAG) { // + U_ab v_b
                        acc[i][2 * a] = fma(u[a].x, v.x, acc[i][2 * a]);
                        acc[i][2 * a] = fma(-u[a].y, v.y, acc[i][2 * a]);
                        acc[i][2 * a + 1] = fma(u[a].x, v.y, acc[i][2 * a + 1]);
                        acc[i][2 * a + 1] = fma(u[a].y, v.x, acc[i][2 * a + 1]);
                    } else { // - conj(U_ba) v_b
                        acc[i][2 * a] = fma(-u[a].x, v.x, acc[i][2 * a]);
                        acc[i][2 * a] = fma(-u[a].y, v.y, acc[i][2 * a]);
                        acc[i][2 * a + 1] = fma(-u[a].x, v.y, acc[i][2 * a + 1]);
                        acc[i][2 * a + 1] = fma(u[a].y, v.x, acc[i][2 * a + 1]);
                    }
                }
            }
        }
    }
}

template <typename Real, int T, bool EXACT, int BS, int MINB>
__global__ void __launch_bounds__(BS, MINB)
dslash_kernel(Geom g, int parity, int N, const typename CxT<Real>::type *__restrict__ links,
              const typename CxT<Real>::type *__restrict__ in, typename CxT<Real>::type *__restrict__ out,
              const typename CxT<Real>::type *__restrict__ xp, Real a, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    if (done && *done) return;
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= g.Vh) return;
    const int j0 = threadIdx.y * T;
    const int nvalid = N - j0; // rhs this thread owns (>= 1 by construction of the launch; may be < T)
    // coordinates of the output site (parity, e): lexicographic s = x + X(y + Y(z + Z t)), e = s / 2
    int s = 2 * e;
    int c[4];
    const int x0 = s % g.X[0];
    int r = s / g.X[0];
    c[1] = r % g.X[1];
    r /= g.X[1];
    c[2] = r % g.X[2];
    c[3] = r / g.X[2];
    c[0] = x0 + ((c[1] + c[2] + c[3] + parity) & 1);
    s = s - x0 + c[0];
    const int stride[4] = {1, g.X[0], g.X[0] * g.X[1], g.X[0] * g.X[1] * g.X[2]};
    const size_t Vh = g.Vh;

    Real acc[T][6];
#pragma unroll
    for (int i = 0; i < T; i++)
#pragma unroll
        for (int k = 0; k < 6; k++) acc[i][k] = (Real)0;

    const Cx *vin = in + (size_t)j0 * 3 * Vh;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
#pragma unroll
        for (int type = 0; type < 2; type++) {
            const int h = type ? 3 : 1;
            int cf = c[mu] + h;
            if (cf >= g.X[mu]) cf -= g.X[mu];
            int cb = c[mu] - h;
            if (cb < 0) cb += g.X[mu];
            const int ef = (s + (cf - c[mu]) * stride[mu]) >> 1;
            const int eb = (s + (cb - c[mu]) * stride[mu]) >> 1;
            // forward: link leaving x (parity of x), vector at x + h mu
            hop<Real, T, EXACT, false>(acc, links + (size_t)(((type * 4 + mu) * 2 + parity) * 9) * Vh + e, Vh, vin + ef,
                                       nvalid);
            // backward: link leaving x - h mu (opposite parity), daggered, vector at x - h mu
            hop<Real, T, EXACT, true>(acc, links + (size_t)(((type * 4 + mu) * 2 + (1 - parity)) * 9) * Vh + eb, Vh,
                                      vin + eb, nvalid);
        }
    }

    Cx *vout = out + (size_t)j0 * 3 * Vh + e;
    const Cx *vxp = xp ? xp + (size_t)j0 * 3 * Vh + e : nullptr;
#pragma unroll
    for (int i = 0; i < T; i++) {
        if (EXACT || i < nvalid) {
#pragma unroll
            for (int cc = 0; cc < 3; cc++) {
                Cx o;
                o.x = acc[i][2 * cc];
                o.y = acc[i][2 * cc + 1];
                if (vxp) {
                    const Cx p = LdSt<Real>::vec(vxp + (size_t)(i * 3 + cc) * Vh);
                    o.x = fma(a, p.x, -o.x);
                    o.y = fma(a, p.y, -o.y);
                }
                LdSt<Real>::out(vout + (size_t)(i * 3 + cc) * Vh, o);
            }
        }
    }
}

// T rhs per thread, G = ceil(N / T) rhs groups per CTA, BS sites per CTA
template <typename Real, int T, int BS, int MINB>
static int launch_t(bkr_ctx *ctx, int parity, int N, const void *in, void *out, const void *xp, double a, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    const Cx *links = sizeof(Real) == 8 ? (const Cx *)ctx->links64 : (const Cx *)ctx->links32;
    const int G = (N + T - 1) / T;
    dim3 block(BS / G >= 32 ? (BS / G) / 32 * 32 : 32, G);
    unsigned blocks = (unsigned)((ctx->g.Vh + block.x - 1) / block.x);
    if (N % T == 0)
        dslash_kernel<Real, T, true, BS, MINB><<<blocks, block, 0, ctx->stream>>>(ctx->g, parity, N, links, (const Cx *)in,
                                                                                  (Cx *)out, (const Cx *)xp, (Real)a, done);
    else
        dslash_kernel<Real, T, false, BS, MINB><<<blocks, block, 0, ctx->stream>>>(ctx->g, parity, N, links, (const Cx *)in,
                                                                                   (Cx *)out, (const Cx *)xp, (Real)a, done);
    return bkr_check_launch(ctx);
}

// register tile T = ceil(N / ceil(N / 8)): N <= 8 -> T = N; 9..16 -> two groups; 17..24 -> three; 25..32 -> four
template <typename Real>
static int launch_n(bkr_ctx *ctx, int parity, int N, const void *in, void *out, const void *xp, double a, const int *done)
{
    const int G = (N + 7) / 8;
    const int T = (N + G - 1) / G;
    switch (T) {
    case 1: return launch_t<Real, 1, 128, 4>(ctx, parity, N, in, out, xp, a, done);
    case 2: return launch_t<Real, 2, 128, 4>(ctx, parity, N, in, out, xp, a, done);
    case 3: return launch_t<Real, 3, 128, 4>(ctx, parity, N, in, out, xp, a, done);
    case 4: return launch_t<Real, 4, 128, 4>(ctx, parity, N, in, out, xp, a, done);
    case 5: return launch_t<Real, 5, 128, 3>(ctx, parity, N, in, out, xp, a, done);
    case 6: return launch_t<Real, 6, 128, 3>(ctx, parity, N, in, out, xp, a, done);
    case 7: return launch_t<Real, 7, 128, 3>(ctx, parity, N, in, out, xp, a, done);
    case 8: return launch_t<Real, 8, 128, 3>(ctx, parity, N, in, out, xp, a, done);
    }
    return BKR_EINVAL;
}

int launch_dslash(bkr_ctx *ctx, int out_parity, int N, int prec, const void *in, void *out, const void *xp, double a,
                  const int *done)
{
    if (prec == BKR_F64) {
        if (!ctx->links64) return BKR_ENOLINKS;
        return launch_n<double>(ctx, out_parity, N, in, out, xp, a, done);
    }
    if (!ctx->links32) return BKR_ENOLINKS;
    return launch_n<float>(ctx, out_parity, N, in, out, xp, a, done);
}
