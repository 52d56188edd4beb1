// Multi-rhs improved-staggered stencil ("Dslash"), PAPER.md:95-101 (eq. 2) and PAPER.md:218-232.
//
//   out(x) = sum_mu [ F_mu(x) in(x+mu) - F_mu(x-mu)^dag in(x-mu) + K_mu(x) in(x+3mu) - K_mu(x-3mu)^dag in(x-3mu) ]
//   optional epilogue  out = a * xp - out   (second half of M = 4 m^2 - D_eo D_oe)
//
// Mapping.  The paper maps threadIdx.x to sites and threadIdx.y to rhs and relies on
// L1 to share the link between the threads of a site, plus a register tile of 1..6 rhs.
// Here the native block layout v[e][a][j] keeps the N rhs of a site contiguous, so:
//   * G adjacent lanes of a warp own one site; lane g holds T "slots" s = g + G*i (a slot = one 16-byte load
//     = 1 complex fp64 or 2 complex fp32), i.e. a register tile of T*VEC rhs;
//   * the 9 complex entries of a link are loaded once per lane with warp-broadcast loads (the G lanes of a
//     site hit the same address, lanes of different sites hit adjacent addresses of the SoA link array),
//     marked evict-first/streaming because every link is used exactly once per call;
//   * a neighbour gather is 3 rows of N contiguous rhs per site: fully coalesced for every hop direction.
#include "common.cuh"

template <typename Real, int VEC> struct SlotT;
template <> struct SlotT<double, 1> { typedef double2 type; };
template <> struct SlotT<float, 2> { typedef float4 type; };
template <> struct SlotT<float, 1> { typedef float2 type; };

template <typename Real, int VEC, int T, int G, bool EXACT, bool DAG>
__device__ __forceinline__ void hop(Real (&acc)[T][VEC][6], const typename CxT<Real>::type *__restrict__ U, int Vh,
                                    int e_link, const typename SlotT<Real, VEC>::type *__restrict__ in, size_t row0,
                                    int NS, int gl)
{
    typedef typename CxT<Real>::type Cx;
    typedef typename SlotT<Real, VEC>::type Slot;
    Cx u[9];
#pragma unroll
    for (int el = 0; el < 9; el++) u[el] = __ldcs(U + (size_t)el * Vh + e_link);
    Slot v[T][3];
#pragma unroll
    for (int i = 0; i < T; i++) {
        int s = gl + G * i;
        if (EXACT || s < NS) {
#pragma unroll
            for (int c = 0; c < 3; c++) v[i][c] = __ldg(in + (row0 + c) * NS + s);
        }
    }
#pragma unroll
    for (int i = 0; i < T; i++) {
        int s = gl + G * i;
        if (EXACT || s < NS) {
#pragma unroll
            for (int w = 0; w < VEC; w++) {
#pragma unroll
                for (int a = 0; a < 3; a++) {
#pragma unroll
                    for (int b = 0; b < 3; b++) {
                        const Real *vb = reinterpret_cast<const Real *>(&v[i][b]) + 2 * w;
                        if (!DAG) { // + U_ab v_b
                            Cx m = u[a * 3 + b];
                            acc[i][w][2 * a] = fma(m.x, vb[0], acc[i][w][2 * a]);
                            acc[i][w][2 * a] = fma(-m.y, vb[1], acc[i][w][2 * a]);
                            acc[i][w][2 * a + 1] = fma(m.x, vb[1], acc[i][w][2 * a + 1]);
                            acc[i][w][2 * a + 1] = fma(m.y, vb[0], acc[i][w][2 * a + 1]);
                        } else { // - conj(U_ba) v_b
                            Cx m = u[b * 3 + a];
                            acc[i][w][2 * a] = fma(-m.x, vb[0], acc[i][w][2 * a]);
                            acc[i][w][2 * a] = fma(-m.y, vb[1], acc[i][w][2 * a]);
                            acc[i][w][2 * a + 1] = fma(-m.x, vb[1], acc[i][w][2 * a + 1]);
                            acc[i][w][2 * a + 1] = fma(m.y, vb[0], acc[i][w][2 * a + 1]);
                        }
                    }
                }
            }
        }
    }
}

template <typename Real, int VEC, int T, int G, bool EXACT>
__global__ void __launch_bounds__(256)
dslash_kernel(Geom g, int parity, int NS, const typename CxT<Real>::type *__restrict__ links,
              const typename SlotT<Real, VEC>::type *__restrict__ in, typename SlotT<Real, VEC>::type *__restrict__ out,
              const typename SlotT<Real, VEC>::type *__restrict__ xp, Real a, const int *done)
{
    typedef typename SlotT<Real, VEC>::type Slot;
    if (done && *done) return;
    int tid = blockIdx.x * 256 + threadIdx.x;
    int e = tid / G, gl = tid % G;
    if (e >= g.Vh) return;
    // coordinates of the output site (parity, e)
    int s = 2 * e;
    int c[4];
    int x0 = s % g.X[0];
    int r = s / g.X[0];
    c[1] = r % g.X[1];
    r /= g.X[1];
    c[2] = r % g.X[2];
    c[3] = r / g.X[2];
    c[0] = x0 + ((c[1] + c[2] + c[3] + parity) & 1);
    s = s - x0 + c[0];
    const int stride[4] = {1, g.X[0], g.X[0] * g.X[1], g.X[0] * g.X[1] * g.X[2]};

    Real acc[T][VEC][6];
#pragma unroll
    for (int i = 0; i < T; i++)
#pragma unroll
        for (int w = 0; w < VEC; w++)
#pragma unroll
            for (int k = 0; k < 6; k++) acc[i][w][k] = (Real)0;

    const size_t Vh = g.Vh;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
#pragma unroll
        for (int type = 0; type < 2; type++) {
            const int h = type ? 3 : 1;
            int cf = c[mu] + h;
            if (cf >= g.X[mu]) cf -= g.X[mu];
            int cb = c[mu] - h;
            if (cb < 0) cb += g.X[mu];
            int ef = (s + (cf - c[mu]) * stride[mu]) >> 1;
            int eb = (s + (cb - c[mu]) * stride[mu]) >> 1;
            // forward: link leaving x (parity of x), vector at x + h mu
            hop<Real, VEC, T, G, EXACT, false>(acc, links + (size_t)(((type * 4 + mu) * 2 + parity) * 9) * Vh, g.Vh, e,
                                               in, (size_t)ef * 3, NS, gl);
            // backward: link leaving x - h mu (opposite parity), daggered, vector at x - h mu
            hop<Real, VEC, T, G, EXACT, true>(acc, links + (size_t)(((type * 4 + mu) * 2 + (1 - parity)) * 9) * Vh, g.Vh,
                                              eb, in, (size_t)eb * 3, NS, gl);
        }
    }

#pragma unroll
    for (int i = 0; i < T; i++) {
        int sl = gl + G * i;
        if (EXACT || sl < NS) {
#pragma unroll
            for (int cc = 0; cc < 3; cc++) {
                Slot o;
                Real *po = reinterpret_cast<Real *>(&o);
#pragma unroll
                for (int w = 0; w < VEC; w++) {
                    po[2 * w] = acc[i][w][2 * cc];
                    po[2 * w + 1] = acc[i][w][2 * cc + 1];
                }
                size_t idx = ((size_t)e * 3 + cc) * NS + sl;
                if (xp) {
                    Slot p = __ldg(xp + idx);
                    const Real *pp = reinterpret_cast<const Real *>(&p);
#pragma unroll
                    for (int k = 0; k < 2 * VEC; k++) po[k] = a * pp[k] - po[k];
                }
                out[idx] = o;
            }
        }
    }
}

template <typename Real, int VEC, int T, int G>
static int launch_tg(bkr_ctx *ctx, int parity, int NS, const void *in, void *out, const void *xp, double a,
                     const int *done)
{
    typedef typename CxT<Real>::type Cx;
    typedef typename SlotT<Real, VEC>::type Slot;
    const Cx *links = sizeof(Real) == 8 ? (const Cx *)ctx->links64 : (const Cx *)ctx->links32;
    size_t threads = (size_t)ctx->g.Vh * G;
    unsigned blocks = (unsigned)((threads + 255) / 256);
    if (NS == T * G)
        dslash_kernel<Real, VEC, T, G, true><<<blocks, 256, 0, ctx->stream>>>(ctx->g, parity, NS, links, (const Slot *)in,
                                                                              (Slot *)out, (const Slot *)xp, (Real)a, done);
    else
        dslash_kernel<Real, VEC, T, G, false><<<blocks, 256, 0, ctx->stream>>>(ctx->g, parity, NS, links, (const Slot *)in,
                                                                               (Slot *)out, (const Slot *)xp, (Real)a, done);
    return bkr_check_launch(ctx);
}

template <typename Real, int VEC>
static int launch_ns(bkr_ctx *ctx, int parity, int NS, const void *in, void *out, const void *xp, double a,
                     const int *done)
{
#define GO(T_, G_) return launch_tg<Real, VEC, T_, G_>(ctx, parity, NS, in, out, xp, a, done)
    if (NS == 1) GO(1, 1);
    if (NS == 2) GO(1, 2);
    if (NS <= 4) GO(2, 2);
    if (NS <= 6) GO(3, 2);
    if (NS <= 8) GO(4, 2);
    if (NS <= 12) GO(3, 4);
    if (NS <= 16) GO(4, 4);
    if (NS <= 24) GO(3, 8);
    if (NS <= 32) GO(4, 8);
#undef GO
    return BKR_EINVAL;
}

int launch_dslash(bkr_ctx *ctx, int out_parity, int N, int prec, const void *in, void *out, const void *xp, double a,
                  const int *done)
{
    if (prec == BKR_F64) {
        if (!ctx->links64) return BKR_ENOLINKS;
        return launch_ns<double, 1>(ctx, out_parity, N, in, out, xp, a, done);
    }
    if (!ctx->links32) return BKR_ENOLINKS;
    if (N % 2 == 0) return launch_ns<float, 2>(ctx, out_parity, N / 2, in, out, xp, a, done);
    return launch_ns<float, 1>(ctx, out_parity, N, in, out, xp, a, done);
}
