// Multi-rhs improved-staggered stencil ("Dslash"), PAPER.md:95-101 (eq. 2) and PAPER.md:218-232.
//
//   out(x) = sum_h W_h(x) in(nbr_h(x)),  16 hops h = (mu, fat|long, forward|backward)  (gather-form links, layout.cu)
//   optional epilogue  out = a * xp - out   (second half of M = 4 m^2 - D_eo D_oe)
//
// Design.
//  * One thread = one output site x T right-hand sides (the paper's register tiling); threadIdx.y =
//    rhs group, so the G = ceil(N/T) groups that work on the same 64 sites share one CTA and one copy of the links
//    (the paper's cache tiling, with shared memory in place of L1).
//  * Links are a pure HBM stream: every matrix is used once per call and, at N <= 16, they are more than half of
//    all bytes.  They never touch registers or the LSU miss path until they are needed: a persistent CTA walks
//    over its tiles and an elected thread streams the (tile, hop) chunks -- 9 x 64 complex, contiguous in the
//    tile-major layout -- into a 4-deep shared-memory ring with 1-D TMA bulk copies (cp.async.bulk + mbarrier
//    complete_tx), three hops ahead of the arithmetic.  Measured on the previous LDG-only kernel: 7.9 warps of 12
//    stalled on the long scoreboard with the FP64 pipe 33 % busy, whatever the register tile.
//  * Neighbour vectors are read with plain 16-byte loads: a warp reads 32 consecutive sites of one (rhs, colour)
//    plane, 512 contiguous bytes in fp64; x/y reuse comes from L1, z/t reuse from L2.
//  * L2 blocking: tiles are visited in an order that sweeps t inside a (y, z) block, so that the 7 time slices a
//    block needs for its t +- 1, +- 3 hops stay L2-resident (tile_order, built on the host below).
//  * Per site and rhs: 16 x 36 = 576 FMAs (1152 flop; the paper counts 1146).
#include "common.cuh"
#include "tma.cuh"

#include <algorithm>
#include <stdlib.h>
#include <vector>

// shared-memory stages of 9 x 64 complex per CTA (template parameter RG of the kernel): the link stream has to be
// requested far enough ahead to cover a loaded HBM round trip (ncu: with 4 stages = 3 hops ahead, 12 % of all warp
// time was spent in the try_wait of the "full" barrier), so the ring is as deep as the CTAs-per-SM budget allows.

template <int T> struct PipeDepth { static const int value = (3 * T) % 12 == 0 ? 12 : (3 * T) % 9 == 0 ? 9 : (3 * T) % 6 == 0 ? 6 : 3 * T; };

// G rhs groups of T rhs each; blockDim = (64, G); MINB CTAs per SM; RG ring stages (a power of two <= 16)
template <typename Real, int T, int G, bool EXACT, int MINB, int DD, int RG>
__global__ void __launch_bounds__(BKR_LINK_TILE *G, MINB)
dslash_kernel(Geom g, int N, int ntiles, const typename CxT<Real>::type *__restrict__ wt, const int *__restrict__ tile_order,
              const typename CxT<Real>::type *__restrict__ in, typename CxT<Real>::type *__restrict__ out,
              const typename CxT<Real>::type *__restrict__ xp, Real a, int parity, const int *done, int opts)
{
    typedef typename CxT<Real>::type Cx;
    constexpr uint32_t STAGE_BYTES = 9 * BKR_LINK_TILE * sizeof(Cx);
    constexpr int D = DD > 0 ? DD : PipeDepth<T>::value; // neighbour loads in flight per thread; divides 3 T
    constexpr int RING = RG;
    static_assert(RG == 2 || RG == 4 || RG == 8 || RG == 16, "ring depth must divide the 16 hops of a tile");
    extern __shared__ __align__(128) unsigned char dsm[];
    Cx(*stage)[9][BKR_LINK_TILE] = reinterpret_cast<Cx(*)[9][BKR_LINK_TILE]>(dsm);
    uint64_t *full = reinterpret_cast<uint64_t *>(dsm + (size_t)RING * STAGE_BYTES);
    uint64_t *empty = full + RING;
    if (done && *done) return;
    const int tid = threadIdx.y * BKR_LINK_TILE + threadIdx.x;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < RING; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 2 * G); // one arrival per warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // CTA b visits the tiles tile_order[b], tile_order[b + grid], ...: at any time the CTAs of the grid work on a window
    // of consecutive entries of the (L2-blocked) order
    const int ntl = ((int)blockIdx.x < ntiles) ? (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int nstages = ntl * 16;
    const uint64_t pol = policy_evict_first();
    auto issue = [&](int st) { // producer: stage st = hop (st % 16) of this CTA's tile number st / 16
        const int tile = tile_order[blockIdx.x + (st >> 4) * gridDim.x];
        const Cx *src = wt + ((size_t)tile * 16 + (st & 15)) * 9 * BKR_LINK_TILE;
        mbar_expect_tx(&full[st % RING], STAGE_BYTES);
        if (opts & 1) tma_load_1d(&stage[st % RING][0][0], src, STAGE_BYTES, &full[st % RING]);
        else tma_load_1d_hint(&stage[st % RING][0][0], src, STAGE_BYTES, &full[st % RING], pol);
    };
    if (tid == 0)
        for (int st = 0; st < RING && st < nstages; st++) issue(st);

    const int j0 = threadIdx.y * T;
    const int nvalid = N - j0;
    const size_t Vh = g.Vh;
    const Cx *vin = in + (size_t)j0 * 3 * Vh;

    for (int k = 0; k < ntl; k++) {
        const int e_raw = tile_order[blockIdx.x + k * gridDim.x] * BKR_LINK_TILE + threadIdx.x;
        const bool valid = e_raw < g.Vh;
        const int e = valid ? e_raw : g.Vh - 1; // tail tile: compute on a clamped site, store nothing
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

        Real acc[T][6];
#pragma unroll
        for (int i = 0; i < T; i++)
#pragma unroll
            for (int q = 0; q < 6; q++) acc[i][q] = (Real)0;

        // Runtime loop over the 16 hops (fully unrolled they are ~100 KB of code and the warps stall on instruction
        // fetch).  The neighbour-vector loads are software pipelined by hand: a register ring of D loads runs D
        // (b, rhs) steps ahead of the FMAs, across hop boundaries, because one warp must keep ~D 512-byte loads in
        // flight to cover L2/HBM latency at 12-16 warps per SM (measured: the compiler's own schedule kept ~2.4).
        const int st0 = k * 16;
        auto nbr = [&](int h) -> const Cx * {
            const int mu = BKR_HOP_MU(h), hop = BKR_HOP_LONG(h) ? 3 : 1;
            const int cm = mu == 0 ? c[0] : mu == 1 ? c[1] : mu == 2 ? c[2] : c[3];
            // select chains, not g.X[mu]: an indexed constant load is a scoreboarded (variable-latency) load, and the
            // in-order warp waited for it at the top of every hop (ncu source page: 8 % of all warp time)
            const int Xm = mu == 0 ? g.X[0] : mu == 1 ? g.X[1] : mu == 2 ? g.X[2] : g.X[3];
            const int sm = mu == 0 ? 1 : mu == 1 ? g.X[0] : mu == 2 ? g.X[0] * g.X[1] : g.X[0] * g.X[1] * g.X[2];
            int cn = BKR_HOP_BACK(h) ? cm - hop : cm + hop;
            if (cn < 0) cn += Xm;
            if (cn >= Xm) cn -= Xm;
            return vin + ((s + (cn - cm) * sm) >> 1);
        };
        // One running pointer walks over the neighbour loads in consumption order n = b T + i (address index
        // (3 i + b) Vh): += 3 Vh inside a colour b, += (1 - 3 (T - 1)) Vh at a colour change, = base of the next hop
        // after the last load of this one.  (Per-load base + k Vh addresses cost ptxas ~90 live registers.)
        const ptrdiff_t d_rhs = 3 * (ptrdiff_t)Vh, d_col = (1 - 3 * (T - 1)) * (ptrdiff_t)Vh;
        const Cx *pl = nbr(0);
        Cx vbuf[D];
#pragma unroll
        for (int n = 0; n < D; n++) {
            if (EXACT || (n % T) < nvalid) vbuf[n] = __ldg(pl);
            pl += ((n + 1) % T) ? d_rhs : d_col;
        }
#pragma unroll 1
        for (int h = 0; h < 16; h++) {
            const int slot = h & (RING - 1);      // (st0 + h) % RING: st0 = 16 k is a multiple of RING
            const uint32_t ph = ((st0 + h) / RING) & 1;
            // producer, one stage behind the consumers: refill the slot of the previous hop with the stage RING
            // hops after it
            if (tid == 0) {
                const int prev = st0 + h - 1;
                if (prev >= 0 && prev + RING < nstages) {
                    mbar_wait(&empty[prev & (RING - 1)], ((prev / RING) & 1));
                    issue(prev + RING);
                }
            }
            const Cx *vnext = nbr(h < 15 ? h + 1 : 15);
            mbar_wait(&full[slot], ph);
            Cx u[3];
#pragma unroll
            for (int n = 0; n < 3 * T; n++) {
                const int b = n / T, i = n % T;
                if (i == 0) {
#pragma unroll
                    for (int aa = 0; aa < 3; aa++) u[aa] = lds_cx(&stage[slot][aa * 3 + b][threadIdx.x]);
                }
                const Cx v = vbuf[n % D];
                const int m = n + D; // the step whose load takes this ring entry (m >= 3 T: step m - 3 T of the next hop)
                if (m == 3 * T) pl = vnext;
                if (m < 3 * T || h < 15) {
                    if (EXACT || (m % T) < nvalid) vbuf[n % D] = __ldg(pl);
                    pl += ((m + 1) % T) ? d_rhs : d_col;
                }
                if (EXACT || i < nvalid) {
#pragma unroll
                    for (int aa = 0; aa < 3; aa++) { // acc_a += W_ab v_b
                        acc[i][2 * aa] = fma(u[aa].x, v.x, acc[i][2 * aa]);
                        acc[i][2 * aa] = fma(-u[aa].y, v.y, acc[i][2 * aa]);
                        acc[i][2 * aa + 1] = fma(u[aa].x, v.y, acc[i][2 * aa + 1]);
                        acc[i][2 * aa + 1] = fma(u[aa].y, v.x, acc[i][2 * aa + 1]);
                    }
                }
            }
            asm volatile("fence.acq_rel.cta;" ::: "memory"); // the slot's loads are complete before it goes back (dslash_win.cu)
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(&empty[slot]);
        }

        if (valid) {
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
                            const Cx p = __ldg(vxp + (size_t)(i * 3 + cc) * Vh);
                            o.x = fma(a, p.x, -o.x);
                            o.y = fma(a, p.y, -o.y);
                        }
                        __stcs(vout + (size_t)(i * 3 + cc) * Vh, o);
                    }
                }
            }
        }
    }
}

// ---------------------------------------------------------------- host: L2 blocking and dispatch

// Order in which the link tiles (64 consecutive even-odd sites) are visited: (y, z) blocks outermost, then t, then
// the sites of the block's time slice.  The block is the largest one whose 7-slice working set (t-3 .. t+3 of the
// input block, N rhs) fits the L2 budget; cost = extra halo reads 6/YB + 6/ZB of the input per output site.
static int build_tile_order(bkr_ctx *ctx, int N, int prec)
{
    const Geom &g = ctx->g;
    const int Xh = g.X[0] / 2, Y = g.X[1], Z = g.X[2], Tt = g.X[3];
    const double budget = (ctx->l2_budget_mb > 0 ? ctx->l2_budget_mb : 48) * 1e6;
    const double site_bytes = 3.0 * std::max(N, ctx->dslash_nblock) * (prec == BKR_F64 ? 16 : 8);
    int bestY = Y, bestZ = Z;
    double best_cost = 1e30, best_ws = 0;
    bool best_fits = false;
    for (int yb = 1; yb <= Y; yb++) {
        if (Y % yb) continue;
        for (int zb = 1; zb <= Z; zb++) {
            if (Z % zb) continue;
            const double ws = 7.0 * Xh * yb * zb * site_bytes;
            const bool fits = ws <= budget || Tt <= 7;
            const double cost = (yb < Y ? 6.0 / yb : 0.0) + (zb < Z ? 6.0 / zb : 0.0);
            bool better;
            if (fits != best_fits) better = fits;
            else if (fits) better = cost < best_cost - 1e-12 || (cost < best_cost + 1e-12 && ws > best_ws);
            else better = ws < best_ws || best_ws == 0;
            if (better) {
                best_fits = fits;
                best_cost = cost;
                best_ws = ws;
                bestY = yb;
                bestZ = zb;
            }
        }
    }
    const int key = bestY * 4096 + bestZ + 1;
    if (ctx->tile_order && ctx->tile_order_key == key) return BKR_OK;
    const int ntiles = link_tiles(g);
    std::vector<std::pair<long long, int>> keys(ntiles);
    const int nyb = Y / bestY;
    for (int k = 0; k < ntiles; k++) {
        const long long e0 = (long long)k * BKR_LINK_TILE;
        const int y = (int)((e0 / Xh) % Y), z = (int)((e0 / ((long long)Xh * Y)) % Z), t = (int)(e0 / ((long long)Xh * Y * Z));
        const long long blk = (long long)(z / bestZ) * nyb + y / bestY;
        keys[k] = std::make_pair((blk * (Tt + 1) + t) * ((long long)ntiles + 1) + k, k);
    }
    std::sort(keys.begin(), keys.end());
    std::vector<int> order(ntiles);
    for (int k = 0; k < ntiles; k++) order[k] = keys[k].second;
    if (!ctx->tile_order) BKR_CUDA(ctx, cudaMalloc((void **)&ctx->tile_order, (size_t)ntiles * sizeof(int)));
    // synchronous copy from pageable memory: the table is tiny and rebuilt only when the blocking changes
    BKR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    BKR_CUDA(ctx, cudaMemcpy(ctx->tile_order, order.data(), (size_t)ntiles * sizeof(int), cudaMemcpyHostToDevice));
    ctx->tile_order_key = key;
    return BKR_OK;
}

// default ring depth: as many 9 x 64-complex stages as leave about 100 KB of the SM's 256 KB for L1 (x-direction
// neighbour reuse lives there)
template <typename Real, int MINB> struct RingDepth {
    static const int per_cta = 150 * 1024 / MINB / (9 * BKR_LINK_TILE * 2 * (int)sizeof(Real));
    static const int value = per_cta >= 16 ? 16 : per_cta >= 8 ? 8 : per_cta >= 4 ? 4 : 2;
};

template <typename Real, int T, int G, int MINB, int DD = 0, int RGG = 0>
static int launch_tg(bkr_ctx *ctx, int parity, int N, const void *in, void *out, const void *xp, double a, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int RG = RGG > 0 ? RGG : RingDepth<Real, MINB>::value;
    constexpr size_t SMEM = (size_t)RG * 9 * BKR_LINK_TILE * sizeof(Cx) + 2 * RG * sizeof(uint64_t);
    const int ntiles = link_tiles(ctx->g);
    const Cx *wt = (sizeof(Real) == 8 ? (const Cx *)ctx->links64 : (const Cx *)ctx->links32) +
                   (size_t)parity * ntiles * 16 * 9 * BKR_LINK_TILE;
    const int opts = 0;
    dim3 block(BKR_LINK_TILE, G);
    unsigned grid = (unsigned)std::min(ntiles, BKR_NUM_SMS * MINB);
    static int attr_dev = -1; // per instantiation: the opt-in is per device
    if (attr_dev != ctx->device) {
        BKR_CUDA(ctx, cudaFuncSetAttribute(dslash_kernel<Real, T, G, true, MINB, DD, RG>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM));
        BKR_CUDA(ctx, cudaFuncSetAttribute(dslash_kernel<Real, T, G, false, MINB, DD, RG>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM));
        attr_dev = ctx->device;
    }
    if (N == T * G)
        dslash_kernel<Real, T, G, true, MINB, DD, RG><<<grid, block, SMEM, ctx->stream>>>(
            ctx->g, N, ntiles, wt, ctx->tile_order, (const Cx *)in, (Cx *)out, (const Cx *)xp, (Real)a, parity, done, opts);
    else
        dslash_kernel<Real, T, G, false, MINB, DD, RG><<<grid, block, SMEM, ctx->stream>>>(
            ctx->g, N, ntiles, wt, ctx->tile_order, (const Cx *)in, (Cx *)out, (const Cx *)xp, (Real)a, parity, done, opts);
    return bkr_check_launch(ctx);
}

// register tile T and rhs groups G:  N <= 8: one group (T = 1,2,3,4,6,8);  9..12: 2 x 6;  13..16: 2 x 8;
// 17..24: 3 x 8;  25..32: 4 x 8
template <typename Real>
static int launch_n(bkr_ctx *ctx, int parity, int N, const void *in, void *out, const void *xp, double a, const int *done)
{
#define GO(T_, G_, M_) return launch_tg<Real, T_, G_, M_>(ctx, parity, N, in, out, xp, a, done)
    // Register budget decides the shape (ptxas -v: the fp64 T = 8 thread needs ~190 registers for 48 accumulators, the
    // 12-deep load ring and the link column; under a 168-register cap it spills ~0.5 KB per thread, and ncu showed the
    // spill traffic, not the stencil, filling the LSU).  fp64: at most 2 CTAs of 128 threads (or 4 of 64) per SM.
    if (sizeof(Real) == 8) {
        if (N == 1) GO(1, 1, 6);
        if (N == 2) GO(2, 1, 6);
        if (N == 3) GO(3, 1, 6);
        if (N == 4) GO(4, 1, 6);
        if (N <= 6) GO(6, 1, 6);
        if (N <= 8) return launch_tg<Real, 8, 1, 4, 12>(ctx, parity, N, in, out, xp, a, done);
        if (N <= 12) GO(6, 2, 3);
        if (N <= 16) return launch_tg<Real, 8, 2, 2, 12>(ctx, parity, N, in, out, xp, a, done);
        if (N <= 24) return launch_tg<Real, 4, 6, 1, 12>(ctx, parity, N, in, out, xp, a, done);
        if (N <= 32) return launch_tg<Real, 8, 4, 1, 12>(ctx, parity, N, in, out, xp, a, done);
        return BKR_EINVAL;
    }
    if (N == 1) GO(1, 1, 6);
    if (N == 2) GO(2, 1, 6);
    if (N == 3) GO(3, 1, 6);
    if (N == 4) GO(4, 1, 6);
    if (N <= 6) GO(6, 1, 6);
    if (N <= 8) GO(8, 1, 6);
    if (N <= 12) GO(6, 2, 3);
    if (N <= 16) GO(8, 2, 3);
    if (N <= 24) GO(8, 3, 2);
    if (N <= 32) GO(8, 4, 1);
#undef GO
    return BKR_EINVAL;
}

int launch_dslash(bkr_ctx *ctx, int out_parity, int N, int prec, const void *in, void *out, const void *xp, double a,
                  const int *done)
{
    if (!(prec == BKR_F64 ? (void *)ctx->links64 : (void *)ctx->links32)) return BKR_ENOLINKS;
    // the row-window kernel takes whole fp64 blocks of 9..32 rhs on X = 32 lattices, every link read once (dslash_row.cu)
    if (!ctx->dslash_nblock) {
        const int rc = launch_dslash_row(ctx, out_parity, N, prec, in, out, xp, a, done);
        if (rc != 1) {
            ctx->dslash_variant = 2;
            return rc;
        }
    }
    // fp64 blocks of 22-24 rhs: ONE window launch, a cluster of 3 CTAs, every link read once per call; as
    // fast as 16 + rest (32^3 x 64, N = 24: 2.21 vs 2.22 ms).  A cluster of 4 (30-32 rhs) is not: 3.04 vs 2.88 ms there and
    // 19.6 vs 16.0 ms at 48^3 x 96 for two launches of a cluster of 2, which read the links twice -- those blocks are
    // split unless BKR_TUNE_DSLASH_CHUNK = 1 asks for the single pass (BKR_TUNE_DSLASH_CHUNK = 2 splits everything).
    if (!ctx->dslash_nblock && prec == BKR_F64 && N > 16 && N <= 32 && 8 * ((N + 7) / 8) - N <= 2 && ctx->dslash_force != 0 &&
        ctx->dslash_force != 2 && ctx->tune[BKR_TUNE_DSLASH_CHUNK] != 2 && (N <= 24 || ctx->tune[BKR_TUNE_DSLASH_CHUNK] == 1)) {
        const int rc = launch_dslash_win(ctx, out_parity, N, prec, in, out, xp, a, done);
        if (rc != 1) {
            ctx->dslash_variant = 1;
            return rc;
        }
    }
    // Other blocks of more than 16 fp64 rhs go through in chunks of 16 (window kernel for the full chunk, the links are then
    // read once per chunk); likewise 11-13 rhs as 8 + rest (window kernel + plain kernel) and fp32 blocks of 17-28 rhs as
    // 16 + rest.  A chunk is a contiguous view of the native block [rhs][colour][site].
    int chunk = 0;
    if (N > 32 || ((ctx->dslash_force < 0 || ctx->dslash_force == 1) && ctx->tune[BKR_TUNE_DSLASH_CHUNK] != 1)) {
        if (prec == BKR_F64 && N > 16) chunk = 16;
        else if (prec == BKR_F64 && N >= 11 && N <= 13) chunk = 8; // 14 = window cluster of 2 (1.29 ms) beats 8 + 6 (1.32 ms)
        else if (prec == BKR_F32 && N > 32) chunk = 32; // 33..64 fp32 rhs: 32 (a window cluster of 2) + rest
        else if (prec == BKR_F32 && N > 16 && N <= 28) chunk = 16;
    }
    if (chunk) {
        const size_t stride = (size_t)3 * ctx->g.Vh * (prec == BKR_F64 ? sizeof(double2) : sizeof(float2));
        ctx->dslash_nblock = N;
        int rc = BKR_OK;
        for (int j = 0; j < N && rc == BKR_OK; j += chunk) {
            const int n = N - j < chunk ? N - j : chunk;
            rc = launch_dslash(ctx, out_parity, n, prec, (const char *)in + j * stride, (char *)out + j * stride,
                               xp ? (const char *)xp + j * stride : nullptr, a, done);
        }
        ctx->dslash_nblock = 0;
        return rc;
    }
    if (ctx->dslash_force != 0 && ctx->dslash_force != 2) {
        const int rc = launch_dslash_win(ctx, out_parity, N, prec, in, out, xp, a, done);
        if (rc != 1) {
            ctx->dslash_variant = 1;
            return rc;
        }
    }
    ctx->dslash_variant = 0;
    BKR_TRY(build_tile_order(ctx, N, prec));
    if (prec == BKR_F64) return launch_n<double>(ctx, out_parity, N, in, out, xp, a, done);
    return launch_n<float>(ctx, out_parity, N, in, out, xp, a, done);
}
