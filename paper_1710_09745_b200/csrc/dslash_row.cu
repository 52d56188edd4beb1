// Multi-rhs improved-staggered stencil, "row window" version (eq. 2): the kernel for
// blocks of 9-16 rhs per CTA (fp64), 17-32 rhs as a cluster of two CTAs.
//
//   out(x) = sum_h W_h(x) in(nbr_h(x)),  16 hops;  optional epilogue out = a * xp - out
//
// Why a third kernel.  The window kernel of dslash_win.cu stages every operand in shared memory
// with TMA and holds 8 rhs per CTA; at N = 16 it runs at 41 % of the FP64 pipe with nothing saturated except the
// shared-memory port budget: per (64-site tile, hop, 8 rhs) the port moves 444 wavefronts (TMA fills + reads) for 288
// cycles of DFMA issue.  This kernel cuts the port traffic per DFMA by 1.6 x:
//  * a CTA holds ALL 16 rhs of a 64-site tile (4 rhs per thread, 4 rhs groups per warp), so a link matrix is written to
//    shared memory once and read once per 16 rhs: a warp is 8 sites x 4 rhs groups, the 4 lanes of a site read the same
//    16 bytes (one broadcast wavefront per link element instead of four);
//  * the z/t neighbours never touch shared memory: plain 16-byte ld.global.nc loads, one hop ahead, into registers
//    (setmaxnreg gives the 8 arithmetic warps 232 registers, the producer warps 40);
//  * the x/y neighbours come from a window of whole x-rows in shared memory (one TMA tensor copy per row of the strip:
//    every input row crosses L2 -> SM once per strip instead of 8 times), cyclic in y;
//  * one thread does all 16 hops of its site: no exchange of partial sums between warp sets;
//  * operands are fetched one column (3 link elements + T vector elements) ahead of the FMAs that use them, barrier
//    probes included, so that the two warps of a scheduler do not both sit on a shared-memory round trip.
// Each link matrix is loaded once per call also for N = 17-32: the two CTAs of a cluster take 16 rhs each and every link
// stage is fetched once, half by each CTA, as a multicast bulk copy into both shared memories.
#include "common.cuh"
#include "tma.cuh"

#include <cuda.h>

#include <algorithm>
#include <string.h>
#include <vector>

struct RowParams {
    Geom g;
    int N, parity;
    const void *wt;  // gather-form links of this output parity
    const void *in;
    void *out;
    const void *xp;
    double a;
    const int *strips; // first tile of each work unit (UL consecutive tiles of one (z, t) strip), in processing order
    int nstrip;
    int UL;    // tiles per unit
    int vec_policy; // L2 priority of the z/t neighbour loads: 0 evict_normal, 1 evict_last
    const int *done;
    int WCH;   // window ring slots (rows)
    int rllog; // log2 of the link ring depth
    uint32_t off_win, off_bar;
};

namespace {

__device__ __forceinline__ uint32_t row_cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void row_cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// arrive on the mbarrier at the same offset in CTA `rank` of the cluster (default .release.cta semantics: the slot was
// only read, by shared-memory loads whose values have been consumed)
__device__ __forceinline__ void row_arrive_remote(uint64_t *bar, uint32_t rank)
{
    asm volatile("{\n\t.reg .b32 ra;\n\tmapa.shared::cluster.u32 ra, %0, %1;\n\t"
                 "mbarrier.arrive.shared::cluster.b64 _, [ra];\n\t}" ::"r"(smem_addr(bar)),
                 "r"(rank)
                 : "memory");
}
__device__ __forceinline__ void row_tma_1d_mc(void *dst, const void *src, uint32_t bytes, uint64_t *bar, uint16_t mask, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster.L2::cache_hint "
                 "[%0], [%1], %2, [%3], %4, %5;" ::"r"(smem_addr(dst)),
                 "l"(src), "r"(bytes), "r"(smem_addr(bar)), "h"(mask), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void row_tma_3d(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, uint64_t *bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
                     smem_addr(dst)),
                 "l"(tm), "r"(smem_addr(bar)), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
// one probe of a barrier phase; the result is consumed later (row_wait_finish) so that FMAs can issue in between
__device__ __forceinline__ uint32_t row_try_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok)
                 : "r"(smem_addr(bar)), "r"(parity));
    return ok;
}
__device__ __forceinline__ void row_wait_finish(uint32_t ok, uint64_t *bar, uint32_t parity)
{
    while (!ok) ok = row_try_wait(bar, parity);
}
// 16-byte neighbour load with an explicit L2 policy.  Without one, ld.global.nc.L1::no_allocate (SASS LDG.E.NA) leaves its
// lines at low priority in L2 as well: ncu showed 7.1 GB of DRAM reads per launch (32^3 x 64, N = 16) against 4.7 GB with
// an evict_normal policy attached -- every z/t neighbour is read 8 times and has to stay.
__device__ __forceinline__ double2 ldg_cx(const double2 *p, uint64_t pol)
{
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}

// acc[i] += W(:, b) v_i(b) for the T rhs of a thread: u[a] = W_ab, v[i] = component b of rhs i.  rhs outermost: the FMAs of
// rhs i need only v[i], so they start as soon as the first vector load of the column has landed (with the link element
// outermost -- better operand reuse, 31.9 against 28.7 TFLOP/s register-only -- the kernel measured 1.9 against 1.5 ms).
template <typename Real, typename Cx, int T> __device__ __forceinline__ void col_fma(Real (&acc)[T][6], const Cx (&u)[3], const Cx (&v)[T])
{
#pragma unroll
    for (int i = 0; i < T; i++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            acc[i][2 * a] = fma(u[a].x, v[i].x, acc[i][2 * a]);
            acc[i][2 * a + 1] = fma(u[a].x, v[i].y, acc[i][2 * a + 1]);
        }
#pragma unroll
    for (int i = 0; i < T; i++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            acc[i][2 * a] = fma(-u[a].y, v[i].y, acc[i][2 * a]);
            acc[i][2 * a + 1] = fma(u[a].y, v[i].x, acc[i][2 * a + 1]);
        }
}

constexpr int ROW_CONSUMER_WARPS = 8;
constexpr int ROW_THREADS = 384; // 8 arithmetic warps + one producer warpgroup (2 lanes of it work)
constexpr uint32_t ROW_DR3 = 0x64333320u; // per window hop: row shift + 3   (y-3, y-1, x+1, x-1, x+3, x-3, y+1, y+3)
constexpr uint32_t ROW_DC2 = 0x22031222u; // per window hop: column shift + 2, before the row-parity offset of the x hops
constexpr uint32_t ROW_ISX = 0x3cu;       // hops 2..5 are x hops

} // namespace

// blockDim = 384: warps 0-7 arithmetic (warp w: sites 8 w .. 8 w + 7 of the 64-site tile, lane = 8 * rhs group + site),
// warp 8 lane 0: link stages, warp 9 lane 0: window rows.
template <typename Real, int T, int C, bool XP, int XH>
__global__ void __launch_bounds__(ROW_THREADS, 1) dslash_row_kernel(const __grid_constant__ CUtensorMap tm_win, const RowParams p)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int NG = 4, NC = NG * T, SPW = 8;
    constexpr int TR = 64 / XH; // x-rows per tile
    constexpr uint32_t LSTAGE = 9 * 64 * sizeof(Cx);
    constexpr uint32_t ROWB = NC * 3 * XH * sizeof(Cx); // one window row: [rhs][colour][XH sites]
    extern __shared__ __align__(1024) unsigned char dsm[];
    unsigned char *const lnk = dsm;
    unsigned char *const win = dsm + p.off_win;
    uint64_t *const bar = reinterpret_cast<uint64_t *>(dsm + p.off_bar);
    uint64_t *const lfull = bar, *const lempty = bar + 8, *const wfull = bar + 16, *const wempty = bar + 48;
    if (p.done && *p.done) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rllog = p.rllog, RL = 1 << rllog, WCH = p.WCH;
    if (threadIdx.x == 0) {
        for (int s = 0; s < RL; s++) {
            mbar_init(&lfull[s], 1);
            mbar_init(&lempty[s], ROW_CONSUMER_WARPS * C);
        }
        for (int s = 0; s < WCH; s++) {
            mbar_init(&wfull[s], 1);
            mbar_init(&wempty[s], ROW_CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (C > 1) row_cluster_sync();
    else __syncthreads();

    const uint32_t rank = C > 1 ? row_cluster_ctarank() : 0u;
    const int cid = blockIdx.x / C, ncl = gridDim.x / C;
    const Geom &g = p.g;
    const int Y = g.X[1], Z = g.X[2], Tt = g.X[3];
    const int Vh = g.Vh;
    const int tps = XH * Y / 64; // tiles per strip
    const int UL = p.UL;
    const int rows_per_unit = UL * TR + 6;

    if (warp >= ROW_CONSUMER_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        const int role = warp - ROW_CONSUMER_WARPS;
        if (lane == 0 && role == 0) {
            // ---------------------------------------------------------------- link stages, one per (tile, hop)
            const uint64_t pol = policy_evict_first();
            const Cx *wt = reinterpret_cast<const Cx *>(p.wt);
            constexpr uint32_t SL = LSTAGE / C;
            int ls = 0;
            for (int si = cid; si < p.nstrip; si += ncl) {
                const int k0 = p.strips[si];
                for (int k = k0; k < k0 + UL; k++)
                    for (int sq = 0; sq < 16; sq++, ls++) {
                        const int h = (sq & 1) ? 8 + (sq >> 1) : (sq >> 1); // stage order w0 z0 w1 z1 ... (see the arithmetic warps)
                        const int slot = ls & (RL - 1), use = ls >> rllog;
                        if (use > 0) mbar_wait(&lempty[slot], (use - 1) & 1);
                        mbar_expect_tx(&lfull[slot], LSTAGE);
                        const unsigned char *src = reinterpret_cast<const unsigned char *>(wt + ((size_t)k * 16 + h) * 9 * 64);
                        if (C == 1) tma_load_1d_hint(lnk + (size_t)slot * LSTAGE, src, LSTAGE, &lfull[slot], pol);
                        else
                            row_tma_1d_mc(lnk + (size_t)slot * LSTAGE + rank * SL, src + rank * SL, SL, &lfull[slot],
                                          (uint16_t)((1u << C) - 1u), pol);
                    }
            }
        } else if (lane == 0 && role == 1) {
            // ---------------------------------------------------------------- window rows: virtual rows -3 .. Y + 2 of a strip
            int q = 0; // absolute row sequence number of this CTA
            for (int si = cid; si < p.nstrip; si += ncl) {
                const int k0 = p.strips[si];
                const int e0 = (k0 - k0 % tps) * 64;   // first site of the strip
                const int y0 = (k0 % tps) * TR;        // first row of the unit
                for (int v = y0 - 3; v < y0 + UL * TR + 3; v++, q++) {
                    const int slot = q % WCH, use = q / WCH;
                    int y = v;
                    if (y < 0) y += Y;
                    if (y >= Y) y -= Y;
                    if (use > 0) mbar_wait(&wempty[slot], (use - 1) & 1);
                    mbar_expect_tx(&wfull[slot], ROWB);
                    row_tma_3d(win + (size_t)slot * ROWB, &tm_win, 2 * (e0 + y * XH), 0, (int)rank * NC, &wfull[slot]);
                }
            }
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
        // ------------------------------------------------------------------ arithmetic warps
        // Stage order inside a tile (link ring and hop loop): w0 z0 w1 z1 ... w7 z7  (w = window hop h = i, z = z/t hop
        // h = 8 + i).  The z/t vectors live in two register buffers; buffer i & 1 serves z hop i and each of its three
        // columns is refilled, right after its FMAs, with the same column of z hop i + 2 -- so a z/t load has four hop
        // times (two window hops, two z/t hops) to arrive, whatever DRAM does.
        const int sg = lane >> 3;            // rhs group
        const int sl = warp * SPW + (lane & 7); // site in tile
        const int r = sl / XH, ex = sl % XH; // row in tile, column
        const int j0 = sg * T;
        const int jg = (int)rank * NC + j0; // first global rhs of this thread
        // rhs index clamped to the block for the plain loads (the window copy zero-fills by itself)
        int ioff3[T]; // 3 x (rhs index relative to jg), clamped to the block
#pragma unroll
        for (int i = 0; i < T; i++) ioff3[i] = 3 * max(-jg, min(i, p.N - 1 - jg));
        const uint32_t VhB = (uint32_t)Vh * (uint32_t)sizeof(Cx); // bytes between the colour planes of a vector (< 2^32 / 24)
        const Cx *const vin = reinterpret_cast<const Cx *>(p.in);
        const Cx *const vxp = reinterpret_cast<const Cx *>(p.xp);
        Cx *const vout = reinterpret_cast<Cx *>(p.out);
        uint64_t vpol; // L2 policy of the z/t neighbour loads
        if (p.vec_policy == 1) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(vpol));
        else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(vpol));
        Cx uA[3], uB[3], wA[T], wB[T]; // link column / window vector operands, two register sets
        Cx vz[2][3 * T];   // z/t neighbour vectors of two hops: [hop parity][colour * T + rhs]
        int ls = 0; // link stage counter
        int Q0 = 0; // absolute row sequence number of the first window row of the current unit
        for (int si = cid; si < p.nstrip; si += ncl) {
            const int k0 = p.strips[si];
            const int klu = k0 % tps;          // first tile of the unit inside its strip
            const int e0s = (k0 - klu) * 64;   // first site of the strip
            const int zc = (e0s / (XH * Y)) % Z, tcd = e0s / (XH * Y * Z);
            // e-index offset of z/t neighbour j = 0..7 (z-3, z-1, z+1, z+3, t-3, t-1, t+1, t+3; periodic): the same for every site of the strip
            auto zoffn = [&](int j) {
                const int hop = 2 * (j & 3) - 3;
                const bool isz = j < 4;
                const int cm = isz ? zc : tcd, Xm = isz ? Z : Tt;
                int cn = cm + hop;
                if (cn < 0) cn += Xm;
                if (cn >= Xm) cn -= Xm;
                return (cn - cm) * (isz ? XH * Y : XH * Y * Z);
            };
            int waited = 0, released = 0; // rows of this unit (q = v - first row + 3) waited for / given back
            for (int kl = 0; kl < UL; kl++) {
                const int e = e0s + (klu + kl) * 64 + sl;
                const int y = (klu + kl) * TR + r;
                const int o = (y + zc + tcd + p.parity) & 1;
                // column b of a z/t neighbour (or xp) tile: T loads of 16 bytes at byte offsets (3 i + b) * VhB from p0
                auto load_vz_col = [&](Cx(&dst)[3 * T], const unsigned char *p0, int b) {
#pragma unroll
                    for (int i = 0; i < T; i++)
                        dst[b * T + i] = ldg_cx(reinterpret_cast<const Cx *>(p0 + (ptrdiff_t)(ioff3[i] + b) * (ptrdiff_t)VhB), vpol);
                };
                auto vz_base = [&](const Cx *base, int eoff) {
                    return reinterpret_cast<const unsigned char *>(base + (size_t)jg * 3 * Vh + eoff);
                };
                // z hops 0 and 1 of this tile, unless the previous tile of the unit has already asked for them
                if (kl == 0) {
                    const unsigned char *p0 = vz_base(vin, e + zoffn(0));
#pragma unroll
                    for (int b = 0; b < 3; b++) load_vz_col(vz[0], p0, b);
                }
                if (kl == 0 || XP) {
                    const unsigned char *p0 = vz_base(vin, e + zoffn(1));
#pragma unroll
                    for (int b = 0; b < 3; b++) load_vz_col(vz[1], p0, b);
                }
                // window rows v <= TR kl + TR + 2, i.e. q <= TR kl + TR + 5
                while (waited <= kl * TR + TR + 5) {
                    const int qq = Q0 + waited;
                    mbar_wait(&wfull[qq % WCH], (qq / WCH) & 1);
                    waited++;
                }
                const int qmod = (Q0 + kl * TR + r) % WCH; // window slot of virtual row y - 3
                Real acc[T][6];
#pragma unroll
                for (int i = 0; i < T; i++)
#pragma unroll
                    for (int qd = 0; qd < 6; qd++) acc[i][qd] = (Real)0;

                // window operand address of hop h (h < 8)
                auto win_ptr = [&](int h) {
                    const int dr3 = (ROW_DR3 >> (4 * h)) & 15, dc = (int)((ROW_DC2 >> (4 * h)) & 15) - 2 + (((ROW_ISX >> h) & 1) ? o : 0);
                    int slot = qmod + dr3; // dr3 <= 6 < WCH
                    if (slot >= WCH) slot -= WCH;
                    return reinterpret_cast<const Cx *>(win + (size_t)slot * ROWB) + j0 * 3 * XH + ((ex + dc) & (XH - 1));
                };
                auto lnk_ptr = [&](int stage) { return reinterpret_cast<const Cx *>(lnk + (size_t)(stage & (RL - 1)) * LSTAGE) + sl; };
                auto load_u = [&](Cx(&u)[3], const Cx *lk, int b) {
#pragma unroll
                    for (int a = 0; a < 3; a++) u[a] = lds_cx(lk + (3 * a + b) * 64);
                };
                auto load_vw = [&](Cx(&w)[T], const Cx *wp, int b) {
#pragma unroll
                    for (int i = 0; i < T; i++) w[i] = lds_cx(wp + (i * 3 + b) * XH);
                };
                auto release_link = [&](int stage) {
                    asm volatile("fence.acq_rel.cta;" ::: "memory"); // the slot's loads are complete before it goes back (dslash_win.cu)
                    __syncwarp();
                    if (lane == 0) {
                        uint64_t *bb = &lempty[stage & (RL - 1)];
                        if (C == 1) mbar_arrive(bb);
                        else
                            for (uint32_t rr = 0; rr < (uint32_t)C; rr++) row_arrive_remote(bb, rr);
                    }
                };
                // One window hop + one z/t hop = six columns.  Operands of a column are loaded while the FMAs of the column
                // before run, into the register set (A or B) that column does not use; six columns bring the roles back to
                // where they started, so nothing is ever copied.  On entry uA, wA hold column 0 of window hop i.
                auto hop_pair = [&](int i, Cx(&vcur)[3 * T]) {
                    const int st = ls + 2 * i;
                    {
                        // ---- window hop i
                        const Cx *lk = lnk_ptr(st);
                        const Cx *wp = win_ptr(i);
                        load_u(uB, lk, 1);
                        load_vw(wB, wp, 1);
                        col_fma<Real, Cx, T>(acc, uA, wA);
                        load_u(uA, lk, 2);
                        load_vw(wA, wp, 2);
                        col_fma<Real, Cx, T>(acc, uB, wB);
                        // probe of the next stage's barrier issued ahead of the FMAs that hide its latency
                        uint64_t *bb = &lfull[(st + 1) & (RL - 1)];
                        const uint32_t par = ((st + 1) >> rllog) & 1;
                        const uint32_t ok = row_try_wait(bb, par);
                        col_fma<Real, Cx, T>(acc, uA, wA);
                        row_wait_finish(ok, bb, par);
                        load_u(uB, lnk_ptr(st + 1), 0);
                        release_link(st);
                        if (i == 1) {
                            // hops 0, 1 were y-3, y-1: rows below the tile are dead from here on (x hops read the tile's own rows)
                            const int new_rel = min(kl * TR + 3, (kl + 1) * TR);
                            if (lane == 0)
                                for (int cc = released; cc < new_rel; cc++) mbar_arrive(&wempty[(Q0 + cc) % WCH]);
                            released = max(released, new_rel);
                        }
                    }
                    {
                        // ---- z/t hop i: vectors from vcur, whose columns are refilled as they are used up
                        const Cx *lk = lnk_ptr(st + 1);
                        // refill source: z hop i + 2 of this tile; from hop 6 on the first z hops of the unit's next tile (hop 7
                        // with the xpay epilogue: the xp tile).  Nothing after the unit's last tile.
                        const bool more = kl + 1 < UL;
                        const bool refill = i < 6 || more || (i == 7 && XP);
                        const unsigned char *np0 = i < 6    ? vz_base(vin, e + zoffn(i + 2))
                                                   : i == 6 ? vz_base(vin, e + 64 + zoffn(0))
                                                   : XP     ? vz_base(vxp, e)
                                                            : vz_base(vin, e + 64 + zoffn(1));
                        Cx(&v0)[T] = *reinterpret_cast<Cx(*)[T]>(&vcur[0]);
                        Cx(&v1)[T] = *reinterpret_cast<Cx(*)[T]>(&vcur[T]);
                        Cx(&v2)[T] = *reinterpret_cast<Cx(*)[T]>(&vcur[2 * T]);
                        load_u(uA, lk, 1);
                        col_fma<Real, Cx, T>(acc, uB, v0);
                        if (refill) load_vz_col(vcur, np0, 0); // column 0 has been read: refill it
                        load_u(uB, lk, 2);
                        col_fma<Real, Cx, T>(acc, uA, v1);
                        if (refill) load_vz_col(vcur, np0, 1);
                        if (i < 7) {
                            uint64_t *bb = &lfull[(st + 2) & (RL - 1)];
                            const uint32_t par = ((st + 2) >> rllog) & 1;
                            const uint32_t ok = row_try_wait(bb, par);
                            col_fma<Real, Cx, T>(acc, uB, v2);
                            row_wait_finish(ok, bb, par);
                            load_u(uA, lnk_ptr(st + 2), 0);
                            load_vw(wA, win_ptr(i + 1), 0);
                        } else {
                            col_fma<Real, Cx, T>(acc, uB, v2);
                        }
                        if (refill) load_vz_col(vcur, np0, 2);
                        release_link(st + 1);
                    }
                };

                // ---- prologue: column 0 of window hop 0
                mbar_wait(&lfull[ls & (RL - 1)], (ls >> rllog) & 1);
                load_u(uA, lnk_ptr(ls), 0);
                load_vw(wA, win_ptr(0), 0);
#pragma unroll
                for (int i = 0; i < 8; i += 2) {
                    hop_pair(i, vz[0]);
                    hop_pair(i + 1, vz[1]);
                }
                // rows the next tile does not need (v < TR (kl + 1) - 3), all of them after the last tile of the unit
                {
                    const int new_rel = kl == UL - 1 ? rows_per_unit : (kl + 1) * TR;
                    asm volatile("fence.acq_rel.cta;" ::: "memory");
                    __syncwarp();
                    if (lane == 0)
                        for (int cc = released; cc < new_rel; cc++) mbar_arrive(&wempty[(Q0 + cc) % WCH]);
                    released = max(released, new_rel);
                }
                ls += 16;
                // ---- epilogue: out = acc  or  a * xp - acc
#pragma unroll
                for (int i = 0; i < T; i++)
#pragma unroll
                    for (int cc = 0; cc < 3; cc++) {
                        Cx ov;
                        ov.x = acc[i][2 * cc];
                        ov.y = acc[i][2 * cc + 1];
                        if (XP) {
                            const Cx xv = vz[1][cc * T + i];
                            ov.x = fma((Real)p.a, xv.x, -ov.x);
                            ov.y = fma((Real)p.a, xv.y, -ov.y);
                        }
                        if (jg + i < p.N) __stcs(vout + ((size_t)(jg + i) * 3 + cc) * Vh + e, ov);
                    }
            }
            Q0 += rows_per_unit;
        }
    }
    // no CTA may leave while a peer can still multicast into its shared memory or arrive on its barriers
    if (C > 1) row_cluster_sync();
}

// ---------------------------------------------------------------- host

typedef CUresult (*RowEncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static RowEncodeFn row_encode_fn()
{
    static RowEncodeFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (RowEncodeFn)ptr;
        else
            cudaGetLastError();
    }
    return fn;
}

// Work units (UL consecutive tiles of one (z, t) strip) in the order they are handed to the CTAs: z blocks outermost, then
// t, then the strips of the block, then the units of a strip.  The CTAs of the grid work on a run of consecutive entries:
// the smaller the run's extent in t (fewer sites in flight: short units; narrow z blocks), the shorter an input line
// has to survive in L2 between its first use (t + 3 neighbour of a strip) and its last (t - 3 neighbour) -- measured with
// ncu: whole strips and 16-z blocks give 7.1 GB of DRAM reads per launch at 32^3 x 64, N = 16,
// against 3.2 GB algorithmic.
static int row_build_units(bkr_ctx *ctx, int N, int prec, int UL)
{
    const Geom &g = ctx->g;
    const int Xh = g.X[0] / 2, Y = g.X[1], Z = g.X[2], Tt = g.X[3];
    const double budget = (ctx->l2_budget_mb > 0 ? ctx->l2_budget_mb : 24) * 1e6;
    const double site_bytes = 3.0 * std::max(N, ctx->dslash_nblock) * (prec == BKR_F64 ? 16 : 8);
    int zb = 1;
    for (int c = 1; c <= Z; c++)
        if (Z % c == 0 && (7.0 * Xh * Y * c * site_bytes <= budget || Tt <= 7)) zb = c;
    const int key = zb * 64 + UL;
    if (ctx->row_strips && ctx->row_key == key) return BKR_OK;
    const int tps = Xh * Y / 64;
    std::vector<int> st;
    for (int zblk = 0; zblk < Z / zb; zblk++)
        for (int t = 0; t < Tt; t++)
            for (int zi = 0; zi < zb; zi++)
                for (int u = 0; u < tps; u += UL) st.push_back((t * Z + zblk * zb + zi) * tps + u);
    if (ctx->row_strips) cudaFree(ctx->row_strips);
    ctx->row_strips = nullptr;
    BKR_CUDA(ctx, cudaMalloc((void **)&ctx->row_strips, st.size() * sizeof(int)));
    BKR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    BKR_CUDA(ctx, cudaMemcpy(ctx->row_strips, st.data(), st.size() * sizeof(int), cudaMemcpyHostToDevice));
    ctx->row_nstrip = (int)st.size();
    ctx->row_key = key;
    return BKR_OK;
}

static const size_t ROW_SMEM_MAX = 232448;

template <typename Real, int T, int C, bool XP, int XH>
static int launch_row_x(bkr_ctx *ctx, int parity, int N, int prec, const void *in, void *out, const void *xp, double a, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int NC = 4 * T, TR = 64 / XH;
    const Geom &g = ctx->g;
    RowParams p;
    memset(&p, 0, sizeof(p));
    const size_t lstage = (size_t)9 * 64 * sizeof(Cx), rowb = (size_t)NC * 3 * XH * sizeof(Cx), bbytes = 80 * 8;
    p.WCH = TR + 6 + 2; // rows a tile reads + two the producer may fill while the tile's lower halo is still in use
    int rl = 8;
    while (rl * lstage + p.WCH * rowb + bbytes > ROW_SMEM_MAX && rl > 2) rl /= 2;
    if (rl * lstage + p.WCH * rowb + bbytes > ROW_SMEM_MAX || p.WCH > 32 || rl < 4) return 1;
    // spare shared memory goes to more window rows (the producer runs further ahead)
    while (p.WCH < 32 && rl * lstage + (p.WCH + 1) * rowb + bbytes <= ROW_SMEM_MAX) p.WCH++;
    p.rllog = rl == 8 ? 3 : 2;
    p.off_win = (uint32_t)(rl * lstage);
    p.off_bar = (uint32_t)(p.off_win + p.WCH * rowb);
    const size_t smem = p.off_bar + bbytes;

    RowEncodeFn fn = row_encode_fn();
    if (!fn) return 1;
    {
        const int tps = XH * g.X[1] / 64;
        int UL = ctx->row_unit_tiles > 0 ? ctx->row_unit_tiles : 2;
        while (UL > 1 && tps % UL) UL--;
        UL = std::min(UL, tps);
        p.UL = UL;
        BKR_TRY(row_build_units(ctx, N, prec, UL));
    }
    CUtensorMap tm;
    {
        const size_t rsz = sizeof(Real);
        cuuint64_t gdim[3] = {(cuuint64_t)2 * g.Vh, 3, (cuuint64_t)N};
        cuuint64_t gstr[2] = {(cuuint64_t)2 * g.Vh * rsz, (cuuint64_t)6 * g.Vh * rsz};
        cuuint32_t box[3] = {(cuuint32_t)(2 * XH), 3, (cuuint32_t)NC};
        cuuint32_t estr[3] = {1, 1, 1};
        if (fn(&tm, sizeof(Real) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void *>(in), gdim,
               gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return 1;
    }
    const int ntiles = link_tiles(g);
    p.g = g;
    p.N = N;
    p.parity = parity;
    p.wt = (sizeof(Real) == 8 ? (const Cx *)ctx->links64 : (const Cx *)ctx->links32) + (size_t)parity * ntiles * 16 * 9 * 64;
    p.in = in;
    p.out = out;
    p.xp = xp;
    p.a = a;
    p.strips = ctx->row_strips;
    p.nstrip = ctx->row_nstrip;
    p.done = done;
    p.vec_policy = ctx->row_vec_policy & 1;

    auto kern = dslash_row_kernel<Real, T, C, XP, XH>;
    static int max_clusters = -1, attr_dev = -1; // per instantiation; the shared-memory opt-in is per device
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(ROW_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = ctx->stream;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (max_clusters < 0 || attr_dev != ctx->device) {
        attr_dev = ctx->device;
        BKR_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ROW_SMEM_MAX));
        cfg.gridDim = dim3((BKR_NUM_SMS / C) * C);
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess || n <= 0) {
            cudaGetLastError();
            max_clusters = 0;
        } else {
            max_clusters = std::min(n, BKR_NUM_SMS / C);
        }
    }
    if (max_clusters == 0) return 1;
    cfg.gridDim = dim3((unsigned)(std::min(max_clusters, p.nstrip) * C));
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, tm, p);
    if (e != cudaSuccess) {
        ctx->last_cuda = (int)e;
        return BKR_ECUDA;
    }
    return bkr_check_launch(ctx);
}

template <typename Real, int T, int C, int XH>
static int launch_row_c(bkr_ctx *ctx, int parity, int N, int prec, const void *in, void *out, const void *xp, double a, const int *done)
{
    if (xp) return launch_row_x<Real, T, C, true, XH>(ctx, parity, N, prec, in, out, xp, a, done);
    return launch_row_x<Real, T, C, false, XH>(ctx, parity, N, prec, in, out, xp, a, done);
}

// 1 = not applicable (the caller tries the other stencil kernels)
int launch_dslash_row(bkr_ctx *ctx, int out_parity, int N, int prec, const void *in, void *out, const void *xp, double a, const int *done)
{
    const Geom &g = ctx->g;
    const int Xh = g.X[0] / 2;
    // Not in the automatic choice: at 32^3 x 64, N = 16 it measures 1.5-1.8 ms against 1.33-1.42 ms for the window kernel
    // (DESIGN.md section 6.1c has the numbers and the reasons); bkr_set_dslash_variant(ctx, 2) selects it.
    if (ctx->dslash_force != 2) return 1;
    if (prec != BKR_F64 || Xh != 16 || (Xh * g.X[1]) % 64 != 0) return 1;
    if (N <= 16) {
        if (N <= 8) return launch_row_c<double, 2, 1, 16>(ctx, out_parity, N, prec, in, out, xp, a, done);
        if (N <= 12) return launch_row_c<double, 3, 1, 16>(ctx, out_parity, N, prec, in, out, xp, a, done);
        return launch_row_c<double, 4, 1, 16>(ctx, out_parity, N, prec, in, out, xp, a, done);
    }
    if (N <= 24) return launch_row_c<double, 3, 2, 16>(ctx, out_parity, N, prec, in, out, xp, a, done);
    if (N <= 32) return launch_row_c<double, 4, 2, 16>(ctx, out_parity, N, prec, in, out, xp, a, done);
    return 1;
}
