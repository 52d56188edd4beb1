// Multi-rhs improved-staggered stencil, "window" version for N >= ~6 (eq. 2).
//
//   out(x) = sum_h W_h(x) in(nbr_h(x)),  16 hops;  optional epilogue out = a * xp - out
//
// Why a second kernel.  With every neighbour vector fetched from L2 by plain loads
// (dslash.cu) each input element crosses the L2 -> SM fabric 16 times per call; at N >= 8 that is 8.6-14.4 GB per
// launch at 32^3 x 64 and the kernel sits on the ~6300 B/clk L2-slice throughput cap of the chip, not on HBM (ncu:
// lts__t_sectors ~ 3.8e8 per launch, DRAM 48 %, FP64 pipe 39 %).  The paper's answer on Pascal was texture/L1 reuse
// between the rhs of a thread block; on B200 the per-hop footprint (N x 48 bytes per site) is too
// large for L1 to hold between hops, so the reuse is made explicit:
//  * A CTA walks a run of consecutive 64-site tiles inside one (z, t) "strip" (all x, y at fixed z, t).  The x- and
//    y-neighbours of a tile lie within +-3 x-rows of it, so a sliding WINDOW of input rows in shared memory serves
//    all 8 x/y hops: every input row is fetched from L2 once per strip instead of 8 times.  z/t hops still cost one
//    L2 fetch each: 9 fetches per site instead of 16.
//  * Nothing is loaded by the arithmetic warps.  One producer lane feeds three shared-memory rings with TMA:
//    links (1-D bulk copy, 9 x 64 complex per hop, as in dslash.cu), window chunks (3-D tensor copy: 32 sites x 3
//    colours x NC rhs) and z/t neighbour stages (tensor copy: 64 sites x 3 colours x NC rhs, shifted by the hop).
//  * A CTA holds NC = T G rhs (8 in fp64, 16 in fp32).  For N > NC a thread-block CLUSTER of C = ceil(N / NC) CTAs
//    works on the same tiles, one rhs slice each, and every link stage is fetched ONCE for the cluster: each CTA
//    issues 1/C of the stage as a multicast bulk copy into all C shared memories (the paper's "load each link once
//    and reuse it across the rhs", across SMs).  Consumers release a link slot by arriving on the
//    empty barrier of every CTA of the cluster.
//  * The 16 hops are split between two warp sets with private accumulators: set A does the 8 x/y hops from the
//    window, set B the 8 z/t hops from the sub-stage ring; B hands its partial sums to A through shared memory once
//    per tile.  Two independent instruction streams per SM sub-partition hide each other's shared-memory latency.
//  * The window is cyclic in y (virtual chunk c of a strip = memory chunk c mod chunks-per-strip), so the wrapped
//    y-neighbours of the first and last rows of a strip come from the window like all others.
#include "common.cuh"
#include "tma.cuh"

#include <cuda.h>

#include <algorithm>
#include <stdlib.h>
#include <string.h>
#include <vector>

#define WIN_CHUNK 32 /* sites per window chunk */
#ifndef WIN_HOP_UNROLL
#define WIN_HOP_UNROLL 1
#endif
static constexpr int HOP_UNROLL = WIN_HOP_UNROLL; // hop loops of the arithmetic warps (2 and 8 measured: no gain)

struct WinParams {
    Geom g;
    int N, parity;
    const void *wt;  // gather-form links of this output parity
    void *out;
    const void *xp;
    double a;
    const int4 *segs; // (first tile, one-past-last tile, first tile of the strip, last tile of the strip)
    int nseg;
    const int *done;
    int HcL;    // window reach below/above a tile, in chunks
    int WCH;    // window ring slots (chunks)
    int nzlog;  // log2 of the z/t stage ring depth
    int rllog;  // log2 of the link ring depth (2 or 3)
    int xover;  // 1: tiles do not start on x-row boundaries (64 % (X/2) != 0): x hops read the chunk below the tile
    int slim;   // 1: window without spare slots (chunks below the tile released after the y-3, y-1 hops)
    int opts;   // tuning bits (BKR_WIN_OPTS): 1 = L2 prefetch of the next tile's links, 2 = of its z/t stages (no gain measured)
    uint32_t off_win, off_zt, off_red, off_bar;
};

// ---------------------------------------------------------------- PTX helpers (cluster, tensor TMA)
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// arrive on the mbarrier at the same shared-memory offset in CTA `rank` of the cluster.  Default (.release.cta)
// semantics as in CUTLASS' ClusterBarrier::arrive: with .release.cluster ptxas emits MEMBAR.ALL.GPU + ERRBAR per arrive
// (measured: 4.6x slower kernel); the slot was only read, by shared-memory loads that have already returned.
__device__ __forceinline__ void mbar_arrive_remote(uint64_t *bar, uint32_t rank)
{
    asm volatile("{\n\t.reg .b32 ra;\n\tmapa.shared::cluster.u32 ra, %0, %1;\n\t"
                 "mbarrier.arrive.shared::cluster.b64 _, [ra];\n\t}" ::"r"(smem_addr(bar)),
                 "r"(rank)
                 : "memory");
}
__device__ __forceinline__ void tma_load_1d_mc(void *dst, const void *src, uint32_t bytes, uint64_t *bar, uint16_t mask,
                                               uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster.L2::cache_hint "
                 "[%0], [%1], %2, [%3], %4, %5;" ::"r"(smem_addr(dst)),
                 "l"(src), "r"(bytes), "r"(smem_addr(bar)), "h"(mask), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, uint64_t *bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
                     smem_addr(dst)),
                 "l"(tm), "r"(smem_addr(bar)), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void tma_prefetch_1d(const void *src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_prefetch_3d(const CUtensorMap *tm, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];" ::"l"(tm), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void mbar_wait_mem(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(smem_addr(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void mbar_arrive_mem(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}

// acc_a += W_ab v_b for one rhs: u[a] = W_ab (a = 0..2), v = in_b
template <typename Real, typename Cx> __device__ __forceinline__ void cfma3(Real (&acc)[6], const Cx (&u)[3], const Cx v)
{
#pragma unroll
    for (int aa = 0; aa < 3; aa++) {
        acc[2 * aa] = fma(u[aa].x, v.x, acc[2 * aa]);
        acc[2 * aa + 1] = fma(u[aa].x, v.y, acc[2 * aa + 1]);
    }
#pragma unroll
    for (int aa = 0; aa < 3; aa++) {
        acc[2 * aa] = fma(-u[aa].y, v.y, acc[2 * aa]);
        acc[2 * aa + 1] = fma(u[aa].y, v.x, acc[2 * aa + 1]);
    }
}

// blockDim = (4 G + 4) warps: warps [0, 2G) = set A (x/y hops), [2G, 4G) = set B (z/t hops), last 4 warps = producers.
// Inside a set, warp w handles sites (w % 4) * 16 + lane % 16 of the 64-site tile and the rhs groups 2 (w / 4) + lane / 16
// (T rhs each); for odd G: rhs group w / 2 and sites (w % 2) * 32 + lane.
template <typename Real, int T, int G, int C, bool XP>
__global__ void __launch_bounds__((4 * G + 4) * 32, 1)
dslash_win_kernel(const __grid_constant__ CUtensorMap tm_win, const __grid_constant__ CUtensorMap tm_zt,
                  const __grid_constant__ CUtensorMap tm_xp, const WinParams p)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int NC = T * G;
    constexpr int NWS = 2 * G;
    constexpr uint32_t LSTAGE = 9 * 64 * sizeof(Cx);
    constexpr uint32_t WCHUNK = NC * 3 * WIN_CHUNK * sizeof(Cx);
    constexpr uint32_t ZSTAGE = NC * 3 * 64 * sizeof(Cx); // one z/t hop: [rhs][colour][64 sites]
    extern __shared__ __align__(1024) unsigned char dsm[];
    unsigned char *const lnk = dsm;
    unsigned char *const win = dsm + p.off_win;
    unsigned char *const zt = dsm + p.off_zt;
    Cx *const red = reinterpret_cast<Cx *>(dsm + p.off_red); // [NC * 3][64]
    uint64_t *const bar = reinterpret_cast<uint64_t *>(dsm + p.off_bar);
    uint64_t *const lfull = bar, *const lempty = bar + 8, *const wfull = bar + 16, *const wempty = bar + 32,
                    *const zfull = bar + 48, *const zempty = bar + 56, *const redfull = bar + 64, *const redempty = bar + 65;
    if (p.done && *p.done) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nzlog = p.nzlog, NZ = 1 << nzlog, rllog = p.rllog, RL = 1 << rllog, WCH = p.WCH, HcL = p.HcL;
    if (threadIdx.x == 0) {
        for (int s = 0; s < RL; s++) {
            mbar_init(&lfull[s], 1);
            mbar_init(&lempty[s], NWS * C);
        }
        for (int s = 0; s < WCH; s++) {
            mbar_init(&wfull[s], 1);
            mbar_init(&wempty[s], NWS);
        }
        for (int s = 0; s < NZ; s++) {
            mbar_init(&zfull[s], 1);
            mbar_init(&zempty[s], NWS);
        }
        mbar_init(redfull, NWS * 32);
        mbar_init(redempty, NWS * 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (C > 1) cluster_sync_all();
    else __syncthreads();

    const uint32_t rank = C > 1 ? cluster_ctarank() : 0u;
    const int cid = blockIdx.x / C, ncl = gridDim.x / C;
    const Geom &g = p.g;
    const int Xh = g.X[0] >> 1;
    const int Vh = g.Vh;

    constexpr int npt = XP ? 9 : 8; // z/t ring stages per tile: 8 hops + the xp tile of the epilogue
    const bool dry = (p.opts & 4) != 0; // tuning probe: no producers, no barriers (results are garbage)
    if (warp >= 2 * NWS) {
        // ------------------------------------------------------------------ producers: one lane in each of 4 warps
        //   role 0: link stages of set A (even sequence numbers)
        //   role 1: link stages of set B (odd sequence numbers)
        //   role 2: z/t neighbour stages (and the xp tile of the epilogue)
        //   role 3: window chunks
        // Each ring has its own in-order issuer, so a full ring never blocks the refill of another one.  Every
        // stage is also requested into L2 one tile ahead (cp.async.bulk.prefetch.L2): the HBM latency is paid there,
        // the shared-memory rings only have to cover the L2 -> SM latency.
        const int role = warp - 2 * NWS;
        if (lane == 0 && !dry) {
            const uint64_t pol = policy_evict_first();
            const Cx *wt = reinterpret_cast<const Cx *>(p.wt);
            const int XhY = Xh * g.X[1];
            constexpr uint32_t SL = LSTAGE / C; // this CTA's slice of a link stage
            // neighbour tile start (even-odd index) of tile k for z/t hop h
            auto zt_src = [&](int k, int h) {
                const int e0 = k * 64;
                const int zc = (e0 / XhY) % g.X[2], tcd = e0 / (XhY * g.X[2]);
                const int mu = BKR_HOP_MU(h), hop = BKR_HOP_LONG(h) ? 3 : 1;
                const int cm = mu == 2 ? zc : tcd, Xm = mu == 2 ? g.X[2] : g.X[3];
                const int smh = mu == 2 ? XhY : XhY * g.X[2];
                int cn = BKR_HOP_BACK(h) ? cm - hop : cm + hop;
                if (cn < 0) cn += Xm;
                if (cn >= Xm) cn -= Xm;
                return e0 + (cn - cm) * smh;
            };
            int tc = 0, wslot = 0, wuse = 0;
            for (int si = cid; si < p.nseg; si += ncl) {
                const int4 sg = p.segs[si];
                const int seg_lo = 2 * sg.x - HcL, seg_hi = 2 * sg.y - 1 + HcL; // virtual (cyclic in y) chunks
                const int cs = 2 * sg.z, ncs = 2 * (sg.w - sg.z + 1);
                auto chunk_site0 = [&](int c, int cs_, int ncs_) { // memory site of virtual chunk c of a strip
                    int r = (c - cs_) % ncs_;
                    if (r < 0) r += ncs_;
                    return (cs_ + r) * WIN_CHUNK;
                };
                const bool has_next = si + ncl < p.nseg;
                int4 sn = sg;
                if (has_next) sn = p.segs[si + ncl];
                int next_c = seg_lo;
                for (int k = sg.x; k < sg.y; k++, tc++) {
                    const int knext = k + 1 < sg.y ? k + 1 : (has_next ? sn.x : -1); // this CTA's next tile
                    if (role == 2) {
                        for (int j = 0; j < npt; j++) {
                            const int zs = npt * tc + j, slot = zs & (NZ - 1), use = zs >> nzlog;
                            if (use > 0) mbar_wait(&zempty[slot], (use - 1) & 1);
                            mbar_expect_tx(&zfull[slot], ZSTAGE);
                            if (j < 8) tma_load_3d(zt + (size_t)slot * ZSTAGE, &tm_zt, 2 * zt_src(k, 8 + j), 0, (int)rank * NC, &zfull[slot]);
                            else tma_load_3d(zt + (size_t)slot * ZSTAGE, &tm_xp, 2 * k * 64, 0, (int)rank * NC, &zfull[slot]);
                            if (j < 8 && knext >= 0 && (p.opts & 2)) tma_prefetch_3d(&tm_zt, 2 * zt_src(knext, 8 + j), 0, (int)rank * NC);
                        }
                        continue;
                    }
                    if (role == 3) {
                        // window chunks, up to what the NEXT tile needs, as far ahead as free slots allow
                        const int hi = min(2 * k + 3 + HcL, seg_hi);
                        while (next_c <= hi) {
                            if (wuse > 0) mbar_wait(&wempty[wslot], (wuse - 1) & 1);
                            mbar_expect_tx(&wfull[wslot], WCHUNK);
                            tma_load_3d(win + (size_t)wslot * WCHUNK, &tm_win, 2 * chunk_site0(next_c, cs, ncs), 0, (int)rank * NC, &wfull[wslot]);
                            next_c++;
                            if (++wslot == WCH) {
                                wslot = 0;
                                wuse++;
                            }
                        }
                        if (k == sg.y - 1 && has_next) // first window of the next segment -> L2
                            for (int cc = 2 * sn.x - HcL; cc <= 2 * sn.x + 1 + HcL; cc++)
                                tma_prefetch_3d(&tm_win, 2 * chunk_site0(cc, 2 * sn.z, 2 * (sn.w - sn.z + 1)), 0, (int)rank * NC);
                        continue;
                    }
                    for (int j = 0; j < 8; j++) {
                        const int h = role ? 8 + j : j;
                        const int ls = 16 * tc + 2 * j + role, slot = ls & (RL - 1), use = ls >> rllog;
                        if (use > 0) mbar_wait(&lempty[slot], (use - 1) & 1);
                        mbar_expect_tx(&lfull[slot], LSTAGE);
                        const unsigned char *src = reinterpret_cast<const unsigned char *>(wt + ((size_t)k * 16 + h) * 9 * 64);
                        if (C == 1)
                            tma_load_1d_hint(lnk + (size_t)slot * LSTAGE, src, LSTAGE, &lfull[slot], pol);
                        else
                            tma_load_1d_mc(lnk + (size_t)slot * LSTAGE + rank * SL, src + rank * SL, SL, &lfull[slot],
                                           (uint16_t)((1u << C) - 1u), pol);
                        if (knext >= 0 && (p.opts & 1))
                            tma_prefetch_1d(reinterpret_cast<const unsigned char *>(wt + ((size_t)knext * 16 + h) * 9 * 64) + rank * SL, SL);
                    }
                }
            }
        }
    } else if (warp < NWS) {
        // ------------------------------------------------------------------ set A: x/y hops from the window
        // The window is cyclic in y: virtual chunk c of a strip is memory chunk cs + (c - cs) mod ncs, so the wrapped
        // neighbours of the first and last rows of a strip are served like all others (no global loads here at all).
        // lanes 0-15 and 16-31 of a warp: the same 16 sites, two rhs groups -- the link loads of the two half-warps hit the
        // same shared-memory addresses (one broadcast wavefront pair instead of two): half the link traffic on the port
        const int sl = (G % 2 == 0) ? (warp & 3) * 16 + (lane & 15) : (warp & 1) * 32 + lane;
        const int j0 = (G % 2 == 0) ? (2 * (warp >> 2) + (lane >> 4)) * T : (warp >> 1) * T;
        int tc = 0, q0 = 0;
        for (int si = cid; si < p.nseg; si += ncl) {
            const int4 sg = p.segs[si];
            const int seg_lo = 2 * sg.x - HcL, seg_hi = 2 * sg.y - 1 + HcL; // virtual chunks of this segment
            const int strip_sites = (sg.w - sg.z + 1) * 64;
            int waited = seg_lo, released = seg_lo;
            for (int k = sg.x; k < sg.y; k++, tc++) {
                const int whi = 2 * k + 1 + HcL;
                while (waited <= whi) {
                    const int qq = q0 + waited - seg_lo;
                    if (!dry) mbar_wait(&wfull[qq % WCH], (qq / WCH) & 1);
                    waited++;
                }
                const int slot2k = (q0 + 2 * k - seg_lo) % WCH;
                const int e = k * 64 + sl;
                int s = 2 * e;
                int c0, c1;
                {
                    const int x0 = s % g.X[0];
                    int r = s / g.X[0];
                    c1 = r % g.X[1];
                    r /= g.X[1];
                    const int c2 = r % g.X[2], c3 = r / g.X[2];
                    c0 = x0 + ((c1 + c2 + c3 + p.parity) & 1);
                    s = s - x0 + c0;
                }
                Real acc[T][6];
#pragma unroll
                for (int i = 0; i < T; i++)
#pragma unroll
                    for (int qd = 0; qd < 6; qd++) acc[i][qd] = (Real)0;
#pragma unroll HOP_UNROLL
                for (int h = 0; h < 8; h++) {
                    const int mu = BKR_HOP_MU(h), hop = BKR_HOP_LONG(h) ? 3 : 1;
                    const int cm = mu == 0 ? c0 : c1, Xm = mu == 0 ? g.X[0] : g.X[1], smh = mu == 0 ? 1 : g.X[0];
                    int cn = BKR_HOP_BACK(h) ? cm - hop : cm + hop;
                    if (cn < 0) cn += Xm;
                    if (cn >= Xm) cn -= Xm;
                    // neighbour position relative to the tile start, moved to its cyclic image inside the window
                    int d = ((s + (cn - cm) * smh) >> 1) - k * 64;
                    if (d >= 64 + WIN_CHUNK * HcL) d -= strip_sites;
                    if (d < -WIN_CHUNK * HcL) d += strip_sites;
                    int sidx = slot2k + (d >> 5); // arithmetic shift = floor
                    if (sidx < 0) sidx += WCH;
                    if (sidx >= WCH) sidx -= WCH;
                    const Cx *wp = reinterpret_cast<const Cx *>(win + (size_t)sidx * WCHUNK) + j0 * 3 * WIN_CHUNK + (d & 31);
                    const int ls = 16 * tc + 2 * h, slot = ls & (RL - 1);
                    const Cx(*lk)[64] = reinterpret_cast<const Cx(*)[64]>(lnk + (size_t)slot * LSTAGE);
                    if (!dry) mbar_wait(&lfull[slot], (ls >> rllog) & 1);
                    // the whole 3 x 3 matrix goes to registers and the slot back to the producer before the arithmetic:
                    // the ring then holds (almost) only data in flight
                    Cx u[3][3]; // u[b][a] = W_ab
#pragma unroll
                    for (int b = 0; b < 3; b++)
#pragma unroll
                        for (int aa = 0; aa < 3; aa++) u[b][aa] = lds_cx(&lk[aa * 3 + b][sl]);
                    __syncwarp();
                    if (lane == 0 && !dry) {
                        if (C == 1) mbar_arrive(&lempty[slot]);
                        else
                            for (uint32_t r = 0; r < (uint32_t)C; r++) mbar_arrive_remote(&lempty[slot], r);
                    }
#pragma unroll
                    for (int b = 0; b < 3; b++) {
                        Cx v[T];
#pragma unroll
                        for (int i = 0; i < T; i++) v[i] = lds_cx(wp + (i * 3 + b) * WIN_CHUNK);
#pragma unroll
                        for (int i = 0; i < T; i++) cfma3<Real, Cx>(acc[i], u[b], v[i]);
                    }
                    if (h == 1 && p.slim) {
                        // hops 0, 1 are y-3, y-1 (common.cuh): the chunks below the tile are dead from here on and go back
                        // to the window producer, which loads the next tile's upper chunks into them
                        const int new_rel = 2 * k - p.xover; // x neighbours reach 2 sites below a tile that starts mid-row
                        __syncwarp();
                        if (lane == 0 && !dry)
                            for (int cc = released; cc < new_rel; cc++) mbar_arrive(&wempty[(q0 + cc - seg_lo) % WCH]);
                        released = max(released, new_rel);
                    }
                }
                // release the window chunks the next tile of this segment does not need
                {
                    const int new_rel = (k == sg.y - 1) ? seg_hi + 1 : 2 * (k + 1) - HcL;
                    __syncwarp();
                    if (lane == 0 && !dry)
                        for (int cc = released; cc < new_rel; cc++) mbar_arrive(&wempty[(q0 + cc - seg_lo) % WCH]);
                    released = max(released, new_rel);
                }
                // hand the partial sums to set B, which finishes the tile
                if (tc > 0 && !dry) mbar_wait_mem(redempty, (tc - 1) & 1);
#pragma unroll
                for (int i = 0; i < T; i++)
#pragma unroll
                    for (int cc = 0; cc < 3; cc++) {
                        Cx o;
                        o.x = acc[i][2 * cc];
                        o.y = acc[i][2 * cc + 1];
                        red[((j0 + i) * 3 + cc) * 64 + sl] = o;
                    }
                if (!dry) mbar_arrive_mem(redfull);
            }
            q0 += seg_hi - seg_lo + 1;
        }
    } else {
        // ------------------------------------------------------------------ set B: z/t hops from the sub-stage ring,
        // then the epilogue: add set A's partial sums, out = acc  or  a * xp - acc
        const int wb = warp - NWS;
        const int sl = (G % 2 == 0) ? (wb & 3) * 16 + (lane & 15) : (wb & 1) * 32 + lane;
        const int j0 = (G % 2 == 0) ? (2 * (wb >> 2) + (lane >> 4)) * T : (wb >> 1) * T;
        const int jg = (int)rank * NC + j0; // first global rhs of this thread
        int tc = 0;
        for (int si = cid; si < p.nseg; si += ncl) {
            const int4 sg = p.segs[si];
            for (int k = sg.x; k < sg.y; k++, tc++) {
                const int e = k * 64 + sl;
                Cx *vout = reinterpret_cast<Cx *>(p.out) + (size_t)jg * 3 * Vh + e;
                Real acc[T][6];
#pragma unroll
                for (int i = 0; i < T; i++)
#pragma unroll
                    for (int qd = 0; qd < 6; qd++) acc[i][qd] = (Real)0;
#pragma unroll HOP_UNROLL
                for (int j = 0; j < 8; j++) {
                    const int ls = 16 * tc + 2 * j + 1, slot = ls & (RL - 1);
                    const Cx(*lk)[64] = reinterpret_cast<const Cx(*)[64]>(lnk + (size_t)slot * LSTAGE);
                    if (!dry) mbar_wait(&lfull[slot], (ls >> rllog) & 1);
                    Cx u[3][3];
#pragma unroll
                    for (int b = 0; b < 3; b++)
#pragma unroll
                        for (int aa = 0; aa < 3; aa++) u[b][aa] = lds_cx(&lk[aa * 3 + b][sl]);
                    __syncwarp();
                    if (lane == 0 && !dry) {
                        if (C == 1) mbar_arrive(&lempty[slot]);
                        else
                            for (uint32_t r = 0; r < (uint32_t)C; r++) mbar_arrive_remote(&lempty[slot], r);
                    }
                    const int zs = npt * tc + j, zslot = zs & (NZ - 1);
                    const Cx *zp = reinterpret_cast<const Cx *>(zt + (size_t)zslot * ZSTAGE) + j0 * 3 * 64 + sl;
                    if (!dry) mbar_wait(&zfull[zslot], (zs >> nzlog) & 1);
#pragma unroll
                    for (int b = 0; b < 3; b++) {
                        Cx v[T];
#pragma unroll
                        for (int i = 0; i < T; i++) v[i] = lds_cx(zp + (i * 3 + b) * 64);
                        if (b == 2) {
                            __syncwarp();
                            if (lane == 0 && !dry) mbar_arrive(&zempty[zslot]);
                        }
#pragma unroll
                        for (int i = 0; i < T; i++) cfma3<Real, Cx>(acc[i], u[b], v[i]);
                    }
                }
                // xp operand of the epilogue: a ninth stage of the z/t ring (the producer copies the tile of xp behind
                // the eight neighbour stages), so no arithmetic warp ever waits on global memory.  (With 3 T plain loads
                // here the second half of M ran 1.83 ms against 1.38 ms for the bare stencil.)
                const int zsx = npt * tc + 8, zslotx = zsx & (NZ - 1);
                const Cx *zpx = reinterpret_cast<const Cx *>(zt + (size_t)zslotx * ZSTAGE) + j0 * 3 * 64 + sl;
                if (XP && !dry) mbar_wait(&zfull[zslotx], (zsx >> nzlog) & 1);
                if (!dry) mbar_wait_mem(redfull, tc & 1);
#pragma unroll
                for (int i = 0; i < T; i++) {
#pragma unroll
                    for (int cc = 0; cc < 3; cc++) {
                        const Cx rb = red[((j0 + i) * 3 + cc) * 64 + sl];
                        Cx o;
                        o.x = acc[i][2 * cc] + rb.x;
                        o.y = acc[i][2 * cc + 1] + rb.y;
                        if (XP) {
                            const Cx xv = lds_cx(zpx + (i * 3 + cc) * 64);
                            o.x = fma((Real)p.a, xv.x, -o.x);
                            o.y = fma((Real)p.a, xv.y, -o.y);
                        }
                        if (jg + i < p.N) __stcs(vout + (size_t)(i * 3 + cc) * Vh, o);
                    }
                }
                if (!dry) mbar_arrive_mem(redempty);
                __syncwarp();
                if (XP && lane == 0 && !dry) mbar_arrive(&zempty[zslotx]);
            }
        }
    }
    // no CTA may leave while a peer can still multicast into its shared memory or arrive on its barriers
    if (C > 1) cluster_sync_all();
}

// ---------------------------------------------------------------- host: tensor maps, segment order, dispatch

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)ptr;
        else
            cudaGetLastError();
    }
    return fn;
}

// view of a native block v[rhs][colour][site] as a rank-3 tensor of reals (2 Vh, 3, N); box = (2 box_sites, box_col, NC)
static bool make_map(CUtensorMap *tm, const void *base, int prec, int Vh, int N, int box_sites, int box_col, int NC)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const size_t rsz = prec == BKR_F64 ? 8 : 4;
    cuuint64_t gdim[3] = {(cuuint64_t)2 * Vh, 3, (cuuint64_t)N};
    cuuint64_t gstr[2] = {(cuuint64_t)2 * Vh * rsz, (cuuint64_t)6 * Vh * rsz};
    cuuint32_t box[3] = {(cuuint32_t)(2 * box_sites), (cuuint32_t)box_col, (cuuint32_t)NC};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(tm, prec == BKR_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3,
                    const_cast<void *>(base), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// Segments (runs of consecutive tiles inside one (z, t) strip) in the order they are handed to the clusters: z blocks
// outermost, then t, then the strips of the block, then the segments of a strip -- the clusters of the grid work on a
// window of consecutive entries, so the 7 time slices a z block needs for its t +- 1, +- 3 hops stay L2 resident
// (same idea as build_tile_order in dslash.cu; the block is the largest whose 7-slice working set fits the budget).
static int build_segments(bkr_ctx *ctx, int N, int prec, int seglen)
{
    const Geom &g = ctx->g;
    const int Xh = g.X[0] / 2, Y = g.X[1], Z = g.X[2], Tt = g.X[3];
    const double budget = (ctx->l2_budget_mb > 0 ? ctx->l2_budget_mb : 48) * 1e6;
    const double site_bytes = 3.0 * std::max(N, ctx->dslash_nblock) * (prec == BKR_F64 ? 16 : 8);
    int zb = 1;
    for (int c = 1; c <= Z; c++)
        if (Z % c == 0 && (7.0 * Xh * Y * c * site_bytes <= budget || Tt <= 7)) zb = c;
    const int key = zb * 64 + seglen;
    if (ctx->win_segs && ctx->win_key == key) return BKR_OK;
    const int ts = Xh * Y / 64; // tiles per strip
    std::vector<int4> segs;
    for (int zblk = 0; zblk < Z / zb; zblk++)
        for (int t = 0; t < Tt; t++)
            for (int zi = 0; zi < zb; zi++) {
                const int z = zblk * zb + zi;
                const int s0 = (t * Z + z) * ts, s1 = s0 + ts - 1;
                for (int k0 = s0; k0 <= s1; k0 += seglen) segs.push_back(make_int4(k0, std::min(k0 + seglen, s1 + 1), s0, s1));
            }
    if (ctx->win_segs) cudaFree(ctx->win_segs);
    ctx->win_segs = nullptr;
    BKR_CUDA(ctx, cudaMalloc((void **)&ctx->win_segs, segs.size() * sizeof(int4)));
    BKR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    BKR_CUDA(ctx, cudaMemcpy(ctx->win_segs, segs.data(), segs.size() * sizeof(int4), cudaMemcpyHostToDevice));
    ctx->win_nseg = (int)segs.size();
    ctx->win_key = key;
    return BKR_OK;
}

static const size_t WIN_SMEM_MAX = 232448;
// returns 1 if this instantiation cannot run the geometry (caller falls back), BKR_OK after a launch, else an error
template <typename Real, int T, int G, int C, bool XP>
static int launch_win_x(bkr_ctx *ctx, int parity, int N, int prec, const void *in, void *out, const void *xp, double a,
                        const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int NC = T * G;
    const Geom &g = ctx->g;
    const int Xh = g.X[0] / 2;
    WinParams p;
    memset(&p, 0, sizeof(p));
    p.HcL = (3 * Xh + WIN_CHUNK - 1) / WIN_CHUNK;
    {
        const char *e = getenv("BKR_WIN_SLIM");
        p.slim = e ? atoi(e) : 1;
    }
    p.xover = (64 % Xh) != 0 ? 1 : 0;
    p.WCH = 2 * p.HcL + 2 + (p.slim ? std::max(0, 2 - (p.HcL - p.xover)) : 2);
    if (p.WCH > 16) return 1;
    const size_t lstage = (size_t)9 * 64 * sizeof(Cx), wbytes = (size_t)p.WCH * NC * 3 * WIN_CHUNK * sizeof(Cx),
                 zstage = (size_t)NC * 3 * 64 * sizeof(Cx), rbytes = (size_t)NC * 3 * 64 * sizeof(Cx), bbytes = 66 * 8;
    // ring depths: as much data in flight as the 227 KB allow (the rings are what hides the ~1 us refill round trip);
    // measured at 32^3 x 64, N = 8: 4 link stages + 2 z/t hop stages 0.69 ms; 8 + 2: 0.72; 4 + 3: 0.74 -- deeper rings do
    // not help, the shared-memory port does the limiting
    const char *zenv = getenv("BKR_WIN_NZ"), *lenv = getenv("BKR_WIN_RL");
    int rl = lenv ? atoi(lenv) : 8, nz = zenv ? atoi(zenv) : 2;
    if (rl != 4 && rl != 8) rl = 8;
    if (nz != 1 && nz != 2 && nz != 4) nz = 2;
    while (rl * lstage + wbytes + nz * zstage + rbytes + bbytes > WIN_SMEM_MAX) {
        if (nz > 2) nz /= 2;
        else if (rl > 4) rl = 4;
        else if (nz > 1) nz /= 2;
        else return 1;
    }
    {
        // clusters of 3-4 CTAs need the deep link ring (the release -> refill round trip crosses SMs): with 4 stages the
        // plain kernel is faster (48^3 x 96, N = 32 fp64: 20.6 vs 19.1 ms), with 8 it is not (32^3 x 64: 3.02 vs 3.10 ms)
        if (C >= 3 && rl < 8 && ctx->dslash_force != 1) return 1;
    }
    if (nz < 2 && !getenv("BKR_WIN_ALLOW_NZ1")) return 1; // one z/t stage: slower than dslash.cu (48^4: 2.6 vs 2.1 ms)
    p.nzlog = nz == 4 ? 2 : nz == 2 ? 1 : 0;
    p.rllog = rl == 8 ? 3 : 2;
    const size_t lbytes = rl * lstage;
    p.off_win = (uint32_t)lbytes;
    p.off_zt = (uint32_t)(lbytes + wbytes);
    p.off_red = (uint32_t)(p.off_zt + nz * zstage);
    p.off_bar = (uint32_t)(p.off_red + rbytes);
    const size_t smem = p.off_bar + bbytes;

    const char *senv = getenv("BKR_WIN_SEGLEN");
    BKR_TRY(build_segments(ctx, N, prec, senv ? std::max(1, atoi(senv)) : 8));
    CUtensorMap tm_win, tm_zt, tm_xp;
    if (!make_map(&tm_win, in, prec, g.Vh, N, WIN_CHUNK, 3, NC) || !make_map(&tm_zt, in, prec, g.Vh, N, 64, 3, NC) ||
        !make_map(&tm_xp, xp ? xp : in, prec, g.Vh, N, 64, 3, NC))
        return 1;

    const int ntiles = link_tiles(g);
    p.g = g;
    p.N = N;
    p.parity = parity;
    p.wt = (sizeof(Real) == 8 ? (const Cx *)ctx->links64 : (const Cx *)ctx->links32) + (size_t)parity * ntiles * 16 * 9 * 64;
    p.out = out;
    p.xp = xp;
    p.a = a;
    p.segs = ctx->win_segs;
    p.nseg = ctx->win_nseg;
    p.done = done;
    {
        const char *oenv = getenv("BKR_WIN_OPTS");
        p.opts = oenv ? atoi(oenv) : 0;
    }

    auto kern = dslash_win_kernel<Real, T, G, C, XP>;
    static int max_clusters = -1, attr_dev = -1; // per instantiation; the shared-memory opt-in is per device
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3((4 * G + 4) * 32);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = ctx->stream;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (max_clusters < 0 || attr_dev != ctx->device) {
        attr_dev = ctx->device;
        BKR_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)WIN_SMEM_MAX));
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
    if (getenv("BKR_WIN_DEBUG"))
        fprintf(stderr, "dslash_win: C=%d max_clusters=%d nseg=%d smem=%zu WCH=%d nz=%d rl=%d\n", C, max_clusters, p.nseg, smem, p.WCH, nz, rl);
    cfg.gridDim = dim3((unsigned)(std::min(max_clusters, p.nseg) * C));
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, tm_win, tm_zt, tm_xp, p);
    if (e != cudaSuccess) {
        ctx->last_cuda = (int)e;
        return BKR_ECUDA;
    }
    return bkr_check_launch(ctx);
}

template <typename Real, int T, int G, int C>
static int launch_win_c(bkr_ctx *ctx, int parity, int N, int prec, const void *in, void *out, const void *xp, double a,
                        const int *done)
{
    if (xp) return launch_win_x<Real, T, G, C, true>(ctx, parity, N, prec, in, out, xp, a, done);
    return launch_win_x<Real, T, G, C, false>(ctx, parity, N, prec, in, out, xp, a, done);
}

// 1 = not applicable (caller uses dslash.cu's kernel)
int launch_dslash_win(bkr_ctx *ctx, int out_parity, int N, int prec, const void *in, void *out, const void *xp, double a,
                      const int *done)
{
    const int mode = ctx->dslash_force == 1 ? 2 : 1; // 1: automatic, 2: whenever the geometry allows (bkr_set_dslash_variant)
    const Geom &g = ctx->g;
    const int Xh = g.X[0] / 2;
    if (mode == 0 || (Xh * g.X[1]) % 64 != 0) return 1;
    // Automatic mode: a cluster of C CTAs costs about C times the NC-rhs kernel whatever N is, the plain kernel of
    // dslash.cu costs ~N; measured crossover at 32^3 x 64: within 2 rhs (fp64) / 3 rhs (fp32) of
    // a full cluster.
    if (prec == BKR_F64) {
        const int C = (N + 7) / 8;
        if (mode == 1 && (N < 7 || 8 * C - N > 2)) return 1;
        if (getenv("BKR_WIN_T8")) { // tuning probe
            if (C == 1) return launch_win_c<double, 8, 1, 1>(ctx, out_parity, N, prec, in, out, xp, a, done);
            if (C == 2) return launch_win_c<double, 8, 1, 2>(ctx, out_parity, N, prec, in, out, xp, a, done);
        }
        if (C == 1) return launch_win_c<double, 4, 2, 1>(ctx, out_parity, N, prec, in, out, xp, a, done);
        if (C == 2) return launch_win_c<double, 4, 2, 2>(ctx, out_parity, N, prec, in, out, xp, a, done);
        if (C == 3) return launch_win_c<double, 4, 2, 3>(ctx, out_parity, N, prec, in, out, xp, a, done);
        if (C == 4) return launch_win_c<double, 4, 2, 4>(ctx, out_parity, N, prec, in, out, xp, a, done);
        return 1;
    }
    const int C = (N + 15) / 16;
    if (mode == 1 && (N < 13 || 16 * C - N > 3)) return 1;
    if (C == 1) return launch_win_c<float, 8, 2, 1>(ctx, out_parity, N, prec, in, out, xp, a, done);
    if (C == 2) return launch_win_c<float, 8, 2, 2>(ctx, out_parity, N, prec, in, out, xp, a, done);
    return 1;
}
