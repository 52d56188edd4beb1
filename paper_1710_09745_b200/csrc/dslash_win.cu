// Multi-rhs improved-staggered stencil, "window" version for N >= ~6 (eq. 2).
//
//   out(x) = sum_h W_h(x) in(nbr_h(x)),  16 hops;  optional epilogue out = a * xp - out
//
// Why a second kernel.  With every neighbour vector fetched from L2 by plain loads
// (dslash.cu) each input element crosses the L2 -> SM fabric 16 times per call and the per-hop footprint (N x 48
// bytes per site) is too large for L1 to hold between hops; the reuse the paper got from the texture cache
// is made explicit:
//  * A CTA walks a run of consecutive 64-site tiles inside one (z, t) "strip" (all x, y at fixed z, t).  The x- and
//    y-neighbours of a tile lie within +-3 x-rows of it, so a sliding WINDOW of input rows in shared memory serves
//    all 8 x/y hops: every input row is fetched from L2 once per strip instead of 8 times.  z/t hops still cost one
//    L2 fetch each: 9 fetches per site instead of 16.
//  * Apart from the xpay operand (3 T / 2 streaming loads per thread, issued at the start of a tile), nothing is loaded
//    from global memory by the arithmetic warps.  Producer lanes (one per warp of two producer warpgroups, 48 registers
//    each after setmaxnreg) feed two shared-memory rings with TMA.  The HOP-STAGE ring holds, per hop pair (h, 8 + h)
//    of a tile, the links of both hops (1-D bulk copies, 9 x 64 complex each) and the z/t neighbour tile of hop 8 + h
//    as two 32-site chunks (3-D tensor copies: 32 sites x 3 colours x NC rhs); the four parts have one lane each (a
//    lane issues at most one bulk copy per ~360 cycles) and complete on ONE full barrier.  The WINDOW ring holds the
//    32-site chunks of the strip.
//  * A CTA holds NC = 2 T rhs (8 in fp64, 16 in fp32).  For N > NC a thread-block CLUSTER of C = ceil(N / NC) CTAs
//    works on the same tiles, one rhs slice each, and every link stage is fetched ONCE for the cluster: each CTA
//    issues 1/C of the stage as a multicast bulk copy into all C shared memories (the paper's "load each link once
//    and reuse it across the rhs", across SMs).  Consumers release a link slot by arriving on the
//    empty barrier of every CTA of the cluster.
//  * The 16 hops are split inside every arithmetic warp: lanes 0-15 do the 8 x/y hops of 16 sites from the window,
//    lanes 16-31 the 8 z/t hops of the same 16 sites from the stage ring -- one instruction stream, only the
//    operand addresses differ -- and the two partial sums meet through 6 T warp shuffles per lane; each half then
//    stores half of the rhs.  (Round 1 gave the two hop sets to different warps, which met through a 24 KB
//    shared-memory buffer and a pair of barriers; the buffer and the barriers are gone.)
//  * The window is cyclic in y (virtual chunk c of a strip = memory chunk c mod chunks-per-strip), so the wrapped
//    y-neighbours of the first and last rows of a strip come from the window like all others.
// What the box measured and this kernel is built around (profiles/r2_onchip_probes.md):
//  * every LDS.128 return costs 4-5 cycles of the register-file write port of its scheduler, the same port the DFMA
//    results use, broadcast or not; with operands from shared memory the FP64 pipe tops out at ~48 of 64 DFMA/clk/SM
//    for T = 4, 6, 8 alike;
//  * TMA fills do not compete with LDS for the shared-memory port (3 % loss), plain global loads do (1:1);
//  * a TMA round trip is 500-700 cycles from L2 on an idle chip, 1300-2500 under load: ring depth decides whether the
//    arithmetic warps wait;
//  * cp.async.bulk.prefetch.L2 of the link stream one to three tiles ahead made the kernel 20-50 % SLOWER (tried
//    twice, with and without the evict-first policy) and is not used.
#include "common.cuh"
#include "tma.cuh"

#include <cuda.h>

#include <algorithm>
#include <stdlib.h>
#include <string.h>
#include <type_traits>
#include <vector>

#define WIN_CHUNK 32 /* sites per window chunk */
#define WIN_CONSUMER_WARPS 8
#define WIN_PRODUCER_WARPS 8
#define WIN_THREADS ((WIN_CONSUMER_WARPS + WIN_PRODUCER_WARPS) * 32)
#define WIN_CONSUMER_REGS 208 /* 256 x 208 + 256 x 48 = 65536 */

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
    int D;      // hop-stage ring depth
    int xover;  // 1: tiles do not start on x-row boundaries (64 % (X/2) != 0): x hops read the chunk below the tile
    int slim;   // 1: window without spare slots (chunks below the tile released after the y-3, y-1 hops)
    uint32_t off_win, off_bar;
    uint32_t zero; // 0 at run time, unknown to the compiler: ties a barrier arrival to the registers of the loads it follows
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
// blocking wait with a long suspend-time hint: the thread sleeps in hardware until the phase completes instead of
// spinning (ncu: with the default hint the producer lanes executed a third of all instructions of the kernel and
// took issue slots from the arithmetic warps of their schedulers)
__device__ __forceinline__ void mbar_wait_slow(uint64_t *bar, uint32_t parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}" ::"r"(
                     smem_addr(bar)),
                 "r"(parity), "r"(0x989680)
                 : "memory");
}
// one non-blocking probe of a barrier phase (test_wait); the result is consumed later (mbar_finish) so that FMAs can
// issue in between
__device__ __forceinline__ uint32_t mbar_try(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok)
                 : "r"(smem_addr(bar)), "r"(parity));
    return ok;
}
__device__ __forceinline__ void mbar_finish(uint32_t ok, uint64_t *bar, uint32_t parity)
{
    if (!ok)
        asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}" ::"r"(
                         smem_addr(bar)),
                     "r"(parity), "r"(0x989680));
}
// streaming 16 / 8-byte global load of the xpay operand (read once per call)
__device__ __forceinline__ double2 ldg_stream(const double2 *p)
{
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ float2 ldg_stream(const float2 *p)
{
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

// acc[i] += W(:, b) v_i(b) for the T rhs of a thread: u[a] = W_ab, v[i] = component b of rhs i
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
// 16 / 8-byte shared-memory load at a shared-space address plus an immediate offset
template <typename Cx> __device__ __forceinline__ Cx lds_at(uint32_t addr, uint32_t off);
template <> __device__ __forceinline__ double2 lds_at<double2>(uint32_t addr, uint32_t off)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr + off));
    return v;
}
template <> __device__ __forceinline__ float2 lds_at<float2>(uint32_t addr, uint32_t off)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr + off));
    return v;
}
__device__ __forceinline__ uint32_t lo_bits(double v) { return (uint32_t)__double2loint(v); }
__device__ __forceinline__ uint32_t lo_bits(float v) { return __float_as_uint(v); }
__device__ __forceinline__ double shfl_x16(double v) { return __shfl_xor_sync(0xffffffffu, v, 16); }
__device__ __forceinline__ float shfl_x16(float v) { return __shfl_xor_sync(0xffffffffu, v, 16); }

// blockDim = 16 warps: warps 0-7 arithmetic, warps 8-15 producers (lane 0 of warps 8-13 works).
// Arithmetic warp w: sites (w % 4) * 16 + lane % 16 of the 64-site tile, rhs group w / 4 (T rhs), hop set lane / 16.
// A HOP STAGE of the ring holds everything hop pair (h, 8 + h) of a tile needs besides the window:
//   [ links of hop h : 9 x 64 | links of hop 8 + h : 9 x 64 | z/t neighbours of hop 8 + h: 2 chunks of NC x 3 x 32 ]
// filled by four producer lanes (one bulk / tensor copy each) that signal ONE full barrier, released by ONE arrival
// per arithmetic warp (per CTA of the cluster: the link parts are multicast).
template <typename Real, int T, int C, bool XP>
__global__ void __launch_bounds__(WIN_THREADS, 1)
dslash_win_kernel(const __grid_constant__ CUtensorMap tm_win, const WinParams p)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int NC = 2 * T;
    constexpr int NW = WIN_CONSUMER_WARPS;
    constexpr uint32_t LSTAGE = 9 * 64 * sizeof(Cx);
    constexpr uint32_t WCHUNK = NC * 3 * WIN_CHUNK * sizeof(Cx);
    constexpr uint32_t HSTAGE = 2 * LSTAGE + 2 * WCHUNK;
    constexpr uint32_t PLANE = WIN_CHUNK * sizeof(Cx); // bytes between the (rhs, colour) planes of a chunk
    extern __shared__ __align__(1024) unsigned char dsm[];
    unsigned char *const stg = dsm;
    unsigned char *const win = dsm + p.off_win;
    uint64_t *const bar = reinterpret_cast<uint64_t *>(dsm + p.off_bar);
    uint64_t *const hfull = bar, *const hempty = bar + 8, *const wfull = bar + 16, *const wempty = bar + 32;
    if (p.done && *p.done) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int D = p.D, WCH = p.WCH, HcL = p.HcL;
    if (threadIdx.x == 0) {
        for (int s = 0; s < D; s++) {
            mbar_init(&hfull[s], 4);
            mbar_init(&hempty[s], NW * C);
        }
        for (int s = 0; s < WCH; s++) {
            mbar_init(&wfull[s], 1);
            mbar_init(&wempty[s], NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (C > 1) cluster_sync_all();
    else __syncthreads();

    const uint32_t rank = C > 1 ? cluster_ctarank() : 0u;
    const int cid = blockIdx.x / C, ncl = gridDim.x / C;
    const Geom &g = p.g;
    const int Xh = g.X[0] >> 1;
    const int Vh = g.Vh;
    const int XhY = Xh * g.X[1];

    if (warp >= NW) {
        // ------------------------------------------------------------------ producers: lane 0 of five warps
        //   role 0: links of the x/y hops        role 1: links of the z/t hops
        //   role 2, 3: lower / upper 32-site chunk of the z/t neighbour tile
        //   role 4: window chunks
        // (one lane issues at most one bulk copy per ~360 cycles, measured: hence one lane per part of a stage)
        asm volatile("setmaxnreg.dec.sync.aligned.u32 48;");
        const int role = warp - NW;
        if (lane == 0 && role < 5) {
            const uint64_t pol = policy_evict_first();
            const Cx *wt = reinterpret_cast<const Cx *>(p.wt);
            constexpr uint32_t SL = LSTAGE / C; // this CTA's slice of a link stage
            int wslot = 0, wuse = 0;
            int hslot = 0, huse = 0; // hop-stage ring position (roles 0-3)
            for (int si = cid; si < p.nseg; si += ncl) {
                const int4 sg = p.segs[si];
                const int seg_lo = 2 * sg.x - HcL, seg_hi = 2 * sg.y - 1 + HcL; // virtual (cyclic in y) chunks
                const int cs = 2 * sg.z, ncs = 2 * (sg.w - sg.z + 1);
                int next_c = seg_lo;
                // z/t neighbour offsets (in sites) of the strip, hop j = 0..7: z-3, z-1, z+1, z+3, t-3, t-1, t+1, t+3
                const int zc = (sg.z * 64 / XhY) % g.X[2], tcd = sg.z * 64 / (XhY * g.X[2]);
                for (int k = sg.x; k < sg.y; k++) {
                    if (role == 4) {
                        // window chunks, up to what the NEXT tile needs, as far ahead as free slots allow
                        const int hi = min(2 * k + 3 + HcL, seg_hi);
                        while (next_c <= hi) {
                            int r = (next_c - cs) % ncs; // memory chunk of virtual chunk next_c of the strip
                            if (r < 0) r += ncs;
                            if (wuse > 0) mbar_wait_slow(&wempty[wslot], (wuse - 1) & 1);
                            mbar_expect_tx(&wfull[wslot], WCHUNK);
                            tma_load_3d(win + (size_t)wslot * WCHUNK, &tm_win, 2 * (cs + r) * WIN_CHUNK, 0, (int)rank * NC, &wfull[wslot]);
                            next_c++;
                            if (++wslot == WCH) {
                                wslot = 0;
                                wuse++;
                            }
                        }
                        continue;
                    }
                    for (int j = 0; j < 8; j++) {
                        if (huse > 0) mbar_wait_slow(&hempty[hslot], (huse - 1) & 1);
                        unsigned char *const sb = stg + (size_t)hslot * HSTAGE;
                        if (role < 2) {
                            const int h = role ? 8 + j : j;
                            unsigned char *const dst = sb + role * LSTAGE;
                            mbar_expect_tx(&hfull[hslot], LSTAGE);
                            const unsigned char *src = reinterpret_cast<const unsigned char *>(wt + ((size_t)k * 16 + h) * 9 * 64);
                            if (C == 1) tma_load_1d_hint(dst, src, LSTAGE, &hfull[hslot], pol);
                            else tma_load_1d_mc(dst + rank * SL, src + rank * SL, SL, &hfull[hslot], (uint16_t)((1u << C) - 1u), pol);
                        } else {
                            const bool isz = j < 4;
                            const int hop = 2 * (j & 3) - 3;
                            const int cm = isz ? zc : tcd, Xm = isz ? g.X[2] : g.X[3];
                            int cn = cm + hop;
                            if (cn < 0) cn += Xm;
                            if (cn >= Xm) cn -= Xm;
                            const int e0 = k * 64 + (cn - cm) * (isz ? XhY : XhY * g.X[2]) + (role - 2) * WIN_CHUNK;
                            mbar_expect_tx(&hfull[hslot], WCHUNK);
                            tma_load_3d(sb + 2 * LSTAGE + (role - 2) * WCHUNK, &tm_win, 2 * e0, 0, (int)rank * NC, &hfull[hslot]);
                        }
                        if (++hslot == D) {
                            hslot = 0;
                            huse++;
                        }
                    }
                }
            }
        }
    } else {
        // ------------------------------------------------------------------ arithmetic warps
        // Software pipeline: the operands of a COLUMN are 3 link elements W_ab, a = 0..2, and the T vector elements of colour
        // b, for 12 T FMAs.  Column 0 of a hop is loaded (register set A) during column 2 of the hop before, columns 1 and 2
        // (sets B, C) at the start of the hop, the barrier probe of the next stage a column ahead; the hop index is a
        // compile-time constant (a runtime hop loop cost 280 non-FMA instructions per hop and warp, ncu).
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(WIN_CONSUMER_REGS));
        const int set = lane >> 4;                     // 0: x/y hops from the window, 1: z/t hops from the stage ring
        const int sl = (warp & 3) * 16 + (lane & 15);  // site in tile
        const int j0 = (warp >> 2) * T;                // first rhs of this thread inside the CTA's slice
        const int jg = (int)rank * NC + j0;
        const int io = set ? T / 2 : 0;                // first rhs (inside the thread's T) this lane stores
        // this lane's link column base inside a hop stage, and (set 1) its z/t operand
        const uint32_t lkoff = (uint32_t)set * LSTAGE + (uint32_t)sl * (uint32_t)sizeof(Cx);
        const uint32_t ztoff = 2 * LSTAGE + (uint32_t)(sl >> 5) * WCHUNK + (uint32_t)(j0 * 3 * WIN_CHUNK + (sl & 31)) * (uint32_t)sizeof(Cx);
        const uint32_t woff = (uint32_t)(j0 * 3 * WIN_CHUNK) * (uint32_t)sizeof(Cx);
        Cx uA[3], uB[3], uC[3], vA[T], vB[T], vC[T];
        // operand addresses are 32-bit shared-space integers: one base register per hop, immediate offsets per load
        auto load_u = [&](Cx(&u)[3], uint32_t lk, int b) {
#pragma unroll
            for (int aa = 0; aa < 3; aa++) u[aa] = lds_at<Cx>(lk, (uint32_t)((3 * aa + b) * 64) * (uint32_t)sizeof(Cx));
        };
        auto load_v = [&](Cx(&v)[T], uint32_t vp, int b) {
#pragma unroll
            for (int i = 0; i < T; i++) v[i] = lds_at<Cx>(vp, (uint32_t)(i * 3 + b) * PLANE);
        };
        const uint32_t stg_s = smem_addr(stg), win_s = smem_addr(win);
        int hslot = 0; // hop-stage ring position
        uint32_t hph = 0;
        // A slot goes back to its producer as soon as its operands are in registers, up to two columns before they are used
        // -- so the arrival must not overtake those loads.  It does if nothing stops it: mbarrier.arrive is not queued
        // behind earlier shared-memory loads of the warp, and when the load queue is congested (the xpay loads at the start of
        // a tile) a refill -- ~700 cycles away on the idle 16^4 lattice -- landed before loads issued ahead of the arrive had
        // executed: 2e-4 of the xpay launches there read one 32-byte sector of an operand of hop 8 from the chunk of hop 11,
        // the next user of the slot (found by bit-exact reruns, decoded with a plane-indexed input).  The barrier ADDRESS
        // is therefore computed from every register the stage was loaded into (all three columns), ANDed with p.zero = 0,
        // which the compiler cannot know: the arrive cannot issue before the scoreboards of all those loads have cleared.
        // (A dependence on the last column's registers alone moved the failure to the column before; a CTA-scope fence
        // also closes it but waits for the xpay global loads as well.)
        auto dep_of = [&](const Cx(&u)[3], const Cx(&v)[T]) -> uint32_t {
            uint32_t d = lo_bits(u[0].x) | lo_bits(u[1].x) | lo_bits(u[2].x);
#pragma unroll
            for (int i = 0; i < T; i++) d |= lo_bits(v[i].x);
            return d;
        };
        auto release_stage = [&](int s_, uint32_t dep) {
            uint64_t *bb = reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(&hempty[s_]) + dep);
            __syncwarp();
            if (C == 1) {
                if (lane == 0) mbar_arrive(bb);
            } else {
                if (lane < C) mbar_arrive_remote(bb, (uint32_t)lane);
            }
        };
        auto advance = [&]() {
            if (++hslot == D) {
                hslot = 0;
                hph ^= 1u;
            }
        };
        // Window bookkeeping without divisions: ring positions (slot, phase) of the next chunk to wait for, of the next
        // chunk to release and of the first chunk of the current tile advance by conditional subtraction; the position of
        // the site in its x-row (ex, row parity) is divided out once per segment and stepped per tile.
        int wq_slot = 0;     // ring slot of the next chunk to wait for
        uint32_t wq_ph = 0;  // its phase
        int rl_slot = 0;     // ring slot of the next chunk to release
        const int dex = 64 % Xh, drow = 64 / Xh; // a tile further: ex += dex (mod Xh), row += drow (+ carry)
        for (int si = cid; si < p.nseg; si += ncl) {
            const int4 sg = p.segs[si];
            const int seg_lo = 2 * sg.x - HcL, seg_hi = 2 * sg.y - 1 + HcL; // virtual chunks of this segment
            const int zpar = ((sg.z * 64 / XhY) % g.X[2] + sg.z * 64 / (XhY * g.X[2]) + p.parity) & 1; // (z + t + parity) of the strip
            int waited = seg_lo, released = seg_lo;
            // slot of the first chunk of tile sg.x: HcL chunks behind the segment's first chunk (= the next to wait for)
            int t_slot = wq_slot + HcL;
            if (t_slot >= WCH) t_slot -= WCH;
            int ex, rowp;
            {
                const int el = sg.x * 64 + sl - sg.z * 64; // site inside the strip
                ex = el % Xh;
                rowp = (el / Xh + zpar) & 1;
            }
            auto release_to = [&](int new_rel, uint32_t dep) { // lane 0: give the chunks [released, new_rel) back to the window producer
                for (; released < new_rel; released++) {
                    mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(&wempty[rl_slot]) + dep));
                    if (++rl_slot == WCH) rl_slot = 0;
                }
            };
            for (int k = sg.x; k < sg.y; k++) {
                const int e = k * 64 + sl;
                // xpay operand of the rhs this lane will store: requested now, used after the 16 hops
                Cx xv[XP ? T / 2 : 1][3];
                if (XP) {
                    const Cx *xsrc = reinterpret_cast<const Cx *>(p.xp) + (size_t)min(jg + io, p.N - 1) * 3 * Vh + e;
#pragma unroll
                    for (int i = 0; i < T / 2; i++)
#pragma unroll
                        for (int cc = 0; cc < 3; cc++) xv[i][cc] = ldg_stream(xsrc + (size_t)((jg + io + i < p.N ? i : 0) * 3 + cc) * Vh);
                }
                const int whi = 2 * k + 1 + HcL;
                while (waited <= whi) {
                    mbar_wait(&wfull[wq_slot], wq_ph);
                    if (++wq_slot == WCH) {
                        wq_slot = 0;
                        wq_ph ^= 1u;
                    }
                    waited++;
                }
                const int slot2k = t_slot;
                const int par = rowp; // x = 2 ex + par
                // vector operand of hop h (h < 8) of this lane's set: window address (set 0) or stage offset (set 1)
                auto win_ptr = [&](int h) -> uint32_t {
                    const int mu = BKR_HOP_MU(h), hop = BKR_HOP_LONG(h) ? 3 : 1, sgn = BKR_HOP_BACK(h) ? -hop : hop;
                    int d;
                    if (mu == 1) {
                        d = sl + sgn * Xh;
                    } else {
                        int cx = ex + ((par + sgn) >> 1); // column of the neighbour, periodic in x
                        if (cx < 0) cx += Xh;
                        if (cx >= Xh) cx -= Xh;
                        d = sl + cx - ex;
                    }
                    int sidx = slot2k + (d >> 5); // arithmetic shift = floor
                    if (sidx < 0) sidx += WCH;
                    if (sidx >= WCH) sidx -= WCH;
                    return win_s + (uint32_t)sidx * WCHUNK + woff + (uint32_t)(d & 31) * (uint32_t)sizeof(Cx);
                };
                Real acc[T][6];
#pragma unroll
                for (int i = 0; i < T; i++)
#pragma unroll
                    for (int qd = 0; qd < 6; qd++) acc[i][qd] = (Real)0;
                mbar_wait(&hfull[hslot], hph);
                uint32_t sb = stg_s + (uint32_t)hslot * HSTAGE;
                uint32_t lk = sb + lkoff, vp = set ? sb + ztoff : win_ptr(0);
                load_u(uA, lk, 0);
                load_v(vA, vp, 0);
                // One hop: on entry register set A holds column 0; the loads of columns 1 and 2 are issued at once (sets B, C),
                // so that by the end of column 0's FMAs every operand of the stage is in registers and the stage can go back
                // to the producers without the arithmetic waiting for anything (release_stage).
                auto hop = [&](auto HC) {
                    constexpr int h = decltype(HC)::value;
                    load_u(uB, lk, 1);
                    load_v(vB, vp, 1);
                    load_u(uC, lk, 2);
                    load_v(vC, vp, 2);
                    col_fma<Real, Cx, T>(acc, uA, vA);
                    const uint32_t dep = (dep_of(uA, vA) | dep_of(uB, vB) | dep_of(uC, vC)) & p.zero;
                    release_stage(hslot, dep);
                    if (h == 1 && p.slim) {
                        // hops 0, 1 are y-3, y-1 (common.cuh): the chunks below the tile are dead from here on and go back
                        // to the window producer, which loads the next tile's upper chunks into them
                        const int new_rel = 2 * k - p.xover; // x neighbours reach 2 sites below a tile that starts mid-row
                        if (lane == 0) release_to(new_rel, dep);
                        else
                            for (; released < new_rel; released++)
                                if (++rl_slot == WCH) rl_slot = 0;
                    }
                    advance();
                    if constexpr (h < 7) {
                        const uint32_t ok = mbar_try(&hfull[hslot], hph);
                        sb = stg_s + (uint32_t)hslot * HSTAGE;
                        vp = set ? sb + ztoff : win_ptr(h + 1);
                        col_fma<Real, Cx, T>(acc, uB, vB);
                        mbar_finish(ok, &hfull[hslot], hph);
                        lk = sb + lkoff;
                        load_u(uA, lk, 0);
                        load_v(vA, vp, 0);
                    } else {
                        col_fma<Real, Cx, T>(acc, uB, vB);
                    }
                    col_fma<Real, Cx, T>(acc, uC, vC);
                    return dep;
                };
                hop(std::integral_constant<int, 0>{});
                hop(std::integral_constant<int, 1>{});
                hop(std::integral_constant<int, 2>{});
                hop(std::integral_constant<int, 3>{});
                hop(std::integral_constant<int, 4>{});
                hop(std::integral_constant<int, 5>{});
                hop(std::integral_constant<int, 6>{});
                const uint32_t dep_last = hop(std::integral_constant<int, 7>{});
                // release the window chunks the next tile of this segment does not need
                {
                    const int new_rel = (k == sg.y - 1) ? seg_hi + 1 : 2 * (k + 1) - HcL;
                    __syncwarp();
                    if (lane == 0) release_to(new_rel, dep_last); // (issued after hop 15's release: every window load has returned)
                    else
                        for (; released < new_rel; released++)
                            if (++rl_slot == WCH) rl_slot = 0;
                }
                // next tile of the segment: two chunks and 64 sites further
                t_slot += 2;
                if (t_slot >= WCH) t_slot -= WCH;
                ex += dex;
                rowp ^= drow & 1;
                if (ex >= Xh) {
                    ex -= Xh;
                    rowp ^= 1;
                }
                // The two halves of the warp hold the x/y and the z/t part of the same (site, rhs) sums: each half sends the
                // other the partial sums of the T / 2 rhs the other will store and adds what it receives to its own.
                Cx *vout = reinterpret_cast<Cx *>(p.out) + (size_t)(jg + io) * 3 * Vh + e;
#pragma unroll
                for (int i = 0; i < T / 2; i++) {
#pragma unroll
                    for (int cc = 0; cc < 3; cc++) {
                        const Real sx = set ? acc[i][2 * cc] : acc[T / 2 + i][2 * cc];
                        const Real sy = set ? acc[i][2 * cc + 1] : acc[T / 2 + i][2 * cc + 1];
                        const Real mx = set ? acc[T / 2 + i][2 * cc] : acc[i][2 * cc];
                        const Real my = set ? acc[T / 2 + i][2 * cc + 1] : acc[i][2 * cc + 1];
                        Cx o;
                        o.x = mx + shfl_x16(sx);
                        o.y = my + shfl_x16(sy);
                        if (XP) {
                            o.x = fma((Real)p.a, xv[i][cc].x, -o.x);
                            o.y = fma((Real)p.a, xv[i][cc].y, -o.y);
                        }
                        if (jg + io + i < p.N) __stcs(vout + (size_t)(i * 3 + cc) * Vh, o);
                    }
                }
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
template <typename Real, int T, int C, bool XP>
static int launch_win_x(bkr_ctx *ctx, int parity, int N, int prec, const void *in, void *out, const void *xp, double a,
                        const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int NC = 2 * T;
    const Geom &g = ctx->g;
    const int Xh = g.X[0] / 2;
    WinParams p;
    memset(&p, 0, sizeof(p));
    p.HcL = (3 * Xh + WIN_CHUNK - 1) / WIN_CHUNK;
    p.slim = ctx->tune[BKR_TUNE_WIN_SLIM] == 2 ? 0 : 1;
    p.xover = (64 % Xh) != 0 ? 1 : 0;
    p.WCH = 2 * p.HcL + 2 + (p.slim ? std::max(0, 2 - (p.HcL - p.xover)) : 2);
    if (p.WCH > 16) return 1;
    const size_t lstage = (size_t)9 * 64 * sizeof(Cx), wchunk = (size_t)NC * 3 * WIN_CHUNK * sizeof(Cx), wbytes = (size_t)p.WCH * wchunk,
                 hstage = 2 * lstage + 2 * wchunk, bbytes = 64 * 8;
    // Ring depth: what decides whether the arithmetic warps wait is how far ahead of its use a stage can be requested
    // (a TMA round trip is 1300-2500 cycles on the loaded chip, a hop ~850 at the target rate; a slot is released a third of
    // the way into the hop that reads it, so a ring of D stages gives D - 1/3 hops of lead).
    int D = ctx->tune[BKR_TUNE_WIN_STAGES] ? ctx->tune[BKR_TUNE_WIN_STAGES] : 4;
    D = std::min(D, 8);
    while (D >= 2 && D * hstage + wbytes + bbytes > WIN_SMEM_MAX) D--;
    if (D < 2) return 1;
    // clusters of 3-4 CTAs need at least 3 stages (the release -> refill round trip crosses SMs)
    if (C >= 3 && D < 3 && ctx->dslash_force != 1) return 1;
    p.D = D;
    p.off_win = (uint32_t)(D * hstage);
    p.off_bar = (uint32_t)(p.off_win + wbytes);
    const size_t smem = p.off_bar + bbytes;

    BKR_TRY(build_segments(ctx, N, prec, ctx->tune[BKR_TUNE_WIN_SEGLEN] > 0 ? ctx->tune[BKR_TUNE_WIN_SEGLEN] : 8));
    CUtensorMap tm_win;
    if (!make_map(&tm_win, in, prec, g.Vh, N, WIN_CHUNK, 3, NC)) return 1;

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
    p.zero = 0;

    auto kern = dslash_win_kernel<Real, T, C, XP>;
    static int max_clusters = -1, attr_dev = -1; // per instantiation; the shared-memory opt-in is per device
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(WIN_THREADS);
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
    cfg.gridDim = dim3((unsigned)(std::min(max_clusters, p.nseg) * C));
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, tm_win, p);
    if (e != cudaSuccess) {
        ctx->last_cuda = (int)e;
        return BKR_ECUDA;
    }
    return bkr_check_launch(ctx);
}

template <typename Real, int T, int C>
static int launch_win_c(bkr_ctx *ctx, int parity, int N, int prec, const void *in, void *out, const void *xp, double a,
                        const int *done)
{
    if (xp) return launch_win_x<Real, T, C, true>(ctx, parity, N, prec, in, out, xp, a, done);
    return launch_win_x<Real, T, C, false>(ctx, parity, N, prec, in, out, xp, a, done);
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
        if (C == 1) return launch_win_c<double, 4, 1>(ctx, out_parity, N, prec, in, out, xp, a, done);
        if (C == 2) return launch_win_c<double, 4, 2>(ctx, out_parity, N, prec, in, out, xp, a, done);
        if (C == 3) return launch_win_c<double, 4, 3>(ctx, out_parity, N, prec, in, out, xp, a, done);
        if (C == 4) return launch_win_c<double, 4, 4>(ctx, out_parity, N, prec, in, out, xp, a, done);
        return 1;
    }
    const int C = (N + 15) / 16;
    if (mode == 1 && (N < 13 || 16 * C - N > 3)) return 1;
    if (C == 1) return launch_win_c<float, 8, 1>(ctx, out_parity, N, prec, in, out, xp, a, done);
    if (C == 2) return launch_win_c<float, 8, 2>(ctx, out_parity, N, prec, in, out, xp, a, done);
    return 1;
}
