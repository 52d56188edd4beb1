// On-chip probes behind the design of the window stencil (profiles/r2_onchip_probes.md): what a DFMA costs besides the
// FP64 pipe, how shared-memory loads, TMA fills and global loads share the SM's data paths, what a shared-memory fed
// stencil loop can reach, and what a TMA bulk copy costs its issuing lane.  Not on the hot path: bkr_microbench(kind >= 10)
// runs them, `python bench.py --microbench` prints them.  One CTA per SM; CTA 0 times itself with clock64.
//
//   result[0] = SM cycles of the measured region, result[1] = work units per SM, result[2] = second work count (or 0)
//
//   10  LDS.128 conflict-free, 8 warps                      units = bytes delivered to registers
//   11  LDS.128, 8 distinct addresses per warp (broadcast)   units = bytes delivered to registers
//   12  LDS.128 stream + one lane of TMA bulk fills          units = LDS bytes, [2] = TMA bytes
//   13  LDS.128 stream + 4 warps of LDG.128 (L2 resident)    units = LDS bytes, [2] = LDG bytes
//   14  DFMA, one operand reused over 16 (2 register reads)  units = lane DFMAs          15  3 fresh operands
//   16  DFMA (2 reads) + 4 LDS.128 per 64 DFMA               17  + 8 LDS.128 per 64 DFMA
//   18  dry stencil loop T = 4, 8 warps    19  T = 8, 4 warps    20  T = 8, 8 warps     units = lane DFMAs
//   21  TMA 9 KB bulk copies from one lane, ring of 8, L2 resident: units = copies (cycles / copies = issue interval)
//   22  the same, ring of 1: cycles / copies = round trip
#include "common.cuh"
#include "tma.cuh"

namespace {

struct ProbeOut {
    unsigned long long cycles, aux;
};

// ---------------------------------------------------------------- LDS / TMA / LDG sharing
#define PR_STAGE 8192
#define PR_RING 8
// PAT 0: conflict-free, 1: 8 addresses per warp.  PROD 0: none, 1: one TMA lane (warp 15), 2: LDG warps 12-15
template <int PAT, int PROD>
__global__ void __launch_bounds__(512, 1) probe_mix_kernel(const unsigned char *buf, size_t nbytes, int iters, double *sink, ProbeOut *out)
{
    extern __shared__ __align__(1024) unsigned char sm[];
    double2 *data = reinterpret_cast<double2 *>(sm);
    unsigned char *ring = sm + 65536;
    uint64_t *full = reinterpret_cast<uint64_t *>(sm + 131072);
    __shared__ int stop;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) data[i] = make_double2(i, 1);
    if (threadIdx.x == 0) {
        stop = 0;
        for (int s = 0; s < PR_RING; s++) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const unsigned long long c0 = clock64();
    if (warp < 8) {
        double s = 0;
        const int l = PAT == 0 ? lane : (lane & 7);
        for (int it = 0; it < iters; it++) {
            double2 v[8];
#pragma unroll
            for (int i = 0; i < 8; i++) v[i] = lds_cx(&data[((l + it * 32) & 255) + i * 256]);
#pragma unroll
            for (int i = 0; i < 8; i++) s += v[i].x + v[i].y;
        }
        if (s == -1.2345) sink[0] = s;
        __syncwarp();
        if (warp == 0 && lane == 0) *(volatile int *)&stop = 1;
    } else if (PROD == 1 && warp == 15) {
        if (lane == 0) {
            const size_t nstage = nbytes / PR_STAGE;
            size_t st = ((size_t)blockIdx.x * 977) % nstage;
            unsigned long long k = 0;
            for (;; k++) {
                if (*(volatile int *)&stop) break;
                const int slot = (int)(k % PR_RING);
                if (k >= PR_RING) mbar_wait(&full[slot], (uint32_t)((k / PR_RING) - 1) & 1);
                mbar_expect_tx(&full[slot], PR_STAGE);
                tma_load_1d(ring + (size_t)slot * PR_STAGE, buf + st * PR_STAGE, PR_STAGE, &full[slot]);
                if (++st == nstage) st = 0;
            }
            for (unsigned long long j = (k > PR_RING ? k - PR_RING : 0); j < k; j++) mbar_wait(&full[j % PR_RING], (uint32_t)(j / PR_RING) & 1);
            if (blockIdx.x == 0) out->aux = k * PR_STAGE;
        }
    } else if (PROD == 2 && warp >= 12) {
        const double2 *p = reinterpret_cast<const double2 *>(buf);
        const size_t per = 128 * 8, nstep = nbytes / 16 / per;
        size_t step = ((size_t)blockIdx.x * 977) % nstep;
        const int t = threadIdx.x - 12 * 32;
        double s = 0;
        unsigned long long k = 0;
        for (;; k++) {
            if (*(volatile int *)&stop) break;
            double2 v[8];
#pragma unroll
            for (int i = 0; i < 8; i++)
                asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v[i].x), "=d"(v[i].y) : "l"(p + step * per + i * 128 + t));
#pragma unroll
            for (int i = 0; i < 8; i++) s += v[i].x + v[i].y;
            if (++step == nstep) step = 0;
        }
        if (s == -1.2345) sink[0] = s;
        if (t == 0 && blockIdx.x == 0) out->aux = k * per * 16;
    }
    __syncthreads();
    if (threadIdx.x == 0 && blockIdx.x == 0) out->cycles = clock64() - c0;
}

// ---------------------------------------------------------------- DFMA operand patterns, with LDS.128 in between
// PAT 1: acc[i] = fma(a, v[i], acc[i]), a fixed over 16 DFMAs (2 fresh register operands); 2: three fresh operands
template <int PAT, int NLDS>
__global__ void __launch_bounds__(256, 1) probe_fma_kernel(int iters, double seed, double *sink, ProbeOut *out)
{
    __shared__ double2 sm[2048];
    for (int i = threadIdx.x; i < 2048; i += blockDim.x) sm[i] = make_double2(i, 1);
    __syncthreads();
    double acc[16], u[16], v[16];
#pragma unroll
    for (int i = 0; i < 16; i++) {
        acc[i] = seed * (i + 1 + threadIdx.x);
        u[i] = 1.0 + seed * (i + 2) * 1e-6;
        v[i] = seed * (i + 3 + threadIdx.x) * 1e-9;
    }
    const unsigned long long c0 = clock64();
    double s = 0;
    for (int it = 0; it < iters; it++) {
        double2 l[NLDS > 0 ? NLDS : 1];
#pragma unroll
        for (int i = 0; i < NLDS; i++) l[i] = lds_cx(&sm[((threadIdx.x + it * 32) & 1023) + i * 64]);
#pragma unroll
        for (int rep = 0; rep < 4; rep++)
#pragma unroll
            for (int i = 0; i < 16; i++) {
                if (PAT == 1) acc[i] = fma(u[rep], v[i], acc[i]);
                else acc[i] = fma(u[(i + rep) & 15], v[i], acc[i]);
            }
#pragma unroll
        for (int i = 0; i < NLDS; i++) s += l[i].x + l[i].y;
    }
#pragma unroll
    for (int i = 0; i < 16; i++) s += acc[i];
    if (s == -1.2345) sink[0] = s;
    __syncthreads();
    if (threadIdx.x == 0 && blockIdx.x == 0) out->cycles = clock64() - c0;
}

// ---------------------------------------------------------------- dry stencil loop
// The arithmetic warps' loop of dslash_win.cu with operands in static shared memory: thread = site (tid % 64) x T rhs,
// columns of 3 link elements + T vector elements loaded one column ahead of their 12 T FMAs, no barriers, no producers.
template <int T> __device__ __forceinline__ void probe_col_fma(double (&acc)[T][6], const double2 (&u)[3], const double2 (&v)[T])
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

template <int T, int W>
__global__ void __launch_bounds__(W * 32, 1) probe_dry_kernel(int hops, double *sink, ProbeOut *out)
{
    extern __shared__ __align__(1024) unsigned char sm[];
    double2 *lnk = reinterpret_cast<double2 *>(sm);            // 8 stages x 9 x 64
    double2 *vec = reinterpret_cast<double2 *>(sm + 8 * 9216); // 96 KB
    for (int i = threadIdx.x; i < 8 * 576 + 6144; i += blockDim.x) lnk[i] = make_double2(1e-3 * (i & 255), 1e-3);
    __syncthreads();
    const int sl = threadIdx.x & 63, grp = threadIdx.x >> 6;
    double acc[T][6];
#pragma unroll
    for (int i = 0; i < T; i++)
#pragma unroll
        for (int q = 0; q < 6; q++) acc[i][q] = 0;
    auto load_u = [&](double2(&u)[3], const double2 *lk, int b) {
#pragma unroll
        for (int a = 0; a < 3; a++) u[a] = lds_cx(lk + (3 * a + b) * 64);
    };
    auto load_v = [&](double2(&v)[T], const double2 *vp, int b) {
#pragma unroll
        for (int i = 0; i < T; i++) v[i] = lds_cx(vp + (i * 3 + b) * 64);
    };
    auto vptr = [&](int h) { return vec + (((grp * T * 3 * 64) + (h & 3) * 64) & 4095) + sl; };
    const unsigned long long c0 = clock64();
    double2 uA[3], uB[3], vA[T], vB[T];
    load_u(uA, lnk + sl, 0);
    load_v(vA, vptr(0), 0);
    for (int h = 0; h < hops; h += 2) {
        const double2 *lk0 = lnk + (h & 7) * 576 + sl, *lk1 = lnk + ((h + 1) & 7) * 576 + sl, *lk2 = lnk + ((h + 2) & 7) * 576 + sl;
        const double2 *vp0 = vptr(h), *vp1 = vptr(h + 1), *vp2 = vptr(h + 2);
        load_u(uB, lk0, 1); load_v(vB, vp0, 1);
        probe_col_fma<T>(acc, uA, vA);
        load_u(uA, lk0, 2); load_v(vA, vp0, 2);
        probe_col_fma<T>(acc, uB, vB);
        load_u(uB, lk1, 0); load_v(vB, vp1, 0);
        probe_col_fma<T>(acc, uA, vA);
        load_u(uA, lk1, 1); load_v(vA, vp1, 1);
        probe_col_fma<T>(acc, uB, vB);
        load_u(uB, lk1, 2); load_v(vB, vp1, 2);
        probe_col_fma<T>(acc, uA, vA);
        load_u(uA, lk2, 0); load_v(vA, vp2, 0);
        probe_col_fma<T>(acc, uB, vB);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < T; i++)
#pragma unroll
        for (int q = 0; q < 6; q++) s += acc[i][q];
    if (s == -1.2345) sink[0] = s;
    __syncthreads();
    if (threadIdx.x == 0 && blockIdx.x == 0) out->cycles = clock64() - c0;
}

// ---------------------------------------------------------------- TMA bulk copies from one lane
__global__ void __launch_bounds__(64, 1) probe_tma_kernel(const unsigned char *buf, size_t nbytes, int stage, int depth, int iters, ProbeOut *out)
{
    extern __shared__ __align__(1024) unsigned char sm[];
    __shared__ uint64_t full[16];
    if (threadIdx.x == 0) {
        for (int s = 0; s < 16; s++) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const unsigned long long c0 = clock64();
    if (threadIdx.x == 0) {
        const size_t nstage = nbytes / stage;
        size_t st = ((size_t)blockIdx.x * 7919) % nstage;
        for (int k = 0; k < iters; k++) {
            const int slot = k % depth;
            if (k >= depth) mbar_wait(&full[slot], (uint32_t)((k / depth) - 1) & 1);
            mbar_expect_tx(&full[slot], stage);
            tma_load_1d(sm + (size_t)slot * stage, buf + st * stage, stage, &full[slot]);
            st += 131;
            if (st >= nstage) st -= nstage;
        }
        for (int j = (iters > depth ? iters - depth : 0); j < iters; j++) mbar_wait(&full[j % depth], (uint32_t)(j / depth) & 1);
    }
    __syncthreads();
    if (threadIdx.x == 0 && blockIdx.x == 0) out->cycles = clock64() - c0;
}

// kind 23: mma.sync.m16n8k8 TF32 issue rate (legacy tensor path, the one mblas_tf32.cu uses), 8 warps x 8 independent accumulators
__global__ void __launch_bounds__(256, 1) probe_tf32_kernel(int iters, uint32_t seed, double *sink, ProbeOut *out)
{
    float c[8][4];
    uint32_t a[4], b[2];
#pragma unroll
    for (int i = 0; i < 8; i++)
#pragma unroll
        for (int q = 0; q < 4; q++) c[i][q] = 0.f;
#pragma unroll
    for (int q = 0; q < 4; q++) a[q] = seed * (q + 1 + threadIdx.x);
    b[0] = seed;
    b[1] = seed + 1;
    unsigned long long c0 = 0;
    if (threadIdx.x == 0) c0 = clock64();
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++)
            asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                         : "+f"(c[i][0]), "+f"(c[i][1]), "+f"(c[i][2]), "+f"(c[i][3])
                         : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++)
#pragma unroll
        for (int q = 0; q < 4; q++) s += c[i][q];
    if (s == -1.2345f) sink[0] = s;
    __syncthreads();
    if (threadIdx.x == 0 && blockIdx.x == 0) out->cycles = clock64() - c0;
}

// kinds 24..29: dependent-chain latencies of one warp (what bounds the small-matrix kernel, small.cu): cycles per operation of a
// chain of 512 dependent operations, in a 1024-thread CTA whose other warps have exited (24..28) or all take part (29).
//   24 DFMA   25 1.0 / x (+ add)   26 rsqrt (+ add)   27 64-bit shuffle (+ add)   28 shared-memory store -> load round trip
//   29 __syncthreads over 1024 threads
__global__ void __launch_bounds__(1024, 1) probe_latency_kernel(int kind, double seed, double *sink, ProbeOut *out)
{
    __shared__ double sm[1024];
    sm[threadIdx.x] = seed;
    __syncthreads();
    if (kind != 29 && threadIdx.x >= 32) return;
    const int n = 512;
    double x = seed + threadIdx.x;
    const unsigned long long c0 = clock64();
    if (kind == 24) for (int i = 0; i < n; i++) x = fma(x, 1.0000001, 1e-9);
    if (kind == 25) for (int i = 0; i < n; i++) x = 1.0 / x + 1.5;
    if (kind == 26) for (int i = 0; i < n; i++) x = rsqrt(x) + 1.5;
    if (kind == 27) for (int i = 0; i < n; i++) x = __shfl_sync(0xffffffffu, x, (i + 1) & 31) + 1e-9;
    if (kind == 28) for (int i = 0; i < n; i++) {
        volatile double *q = &sm[(threadIdx.x + 32 * (i & 15)) & 1023];
        *q = x;
        x = *q + 1e-9;
    }
    if (kind == 29) for (int i = 0; i < n; i++) {
        __syncthreads();
        x += 1e-9;
    }
    const unsigned long long c1 = clock64();
    if (x == -1.2345) sink[0] = x;
    if (threadIdx.x == 0 && blockIdx.x == 0) out->cycles = c1 - c0;
}

} // namespace

int run_probe(bkr_ctx *ctx, int kind, double *result)
{
    if (kind < 10 || kind > 29 || !result) return BKR_EINVAL;
    const size_t BUF = (size_t)32 << 20; // L2 resident
    unsigned char *buf = nullptr;
    BKR_CUDA(ctx, cudaMalloc((void **)&buf, BUF + 4096));
    BKR_CUDA(ctx, cudaMemsetAsync(buf, 0, BUF + 4096, ctx->stream));
    double *sink = reinterpret_cast<double *>(buf + BUF);
    ProbeOut *out = reinterpret_cast<ProbeOut *>(buf + BUF + 64);
    const int G = BKR_NUM_SMS;
    double units = 0, aux_valid = 0;
    for (int r = 0; r < 2; r++) { // the second launch is the measured one (the first warms L2 and the instruction cache)
        switch (kind) {
        case 10: case 11: case 12: case 13: {
            const int iters = 20000, smem = 131072 + 256;
            auto go = [&](auto kern) {
                cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
                kern<<<G, 512, smem, ctx->stream>>>(buf, BUF, iters, sink, out);
            };
            if (kind == 10) go(probe_mix_kernel<0, 0>);
            if (kind == 11) go(probe_mix_kernel<1, 0>);
            if (kind == 12) go(probe_mix_kernel<0, 1>);
            if (kind == 13) go(probe_mix_kernel<0, 2>);
            units = 8.0 * iters * 8 * 512;
            aux_valid = kind >= 12;
            break;
        }
        case 14: probe_fma_kernel<1, 0><<<G, 256, 0, ctx->stream>>>(20000, 1e-3, sink, out); units = 20000.0 * 64 * 256; break;
        case 15: probe_fma_kernel<2, 0><<<G, 256, 0, ctx->stream>>>(20000, 1e-3, sink, out); units = 20000.0 * 64 * 256; break;
        case 16: probe_fma_kernel<1, 4><<<G, 256, 0, ctx->stream>>>(20000, 1e-3, sink, out); units = 20000.0 * 64 * 256; break;
        case 17: probe_fma_kernel<1, 8><<<G, 256, 0, ctx->stream>>>(20000, 1e-3, sink, out); units = 20000.0 * 64 * 256; break;
        case 18: case 19: case 20: {
            const int hops = 3200, smem = 8 * 9216 + 98304;
            auto go = [&](auto kern, int threads, int T) {
                cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
                kern<<<G, threads, smem, ctx->stream>>>(hops, sink, out);
                units = (double)hops * 36 * T * threads;
            };
            if (kind == 18) go(probe_dry_kernel<4, 8>, 256, 4);
            if (kind == 19) go(probe_dry_kernel<8, 4>, 128, 8);
            if (kind == 20) go(probe_dry_kernel<8, 8>, 256, 8);
            break;
        }
        case 24: case 25: case 26: case 27: case 28: case 29:
            probe_latency_kernel<<<1, 1024, 0, ctx->stream>>>(kind, 1.5, sink, out);
            units = 512;
            break;
        case 23: probe_tf32_kernel<<<G, 256, 0, ctx->stream>>>(20000, 0u, sink, out); units = 20000.0 * 8 * 8 * 2048; break; // flop per SM
        default: {
            const int stage = 9216, depth = kind == 21 ? 8 : 1, iters = 400, smem = stage * depth;
            cudaFuncSetAttribute(probe_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 9216 * 8);
            probe_tma_kernel<<<G, 64, smem, ctx->stream>>>(buf, BUF, stage, depth, iters, out);
            units = iters;
        }
        }
    }
    ProbeOut h;
    cudaError_t e = cudaMemcpyAsync(&h, out, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(buf);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) {
        ctx->last_cuda = (int)e;
        return BKR_ECUDA;
    }
    result[0] = (double)h.cycles;
    result[1] = units;
    result[2] = aux_valid ? (double)h.aux : 0.0;
    return BKR_OK;
}
