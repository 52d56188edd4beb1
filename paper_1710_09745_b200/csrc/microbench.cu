// Register-only / on-chip microbenchmarks that give the rooflines of DESIGN.md section 6.4 their measured denominators
// ("the build must measure the FP64 and FP32 FMA peaks on the box").  Not on the hot path:
// bench.py --microbench calls bkr_microbench() and reports the numbers next to the kernel fractions.
//
//   kind 0  DFMA   fp64 FMA, 16 independent chains per thread            -> flop / launch
//   kind 1  FFMA   fp32 FMA, 16 independent chains per thread            -> flop / launch
//   kind 2  DMMA   mma.sync.m8n8k4.f64, 8 independent accumulators/warp  -> flop / launch
//   kind 3  L2 -> SM read bandwidth, 16-byte ld.global.nc over a 48 MB (L2 resident) buffer -> bytes / launch
//   kind 4  L2 -> SM read bandwidth, 1-D TMA bulk copies (8 KB) into a shared-memory ring   -> bytes / launch
//   kind 5  shared-memory read bandwidth, conflict-free ld.shared.v2.f64                     -> bytes / launch
//   kind 6-9  the stencil's register-only column update (rhs-major / link-major FMA order; 8 / 32 warps per SM) -> flop / launch
#include "common.cuh"
#include "tma.cuh"

#define MB_THREADS 256
#define MB_CTAS_PER_SM 4

template <typename Real> __global__ void __launch_bounds__(MB_THREADS) mb_fma_kernel(Real *out, int iters, Real seed)
{
    Real acc[16];
#pragma unroll
    for (int i = 0; i < 16; i++) acc[i] = seed * (Real)(i + 1 + threadIdx.x);
    const Real a = (Real)1.0000001, b = (Real)1e-9;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 16; i++) acc[i] = fma(acc[i], a, b);
    }
    Real s = 0;
#pragma unroll
    for (int i = 0; i < 16; i++) s += acc[i];
    if (s == (Real)-1.2345) out[0] = s; // never true: keeps the chains alive
}

__global__ void __launch_bounds__(MB_THREADS) mb_dmma_kernel(double *out, int iters, double seed)
{
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) c[i][0] = c[i][1] = seed * (i + 1);
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                         : "+d"(c[i][0]), "+d"(c[i][1])
                         : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == -1.2345) out[0] = s;
}

// the stencil's column update (3 x T complex FMAs from registers only): what the DFMA pipe sustains on that operand pattern
template <int ORDER> __global__ void __launch_bounds__(MB_THREADS) mb_colfma_kernel(double *out, int iters, double seed)
{
    constexpr int T = 4;
    double2 uA[3], uB[3], vA[T], vB[T];
    double acc[T][6];
    for (int a = 0; a < 3; a++) {
        uA[a] = make_double2(seed * (a + 1 + threadIdx.x), seed * (a + 2));
        uB[a] = make_double2(seed * (a + 3), seed * (a + 4 + threadIdx.x));
    }
    for (int i = 0; i < T; i++) {
        vA[i] = make_double2(seed * (i + 5 + threadIdx.x), seed * (i + 6));
        vB[i] = make_double2(seed * (i + 7), seed * (i + 8 + threadIdx.x));
        for (int q = 0; q < 6; q++) acc[i][q] = 0.0;
    }
    auto col = [&](const double2(&u)[3], const double2(&v)[T]) {
        if (ORDER == 0) {
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
        } else {
            // link element outermost: 2 T consecutive FMAs share their first operand
#pragma unroll
            for (int a = 0; a < 3; a++) {
#pragma unroll
                for (int i = 0; i < T; i++) {
                    acc[i][2 * a] = fma(u[a].x, v[i].x, acc[i][2 * a]);
                    acc[i][2 * a + 1] = fma(u[a].x, v[i].y, acc[i][2 * a + 1]);
                }
#pragma unroll
                for (int i = 0; i < T; i++) {
                    acc[i][2 * a] = fma(-u[a].y, v[i].y, acc[i][2 * a]);
                    acc[i][2 * a + 1] = fma(u[a].y, v[i].x, acc[i][2 * a + 1]);
                }
            }
        }
    };
    for (int it = 0; it < iters; it++) {
        col(uA, vA);
        col(uB, vB);
    }
    double s = 0;
    for (int i = 0; i < T; i++)
        for (int q = 0; q < 6; q++) s += acc[i][q];
    if (s == -1.2345) out[0] = s;
}

// every CTA streams over the whole buffer (staggered start), 4 independent 16-byte loads per thread per step
__global__ void __launch_bounds__(MB_THREADS) mb_l2_ldg_kernel(const double2 *buf, size_t n16, int passes, double *out)
{
    double s = 0;
    const size_t per = (size_t)MB_THREADS * 4;
    const size_t nstep = n16 / per;
    size_t step = ((size_t)blockIdx.x * 977) % nstep;
    const size_t total = (size_t)passes * nstep / gridDim.x; // each CTA reads 1/gridDim of passes x buffer
    for (size_t k = 0; k < total; k++) {
        const double2 *p = buf + step * per + threadIdx.x;
        double2 v[4];
#pragma unroll
        for (int i = 0; i < 4; i++)
            asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v[i].x), "=d"(v[i].y) : "l"(p + i * MB_THREADS));
#pragma unroll
        for (int i = 0; i < 4; i++) s += v[i].x + v[i].y;
        if (++step == nstep) step = 0;
    }
    if (s == -1.2345) out[0] = s;
}

#define MB_TMA_STAGE 8192
#define MB_TMA_RING 8
__global__ void __launch_bounds__(64) mb_l2_tma_kernel(const unsigned char *buf, size_t nbytes, int passes, double *out)
{
    extern __shared__ __align__(128) unsigned char sm[];
    uint64_t *full = reinterpret_cast<uint64_t *>(sm + MB_TMA_RING * MB_TMA_STAGE);
    uint64_t *empty = full + MB_TMA_RING;
    if (threadIdx.x == 0) {
        for (int s = 0; s < MB_TMA_RING; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const size_t nstage = nbytes / MB_TMA_STAGE;
    const size_t total = (size_t)passes * nstage / gridDim.x;
    size_t st = ((size_t)blockIdx.x * 977) % nstage;
    if (threadIdx.x == 0) {
        for (size_t k = 0; k < total; k++) {
            const int slot = (int)(k % MB_TMA_RING);
            const uint32_t use = (uint32_t)(k / MB_TMA_RING);
            if (use > 0) mbar_wait(&empty[slot], (use - 1) & 1);
            mbar_expect_tx(&full[slot], MB_TMA_STAGE);
            tma_load_1d(sm + (size_t)slot * MB_TMA_STAGE, buf + st * MB_TMA_STAGE, MB_TMA_STAGE, &full[slot]);
            if (++st == nstage) st = 0;
        }
    } else if (threadIdx.x == 32) {
        for (size_t k = 0; k < total; k++) {
            const int slot = (int)(k % MB_TMA_RING);
            mbar_wait(&full[slot], (uint32_t)(k / MB_TMA_RING) & 1);
            mbar_arrive(&empty[slot]);
        }
        if (total == (size_t)-1) out[0] = 0;
    }
}

__global__ void __launch_bounds__(MB_THREADS) mb_smem_kernel(double *out, int iters)
{
    __shared__ double2 sm[MB_THREADS * 4];
    for (int i = threadIdx.x; i < MB_THREADS * 4; i += MB_THREADS) sm[i] = make_double2(i, 1);
    __syncthreads();
    double s = 0;
    for (int it = 0; it < iters; it++) {
        double2 v[4];
#pragma unroll
        for (int i = 0; i < 4; i++) v[i] = lds_cx(&sm[((threadIdx.x + it) & (MB_THREADS - 1)) + i * MB_THREADS]);
#pragma unroll
        for (int i = 0; i < 4; i++) s += v[i].x + v[i].y;
    }
    if (s == -1.2345) out[0] = s;
}

int run_microbench(bkr_ctx *ctx, int kind, int reps, double *result)
{
    if (kind >= 10) return run_probe(ctx, kind, result);
    if (kind < 0 || kind > 9 || reps < 1 || !result) return BKR_EINVAL;
    const size_t BUF = (size_t)48 << 20;
    void *buf = nullptr;
    BKR_CUDA(ctx, cudaMalloc(&buf, BUF));
    cudaMemsetAsync(buf, 0, BUF, ctx->stream);
    double *out = (double *)buf;
    const int grid = BKR_NUM_SMS * MB_CTAS_PER_SM;
    const int iters = 4096, passes = 64;
    double units = 0;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    if (kind == 4) cudaFuncSetAttribute(mb_l2_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, MB_TMA_RING * MB_TMA_STAGE + 256);
    for (int r = -2; r < reps; r++) { // two warm-up launches
        if (r == 0) cudaEventRecord(e0, ctx->stream);
        switch (kind) {
        case 0:
            mb_fma_kernel<double><<<grid, MB_THREADS, 0, ctx->stream>>>(out, iters, 1e-3);
            units = 2.0 * 16 * iters * (double)grid * MB_THREADS;
            break;
        case 1:
            mb_fma_kernel<float><<<grid, MB_THREADS, 0, ctx->stream>>>((float *)out, iters, 1e-3f);
            units = 2.0 * 16 * iters * (double)grid * MB_THREADS;
            break;
        case 2:
            mb_dmma_kernel<<<grid, MB_THREADS, 0, ctx->stream>>>(out, iters, 1e-3);
            units = 2.0 * 8 * 8 * 4 * 8 * iters * (double)grid * (MB_THREADS / 32);
            break;
        case 3:
            mb_l2_ldg_kernel<<<grid, MB_THREADS, 0, ctx->stream>>>((const double2 *)buf, BUF / 16, passes, out);
            units = (double)((size_t)passes * (BUF / 16 / (MB_THREADS * 4)) / grid) * grid * MB_THREADS * 4 * 16;
            break;
        case 4:
            mb_l2_tma_kernel<<<grid, 64, MB_TMA_RING * MB_TMA_STAGE + 256, ctx->stream>>>((const unsigned char *)buf, BUF, passes, out);
            units = (double)((size_t)passes * (BUF / MB_TMA_STAGE) / grid) * grid * MB_TMA_STAGE;
            break;
        case 5:
            mb_smem_kernel<<<grid, MB_THREADS, 0, ctx->stream>>>(out, iters);
            units = 4.0 * 16 * iters * (double)grid * MB_THREADS;
            break;
        case 6: // the stencil's FMA pattern, 8 warps per SM (its occupancy)
            mb_colfma_kernel<0><<<BKR_NUM_SMS, MB_THREADS, 0, ctx->stream>>>(out, iters, 1e-3);
            units = 2.0 * 96 * iters * (double)BKR_NUM_SMS * MB_THREADS;
            break;
        case 7:
            mb_colfma_kernel<1><<<BKR_NUM_SMS, MB_THREADS, 0, ctx->stream>>>(out, iters, 1e-3);
            units = 2.0 * 96 * iters * (double)BKR_NUM_SMS * MB_THREADS;
            break;
        case 8: // same, 32 warps per SM
            mb_colfma_kernel<0><<<grid, MB_THREADS, 0, ctx->stream>>>(out, iters, 1e-3);
            units = 2.0 * 96 * iters * (double)grid * MB_THREADS;
            break;
        case 9:
            mb_colfma_kernel<1><<<grid, MB_THREADS, 0, ctx->stream>>>(out, iters, 1e-3);
            units = 2.0 * 96 * iters * (double)grid * MB_THREADS;
            break;
        }
    }
    cudaEventRecord(e1, ctx->stream);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) {
        ctx->last_cuda = (int)e;
        return BKR_ECUDA;
    }
    result[0] = ms / reps;
    result[1] = units;
    result[2] = 0.0;
    return BKR_OK;
}
