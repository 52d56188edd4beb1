// Multi-BLAS for fp32 blocks on the TF32 tensor path (PAPER.md:245-299 for the operations).
//
// mblas.cu widens fp32 operands and contracts them with FP64 DMMA, whose 37 TFLOP/s bind at N >= 16 when the data are
// only 8 bytes per complex number.  Here every real product is split as (the "3xTF32" error-corrected scheme)
//     x = x_hi + x_lo,   x_hi = x rounded to TF32 (11 significant bits),   x_lo = x - x_hi truncated to TF32 by the tensor core,
//     x y ~= x_lo y_hi + x_hi y_lo + x_hi y_hi                              (x_lo y_lo ~ 2^-22 |x y| dropped)
// and issued as three mma.sync.m16n8k8 TF32 instructions with fp32 accumulators (measured 280 TFLOP/s = 93 TFLOP/s of
// split products: bkr_microbench kind 23, profiles/r2_onchip_probes.md section 6).  NOT the default: its ~3e-7 errors
// cost the fp32-inner solver 25-30 % more iterations at config 3, tol 1e-10 (mblas.cuh);
// BKR_TUNE_F32_MATH selects it.
// Partial sums stay in fp32 only over short runs: an update has <= 64 terms per output and rounds to fp32 anyway; a
// reduction adds its fp32 accumulators into fp64 ones every TF_FLUSH k-steps (64 rows), so the long sum over the lattice
// is fp64 as in mblas.cu.  Error against the fp64 product of the same fp32 inputs: <= ~1e-6 relative to the largest entry
// (tests/test_gpu_tf32.py), against 6e-8 of input rounding.  The rings, the TMA producer warp, the chunk strides, the
// fixed-order two-stage reduction and the partials layout are those of mblas.cu, so launch_gram_finish / small_kernel
// take the result unchanged.
//
// Fragments of mma.m16n8k8 (g = lane / 4, t = lane % 4):
//   A (16 x 8):  a0 = A[g][t]   a1 = A[g + 8][t]   a2 = A[g][t + 4]   a3 = A[g + 8][t + 4]
//   B (8 x 8):   b0 = B[t][g]   b1 = B[t + 4][g]
//   C (16 x 8):  c0 = C[g][2t]  c1 = C[g][2t + 1]  c2 = C[g + 8][2t]  c3 = C[g + 8][2t + 1]
// A complex product is four real ones; the minus sign of Re (x y) = xr yr - xi yi goes into the A operand (sign bit).
#include "mblas.cuh"

static const int TF_CW = 8;    // consumer warps
static const int TF_FLUSH = 8; // k-steps (8 rows each) between fp32 -> fp64 flushes of a reduction

__device__ __forceinline__ void hmma_tf32(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// x -> (hi, lo): hi = x rounded to nearest TF32 (ties away from zero), lo = x - hi (exact, |lo| <= 2^-12 |x|).  The tensor
// core ignores the 13 low bits of an operand, i.e. truncates lo to TF32: an error <= 2^-22 |x|, the size of the dropped
// lo x lo term.  Three integer / fp32 instructions per value (cvt.rna.tf32 compiles to four and handles NaN / Inf).
__device__ __forceinline__ void split_tf32(float x, uint32_t &hi, uint32_t &lo)
{
    const uint32_t h = (__float_as_uint(x) + 0x1000u) & 0xffffe000u;
    hi = h;
    lo = __float_as_uint(x - __uint_as_float(h));
}

struct FragA { // a 16 x 8 operand, split
    uint32_t hi[4], lo[4];
};
struct FragB { // an 8 x 8 operand, split
    uint32_t hi[2], lo[2];
};

__device__ __forceinline__ void split_a(const float (&x)[4], FragA &f)
{
#pragma unroll
    for (int e = 0; e < 4; e++) split_tf32(x[e], f.hi[e], f.lo[e]);
}
__device__ __forceinline__ FragA neg_a(const FragA &f)
{
    FragA n;
#pragma unroll
    for (int e = 0; e < 4; e++) {
        n.hi[e] = f.hi[e] ^ 0x80000000u;
        n.lo[e] = f.lo[e] ^ 0x80000000u;
    }
    return n;
}
__device__ __forceinline__ float2 lds_f2(const unsigned char *p) { return *reinterpret_cast<const float2 *>(p); }

// coefficient fragments (an N x N fp64 matrix, split once per CTA): per (ig, tj) and lane two uint4
//   {ar_hi0, ar_hi1, ar_lo0, ar_lo1}, {ai_hi0, ai_hi1, ai_lo0, ai_lo1},   b0 = a[8 ig + t][8 tj + g], b1 = a[8 ig + t + 4][8 tj + g]
__device__ __forceinline__ void fill_coeff(uint4 *dst, const double2 *__restrict__ a, int N, int NIG, int NTJ)
{
    for (int idx = threadIdx.x; idx < NIG * NTJ * 32; idx += blockDim.x) {
        const int ln = idx & 31, f = idx >> 5;
        const int ig = f / NTJ, tj = f % NTJ;
        const int g = ln >> 2, t = ln & 3;
        const int j = 8 * tj + g, i0 = 8 * ig + t, i1 = i0 + 4;
        const double2 v0 = (i0 < N && j < N) ? a[i0 * N + j] : make_double2(0.0, 0.0);
        const double2 v1 = (i1 < N && j < N) ? a[i1 * N + j] : make_double2(0.0, 0.0);
        uint4 re, im;
        split_tf32((float)v0.x, re.x, re.z);
        split_tf32((float)v1.x, re.y, re.w);
        split_tf32((float)v0.y, im.x, im.z);
        split_tf32((float)v1.y, im.y, im.w);
        dst[(size_t)(2 * f) * 32 + ln] = re;
        dst[(size_t)(2 * f + 1) * 32 + ln] = im;
    }
}
__device__ __forceinline__ void load_coeff(const uint4 *src, int f, int lane, FragB &br, FragB &bi)
{
    const uint4 re = src[(size_t)(2 * f) * 32 + lane], im = src[(size_t)(2 * f + 1) * 32 + lane];
    br.hi[0] = re.x; br.hi[1] = re.y; br.lo[0] = re.z; br.lo[1] = re.w;
    bi.hi[0] = im.x; bi.hi[1] = im.y; bi.lo[0] = im.z; bi.lo[1] = im.w;
}

// A fragments of 16 rows (row_lo = 16 u + g, row_hi = row_lo + 8) of the vectors 8 ig + t, 8 ig + t + 4 of a block in the
// ring (chunk stride rs): real and imaginary parts
__device__ __forceinline__ void load_rows_a(const unsigned char *st, uint32_t rs, int N, int ig, int row_lo, int t, FragA &fr, FragA &fi)
{
    const int i0 = 8 * ig + t, i1 = i0 + 4;
    const float2 z = make_float2(0.f, 0.f);
    const float2 w0 = i0 < N ? lds_f2(st + (size_t)i0 * rs + (size_t)row_lo * 8) : z;
    const float2 w1 = i0 < N ? lds_f2(st + (size_t)i0 * rs + (size_t)(row_lo + 8) * 8) : z;
    const float2 w2 = i1 < N ? lds_f2(st + (size_t)i1 * rs + (size_t)row_lo * 8) : z;
    const float2 w3 = i1 < N ? lds_f2(st + (size_t)i1 * rs + (size_t)(row_lo + 8) * 8) : z;
    const float re[4] = {w0.x, w1.x, w2.x, w3.x}, im[4] = {w0.y, w1.y, w2.y, w3.y};
    split_a(re, fr);
    split_a(im, fi);
}

// One i-group of z += W a on NTJ column tiles.  Four accumulators per tile, one per real product, so that consecutive
// tensor instructions never wait on each other (a single accumulator per part made the kernels latency bound):
//   z[tj][0] += Wr ar   z[tj][1] += -Wi ai   (Re = [0] + [1])      z[tj][2] += Wr ai   z[tj][3] += Wi ar   (Im = [2] + [3])
// tri: 1 = a upper triangular (tiles with ig > tj are zero), 2 = lower triangular (ig < tj), 0 = full
template <int NTJ>
__device__ __forceinline__ void cx_update_ig(float (&z)[NTJ][4][4], const FragA &wr, const FragA &wi, const uint4 *coef, int ig, int lane, int tri)
{
    const FragA nwi = neg_a(wi);
#pragma unroll
    for (int tj = 0; tj < NTJ; tj++) {
        if ((tri == 1 && ig > tj) || (tri == 2 && ig < tj)) continue;
        FragB br, bi;
        load_coeff(coef, ig * NTJ + tj, lane, br, bi);
        hmma_tf32(z[tj][0], wr.lo, br.hi[0], br.hi[1]);
        hmma_tf32(z[tj][1], nwi.lo, bi.hi[0], bi.hi[1]);
        hmma_tf32(z[tj][2], wr.lo, bi.hi[0], bi.hi[1]);
        hmma_tf32(z[tj][3], wi.lo, br.hi[0], br.hi[1]);
        hmma_tf32(z[tj][0], wr.hi, br.lo[0], br.lo[1]);
        hmma_tf32(z[tj][1], nwi.hi, bi.lo[0], bi.lo[1]);
        hmma_tf32(z[tj][2], wr.hi, bi.lo[0], bi.lo[1]);
        hmma_tf32(z[tj][3], wi.hi, br.lo[0], br.lo[1]);
        hmma_tf32(z[tj][0], wr.hi, br.hi[0], br.hi[1]);
        hmma_tf32(z[tj][1], nwi.hi, bi.hi[0], bi.hi[1]);
        hmma_tf32(z[tj][2], wr.hi, bi.hi[0], bi.hi[1]);
        hmma_tf32(z[tj][3], wi.hi, br.hi[0], br.hi[1]);
    }
}
// X == Y: -Xi^dag Xr is minus the transpose of Xr^dag Xi, so c[3] is not computed; the caller forms Im G = A - A^T from
// A = sum of c[2] at the end (the symmetry of the reduction, used on the imaginary part as well)
__device__ __forceinline__ void cx_gram_tile_alias(float (&c)[4][4], const FragA &xr, const FragA &xi, const FragB &yr, const FragB &yi)
{
    hmma_tf32(c[0], xr.lo, yr.hi[0], yr.hi[1]);
    hmma_tf32(c[1], xi.lo, yi.hi[0], yi.hi[1]);
    hmma_tf32(c[2], xr.lo, yi.hi[0], yi.hi[1]);
    hmma_tf32(c[0], xr.hi, yr.lo[0], yr.lo[1]);
    hmma_tf32(c[1], xi.hi, yi.lo[0], yi.lo[1]);
    hmma_tf32(c[2], xr.hi, yi.lo[0], yi.lo[1]);
    hmma_tf32(c[0], xr.hi, yr.hi[0], yr.hi[1]);
    hmma_tf32(c[1], xi.hi, yi.hi[0], yi.hi[1]);
    hmma_tf32(c[2], xr.hi, yi.hi[0], yi.hi[1]);
}
template <int NTJ> __device__ __forceinline__ void zero_z(float (&z)[NTJ][4][4])
{
#pragma unroll
    for (int tj = 0; tj < NTJ; tj++)
#pragma unroll
        for (int c = 0; c < 4; c++)
#pragma unroll
            for (int e = 0; e < 4; e++) z[tj][c][e] = 0.f;
}
// the same four products for a reduction tile: c[0] += Xr Yr, c[1] += Xi Yi (Re = [0] + [1]), c[2] += Xr Yi, c[3] += -Xi Yr (Im = [2] + [3])
__device__ __forceinline__ void cx_gram_tile(float (&c)[4][4], const FragA &xr, const FragA &xi, const FragA &nxi, const FragB &yr, const FragB &yi)
{
    hmma_tf32(c[0], xr.lo, yr.hi[0], yr.hi[1]);
    hmma_tf32(c[1], xi.lo, yi.hi[0], yi.hi[1]);
    hmma_tf32(c[2], xr.lo, yi.hi[0], yi.hi[1]);
    hmma_tf32(c[3], nxi.lo, yr.hi[0], yr.hi[1]);
    hmma_tf32(c[0], xr.hi, yr.lo[0], yr.lo[1]);
    hmma_tf32(c[1], xi.hi, yi.lo[0], yi.lo[1]);
    hmma_tf32(c[2], xr.hi, yi.lo[0], yi.lo[1]);
    hmma_tf32(c[3], nxi.hi, yr.lo[0], yr.lo[1]);
    hmma_tf32(c[0], xr.hi, yr.hi[0], yr.hi[1]);
    hmma_tf32(c[1], xi.hi, yi.hi[0], yi.hi[1]);
    hmma_tf32(c[2], xr.hi, yi.hi[0], yi.hi[1]);
    hmma_tf32(c[3], nxi.hi, yr.hi[0], yr.hi[1]);
}

// ------------------------------------------------------------------------------------------ streaming update
// Z = C + W a, all blocks fp32 (update_tma_kernel<float, float> of mblas.cu).  A unit = 16 rows per warp.
template <int NIG, int NTJ, bool HASC, int CW>
__global__ void __launch_bounds__((CW + 1) * 32, 1)
update_tf32_kernel(size_t L, int N, RingPlan rp, const double2 *__restrict__ a, const float2 *C, const float2 *__restrict__ W, float2 *Z,
                   const int *done, int tri)
{
    extern __shared__ __align__(128) unsigned char dsm[];
    uint64_t *full = reinterpret_cast<uint64_t *>(dsm);
    uint64_t *empty = full + MB_MAX_STAGES;
    uint4 *coef = reinterpret_cast<uint4 *>(dsm + 128);
    unsigned char *ring = dsm + rp.off_ring;
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        for (int s = 0; s < rp.nstg; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], CW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fill_coeff(coef, a, N, NIG, NTJ);
    __syncthreads();

    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const int my = (int)((ntiles > blockIdx.x) ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0);

    if (warp == CW) { // ---------------- producer
        const uint64_t pol = policy_evict_first();
        for (int it = 0; it < my; it++) {
            const int s = it % rp.nstg;
            if (it >= rp.nstg) mbar_wait(&empty[s], ((it / rp.nstg) - 1) & 1);
            const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
            const uint32_t rows = (uint32_t)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
            unsigned char *st = ring + (size_t)s * rp.stage_bytes;
            if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)N * rows * (uint32_t)(HASC ? 16 : 8));
            __syncwarp();
            if (lane < N) {
                tma_load_1d_hint(st + (size_t)lane * rp.rs_a, W + (size_t)lane * L + r0, rows * 8u, &full[s], pol);
                if (HASC) tma_load_1d_hint(st + rp.off_b + (size_t)lane * rp.rs_b, C + (size_t)lane * L + r0, rows * 8u, &full[s], pol);
            }
        }
        return;
    }

    // ---------------- consumers
    const int g = lane >> 2, t = lane & 3;
    for (int it = 0; it < my; it++) {
        const int s = it % rp.nstg;
        const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
        const int rows = (int)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
        const unsigned char *stW = ring + (size_t)s * rp.stage_bytes;
        const unsigned char *stC = stW + rp.off_b;
        mbar_wait_acq(&full[s], (it / rp.nstg) & 1);
        for (int u = warp; u < (rows + 15) / 16; u += CW) {
            const int row_lo = 16 * u + g;
            float z[NTJ][4][4];
            zero_z<NTJ>(z);
#pragma unroll
            for (int ig = 0; ig < NIG; ig++) {
                FragA wr, wi;
                load_rows_a(stW, rp.rs_a, N, ig, row_lo, t, wr, wi);
                cx_update_ig<NTJ>(z, wr, wi, coef, ig, lane, tri);
            }
#pragma unroll
            for (int tj = 0; tj < NTJ; tj++)
#pragma unroll
                for (int e = 0; e < 4; e++) {
                    const int j = 8 * tj + 2 * t + (e & 1), row = row_lo + 8 * (e >> 1);
                    if (j < N && row < rows) {
                        float re = z[tj][0][e] + z[tj][1][e], im = z[tj][2][e] + z[tj][3][e];
                        if (HASC) {
                            const float2 c = lds_f2(stC + (size_t)j * rp.rs_b + (size_t)row * 8);
                            re += c.x;
                            im += c.y;
                        }
                        __stcs(Z + (size_t)j * L + r0 + row, make_float2(re, im));
                    }
                }
        }
        // (the stores take their data from everything the stage was loaded for: the release cannot move above them)
        __syncwarp();
        if (lane == 0) mbar_arrive_rel(&empty[s]);
    }
}

template <int NIG, int NTJ>
static int update_tf32_go(bkr_ctx *ctx, size_t L, int N, const double2 *a, const void *C, const void *W, void *Z, const int *done, int tri)
{
    constexpr int CW = TF_CW;
    const size_t fixed = 128 + (size_t)NIG * NTJ * 2 * 32 * sizeof(uint4);
    const RingPlan rp = plan_ring(L, fixed, 4, N, 8, 32, C ? N : 0, 8, 16);
    if (rp.nstg < 2) return BKR_EINVAL;
    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const unsigned grid = (unsigned)(ntiles < (size_t)BKR_NUM_SMS ? ntiles : (size_t)BKR_NUM_SMS);
    static int attr_dev = -1; // per instantiation: the opt-in is per device
    if (attr_dev != ctx->device) {
        BKR_CUDA(ctx, cudaFuncSetAttribute(update_tf32_kernel<NIG, NTJ, true, CW>, cudaFuncAttributeMaxDynamicSharedMemorySize, MB_SMEM_BUDGET));
        BKR_CUDA(ctx, cudaFuncSetAttribute(update_tf32_kernel<NIG, NTJ, false, CW>, cudaFuncAttributeMaxDynamicSharedMemorySize, MB_SMEM_BUDGET));
        attr_dev = ctx->device;
    }
    if (C)
        update_tf32_kernel<NIG, NTJ, true, CW><<<grid, (CW + 1) * 32, rp.smem, ctx->stream>>>(L, N, rp, a, (const float2 *)C, (const float2 *)W,
                                                                                           (float2 *)Z, done, tri);
    else
        update_tf32_kernel<NIG, NTJ, false, CW><<<grid, (CW + 1) * 32, rp.smem, ctx->stream>>>(L, N, rp, a, nullptr, (const float2 *)W,
                                                                                            (float2 *)Z, done, tri);
    return bkr_check_launch(ctx);
}

int launch_block_update_tf32(bkr_ctx *ctx, int N, const double2 *a, const void *C, const void *W, void *Z, const int *done, int tri)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    switch ((N + 7) / 8) {
    case 1: return update_tf32_go<1, 1>(ctx, L, N, a, C, W, Z, done, tri);
    case 2: return update_tf32_go<2, 2>(ctx, L, N, a, C, W, Z, done, tri);
    case 3: return update_tf32_go<3, 3>(ctx, L, N, a, C, W, Z, done, tri);
    case 4: return update_tf32_go<4, 4>(ctx, L, N, a, C, W, Z, done, tri);
    }
    return BKR_EINVAL;
}

// ------------------------------------------------------------------------------------------ Gram, stage 1
// G = X^dag Y for fp32 blocks: mma tiles of 16 (i) x 8 (j) over k-steps of 8 rows,
//   A[m][k] = X[i0 + m][row k]    B[k][n] = Y[8 nt + n][row k]
//   Re G += Xr Yr + Xi Yi     Im G += Xr Yi - Xi Yr.
// A CTA (blockIdx.y) owns the 16 rows i0 = 16 blockIdx.y .. i0 + 15 of G and the column tiles from jlo on, where
// jlo = i0 for a Hermitian product (tiles wholly below the diagonal are not computed) and 0 otherwise.
// ALIAS (X == Y, Hermitian): one copy of the vectors i0 .. N - 1 in the ring serves both operands, and the B
// fragments of the two column tiles inside the CTA's own 16 rows are the A fragments' registers.
// fp32 accumulators are added into fp64 ones every TF_FLUSH k-steps.  Chunk stride = 32 (mod 128) bytes: the four
// chunks x 32 contiguous bytes a half warp reads per 8-byte load are conflict-free.  Chunk slots of vectors >= N are
// zeroed once and never written.  Deterministic as gram_tma_kernel.
template <int NTN, bool HERM, bool ALIAS, int CW>
__global__ void __launch_bounds__((CW + 1) * 32, 1)
gram_tf32_kernel(size_t L, int N, RingPlan rp, const float2 *__restrict__ X, const float2 *__restrict__ Y, double2 *__restrict__ partials,
                 const int *done)
{
    extern __shared__ __align__(128) unsigned char dsm[];
    uint64_t *full = reinterpret_cast<uint64_t *>(dsm);
    uint64_t *empty = full + MB_MAX_STAGES;
    double2 *red = reinterpret_cast<double2 *>(dsm + 128); // [16][N]: this CTA's rows of G
    unsigned char *ring = dsm + rp.off_ring;
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int i0 = 16 * blockIdx.y;
    const int jlo = HERM ? i0 : 0;
    const int nxv = ALIAS ? N - i0 : min(N - i0, 16); // vectors in the A area (ALIAS: both operands)
    const int nyv = ALIAS ? 0 : N - jlo;              // vectors in the B area
    if (threadIdx.x == 0) {
        for (int s = 0; s < rp.nstg; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], CW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {
        uint4 *z = reinterpret_cast<uint4 *>(ring);
        const size_t n16 = (size_t)rp.nstg * rp.stage_bytes / 16;
        for (size_t o = threadIdx.x; o < n16; o += blockDim.x) z[o] = make_uint4(0, 0, 0, 0);
    }
    for (int o = threadIdx.x; o < 16 * N; o += blockDim.x) red[o] = make_double2(0.0, 0.0);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const int my = (int)((ntiles > blockIdx.x) ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0);

    if (warp == CW) { // ---------------- producer
        const uint64_t pol = policy_evict_first();
        for (int it = 0; it < my; it++) {
            const int s = it % rp.nstg;
            if (it >= rp.nstg) mbar_wait(&empty[s], ((it / rp.nstg) - 1) & 1);
            const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
            const uint32_t rows = (uint32_t)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
            unsigned char *st = ring + (size_t)s * rp.stage_bytes;
            if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)(nxv + nyv) * rows * 8u);
            __syncwarp();
            if (lane < nxv) tma_load_1d_hint(st + (size_t)lane * rp.rs_a, X + (size_t)(i0 + lane) * L + r0, rows * 8u, &full[s], pol);
            if (lane < nyv) tma_load_1d_hint(st + rp.off_b + (size_t)lane * rp.rs_b, Y + (size_t)(jlo + lane) * L + r0, rows * 8u, &full[s], pol);
        }
        return;
    }

    // ---------------- consumers
    const int g = lane >> 2, t = lane & 3;
    const int ntn = (N - jlo + 7) / 8; // column tiles this CTA computes (<= NTN)
    float c[NTN][4][4]; // four independent products per tile (cx_gram_tile)
    double dre[NTN][4], dim[NTN][4];
#pragma unroll
    for (int nt = 0; nt < NTN; nt++)
#pragma unroll
        for (int e = 0; e < 4; e++) dre[nt][e] = dim[nt][e] = 0.0;
    zero_z<NTN>(c);
    auto flush = [&]() {
#pragma unroll
        for (int nt = 0; nt < NTN; nt++)
#pragma unroll
            for (int e = 0; e < 4; e++) {
                dre[nt][e] += (double)(c[nt][0][e] + c[nt][1][e]);
                dim[nt][e] += (double)(c[nt][2][e] + c[nt][3][e]);
            }
        zero_z<NTN>(c);
    };

    int ksteps = 0;
    for (int it = 0; it < my; it++) {
        const int s = it % rp.nstg;
        const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
        const int rows = (int)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
        const unsigned char *stX = ring + (size_t)s * rp.stage_bytes;
        const unsigned char *stY = ALIAS ? stX : stX + rp.off_b;
        const uint32_t rsy = ALIAS ? rp.rs_a : rp.rs_b;
        mbar_wait_acq(&full[s], (it / rp.nstg) & 1);
        const int nks = rows / 8;
        // column tiles past the block (nt >= ntn, the lower CTA row of a Hermitian product) read zeroed chunk slots: no
        // branch in the loop, so that the tensor instructions of all tiles interleave
        for (int k = 0;; k++) {
            const int ks = warp + k * CW;
            if (ks >= nks) break;
            const unsigned char *px = stX + (size_t)(8 * ks + t) * 8;
            const float2 x0 = lds_f2(px + (size_t)g * rp.rs_a), x1 = lds_f2(px + (size_t)(g + 8) * rp.rs_a);
            const float2 x2 = lds_f2(px + (size_t)g * rp.rs_a + 32), x3 = lds_f2(px + (size_t)(g + 8) * rp.rs_a + 32);
            float2 y0[NTN], y1[NTN];
#pragma unroll
            for (int nt = 0; nt < NTN; nt++) {
                if (ALIAS && nt < 2) continue;
                const unsigned char *py = stY + (size_t)(8 * nt + g) * rsy + (size_t)(8 * ks + t) * 8;
                y0[nt] = lds_f2(py);
                y1[nt] = lds_f2(py + 32);
            }
            FragA xr, xi;
            {
                const float re[4] = {x0.x, x1.x, x2.x, x3.x}, im[4] = {x0.y, x1.y, x2.y, x3.y};
                split_a(re, xr);
                split_a(im, xi);
            }
            const FragA nxi = neg_a(xi);
#pragma unroll
            for (int nt = 0; nt < NTN; nt++) {
                FragB yr, yi;
                if (ALIAS && nt < 2) { // the column tile lies inside this CTA's own 16 vectors: same registers
                    yr.hi[0] = xr.hi[nt]; yr.hi[1] = xr.hi[nt + 2]; yr.lo[0] = xr.lo[nt]; yr.lo[1] = xr.lo[nt + 2];
                    yi.hi[0] = xi.hi[nt]; yi.hi[1] = xi.hi[nt + 2]; yi.lo[0] = xi.lo[nt]; yi.lo[1] = xi.lo[nt + 2];
                } else {
                    split_tf32(y0[nt].x, yr.hi[0], yr.lo[0]);
                    split_tf32(y1[nt].x, yr.hi[1], yr.lo[1]);
                    split_tf32(y0[nt].y, yi.hi[0], yi.lo[0]);
                    split_tf32(y1[nt].y, yi.hi[1], yi.lo[1]);
                }
                cx_gram_tile(c[nt], xr, xi, nxi, yr, yi);
            }
            if ((++ksteps & (TF_FLUSH - 1)) == 0) flush();
        }
        // release through an address that depends on the accumulators (which took everything loaded from the stage)
        uint32_t dep = 0;
#pragma unroll
        for (int nt = 0; nt < NTN; nt++)
#pragma unroll
            for (int e = 0; e < 4; e++)
                dep |= (uint32_t)__double2loint(dre[nt][e]) | (uint32_t)__double2loint(dim[nt][e]) | __float_as_uint(c[nt][0][e]) |
                       __float_as_uint(c[nt][1][e]) | __float_as_uint(c[nt][2][e]) | __float_as_uint(c[nt][3][e]);
        dep &= rp.zero;
        __syncwarp();
        if (lane == 0) mbar_arrive_rel(reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(&empty[s]) + dep));
    }

    flush();
    // fixed-order reduction over the consumer warps, then one partial (this CTA's 16 rows of G) per CTA
    for (int w = 0; w < CW; w++) {
        if (warp == w) {
#pragma unroll
            for (int nt = 0; nt < NTN; nt++)
#pragma unroll
                for (int e = 0; e < 4; e++) {
                    const int il = g + 8 * (e >> 1), j = jlo + 8 * nt + 2 * t + (e & 1);
                    if (nt < ntn && i0 + il < N && j < N) {
                        double2 v = red[il * N + j];
                        v.x += dre[nt][e];
                        v.y += dim[nt][e];
                        red[il * N + j] = v;
                    }
                }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(CW * 32) : "memory");
    }
    const int nrow = min(16, N - i0);
    for (int o = threadIdx.x; o < nrow * N; o += CW * 32) partials[(size_t)blockIdx.x * N * N + (size_t)i0 * N + o] = red[o];
}

template <int NTN>
static int gram_tf32_go(bkr_ctx *ctx, size_t L, int N, const void *X, const void *Y, int hermitian, int *num_partials, const int *done)
{
    constexpr int CW = NTN <= 2 ? 12 : TF_CW; // measured: 8 warps 0.111 ms, 12 0.097, 14 0.104 (32^4, N = 16, two blocks)
    const bool alias = hermitian && X == Y;
    const size_t fixed = 128 + (size_t)16 * N * sizeof(double2);
    const RingPlan rp = plan_ring(L, fixed, 3, (alias && NTN > 2) ? 8 * NTN : 16, 8, 32, alias ? 0 : 8 * NTN, 8, 32); // A area: >= 16 slots
    if (rp.nstg < 2) return BKR_EINVAL;
    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const unsigned gx = (unsigned)(ntiles < (size_t)BKR_NUM_SMS ? ntiles : (size_t)BKR_NUM_SMS);
    const dim3 grid(gx, (N + 15) / 16);
#define GRAM_TF32_LAUNCH(H_, A_)                                                                                                   \
    do {                                                                                                                           \
        static int attr_dev = -1;                                                                                                  \
        if (attr_dev != ctx->device) {                                                                                             \
            BKR_CUDA(ctx, cudaFuncSetAttribute(gram_tf32_kernel<NTN, H_, A_, CW>, cudaFuncAttributeMaxDynamicSharedMemorySize, MB_SMEM_BUDGET)); \
            attr_dev = ctx->device;                                                                                                \
        }                                                                                                                          \
        gram_tf32_kernel<NTN, H_, A_, CW><<<grid, (CW + 1) * 32, rp.smem, ctx->stream>>>(L, N, rp, (const float2 *)X, (const float2 *)Y,  \
                                                                                       ctx->partials, done);                      \
    } while (0)
    if (alias) GRAM_TF32_LAUNCH(true, true);
    else if (hermitian) GRAM_TF32_LAUNCH(true, false);
    else GRAM_TF32_LAUNCH(false, false);
#undef GRAM_TF32_LAUNCH
    *num_partials = (int)gx;
    return bkr_check_launch(ctx);
}

// fp32 blocks, N <= 32; partials as launch_gram_partials (Hermitian: entries below the 16-row diagonal blocks are not written)
int launch_gram_partials_tf32(bkr_ctx *ctx, int N, const void *X, const void *Y, int hermitian, int *num_partials, const int *done)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    BKR_TRY(ensure_partials(ctx, (size_t)2 * BKR_NUM_SMS * BKR_MAX_N * BKR_MAX_N * sizeof(double2)));
    switch ((N + 7) / 8) {
    case 1: return gram_tf32_go<1>(ctx, L, N, X, Y, hermitian, num_partials, done);
    case 2: return gram_tf32_go<2>(ctx, L, N, X, Y, hermitian, num_partials, done);
    case 3: return gram_tf32_go<3>(ctx, L, N, X, Y, hermitian, num_partials, done);
    case 4: return gram_tf32_go<4>(ctx, L, N, X, Y, hermitian, num_partials, done);
    }
    return BKR_EINVAL;
}

// ------------------------------------------------------------------------------------------ fused Q / P / X update
// pqx_update_kernel of mblas.cu for fp32 Q, P (X fp64):  Q = Q' Si,  Pn = Q + P Sd,  X += P Wm  in one pass.  The increment
// P Wm is formed in fp32 (<= 64 split products per entry) and added to the fp64 X.
template <int NIG, int NTJ, int CW>
__global__ void __launch_bounds__((CW + 1) * 32, 1)
pqx_tf32_kernel(size_t L, int N, Ring3 rp, const double2 *__restrict__ Si, const double2 *__restrict__ Sd, const double2 *__restrict__ Wm,
                float2 *Q, const float2 *__restrict__ P, float2 *__restrict__ Pn, double2 *X, const SolverFlags *fl)
{
    constexpr int NC = NIG * NTJ * 2 * 32; // uint4 per coefficient matrix
    extern __shared__ __align__(128) unsigned char dsm[];
    uint64_t *full = reinterpret_cast<uint64_t *>(dsm);
    uint64_t *empty = full + MB_MAX_STAGES;
    uint4 *c0 = reinterpret_cast<uint4 *>(dsm + 128), *c1 = c0 + NC, *c2 = c1 + NC; // Si, Sd, Wm
    unsigned char *ring = dsm + rp.off_ring;
    const bool doX = fl->xpend != 0, doP = fl->done == 0;
    if (!doX && !doP) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        for (int s = 0; s < rp.nstg; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], CW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fill_coeff(c0, Si, N, NIG, NTJ);
    fill_coeff(c1, Sd, N, NIG, NTJ);
    fill_coeff(c2, Wm, N, NIG, NTJ);
    __syncthreads();

    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const int my = (int)((ntiles > blockIdx.x) ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0);

    if (warp == CW) { // ---------------- producer
        const uint64_t pol = policy_evict_first();
        for (int it = 0; it < my; it++) {
            const int s = it % rp.nstg;
            if (it >= rp.nstg) mbar_wait(&empty[s], ((it / rp.nstg) - 1) & 1);
            const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
            const uint32_t rows = (uint32_t)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
            unsigned char *st = ring + (size_t)s * rp.stage_bytes;
            if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)N * rows * (uint32_t)(8 + (doP ? 8 : 0) + (doX ? 16 : 0)));
            __syncwarp();
            if (lane < N) {
                tma_load_1d_hint(st + (size_t)lane * rp.rs_p, P + (size_t)lane * L + r0, rows * 8u, &full[s], pol);
                if (doP) tma_load_1d_hint(st + rp.off_q + (size_t)lane * rp.rs_q, Q + (size_t)lane * L + r0, rows * 8u, &full[s], pol);
                if (doX) tma_load_1d_hint(st + rp.off_x + (size_t)lane * rp.rs_x, X + (size_t)lane * L + r0, rows * 16u, &full[s], pol);
            }
        }
        return;
    }

    // ---------------- consumers
    const int g = lane >> 2, t = lane & 3;
    for (int it = 0; it < my; it++) {
        const int s = it % rp.nstg;
        const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
        const int rows = (int)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
        const unsigned char *stP = ring + (size_t)s * rp.stage_bytes;
        const unsigned char *stQ = stP + rp.off_q, *stX = stP + rp.off_x;
        mbar_wait_acq(&full[s], (it / rp.nstg) & 1);
        for (int u = warp; u < (rows + 15) / 16; u += CW) {
            const int row_lo = 16 * u + g;
            FragA pr[NIG], pi[NIG];
#pragma unroll
            for (int ig = 0; ig < NIG; ig++) load_rows_a(stP, rp.rs_p, N, ig, row_lo, t, pr[ig], pi[ig]);
            float z[NTJ][4][4];
            if (doP) {
                zero_z<NTJ>(z);
#pragma unroll
                for (int ig = 0; ig < NIG; ig++) { // Q = Q' Si, Si upper triangular
                    FragA qr, qi;
                    load_rows_a(stQ, rp.rs_q, N, ig, row_lo, t, qr, qi);
                    cx_update_ig<NTJ>(z, qr, qi, c0, ig, lane, 1);
                }
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++)
#pragma unroll
                    for (int e = 0; e < 4; e++) {
                        const int j = 8 * tj + 2 * t + (e & 1), row = row_lo + 8 * (e >> 1);
                        if (j < N && row < rows) __stcs(Q + (size_t)j * L + r0 + row, make_float2(z[tj][0][e] + z[tj][1][e], z[tj][2][e] + z[tj][3][e]));
                    }
#pragma unroll
                for (int ig = 0; ig < NIG; ig++) cx_update_ig<NTJ>(z, pr[ig], pi[ig], c1, ig, lane, 2); // + P Sd, Sd lower triangular
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++)
#pragma unroll
                    for (int e = 0; e < 4; e++) {
                        const int j = 8 * tj + 2 * t + (e & 1), row = row_lo + 8 * (e >> 1);
                        if (j < N && row < rows) __stcs(Pn + (size_t)j * L + r0 + row, make_float2(z[tj][0][e] + z[tj][1][e], z[tj][2][e] + z[tj][3][e]));
                    }
            }
            if (doX) {
                zero_z<NTJ>(z);
#pragma unroll
                for (int ig = 0; ig < NIG; ig++) cx_update_ig<NTJ>(z, pr[ig], pi[ig], c2, ig, lane, 0);
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++)
#pragma unroll
                    for (int e = 0; e < 4; e++) {
                        const int j = 8 * tj + 2 * t + (e & 1), row = row_lo + 8 * (e >> 1);
                        if (j < N && row < rows) {
                            const double2 c = *reinterpret_cast<const double2 *>(stX + (size_t)j * rp.rs_x + (size_t)row * 16);
                            __stcs(X + (size_t)j * L + r0 + row, make_double2(c.x + (double)(z[tj][0][e] + z[tj][1][e]), c.y + (double)(z[tj][2][e] + z[tj][3][e])));
                        }
                    }
            }
        }
        // (the stores take their data from everything the stage was loaded for: the release cannot move above them)
        __syncwarp();
        if (lane == 0) mbar_arrive_rel(&empty[s]);
    }
}

template <int NIG>
static int pqx_tf32_go(bkr_ctx *ctx, size_t L, int N, const double2 *Si, const double2 *Sd, const double2 *Wm, void *Q, const void *P, void *Pn,
                       double2 *X, const SolverFlags *fl)
{
    constexpr int CW = NIG == 2 ? 11 : TF_CW;
    const size_t fixed = (128 + (size_t)3 * NIG * NIG * 2 * 32 * sizeof(uint4) + 127) / 128 * 128;
    const Ring3 rp = plan_ring3(L, N, fixed, 8);
    if (rp.nstg < 2) return BKR_EINVAL;
    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const unsigned grid = (unsigned)(ntiles < (size_t)BKR_NUM_SMS ? ntiles : (size_t)BKR_NUM_SMS);
    static int attr_dev = -1; // per instantiation: the opt-in is per device
    if (attr_dev != ctx->device) {
        BKR_CUDA(ctx, cudaFuncSetAttribute(pqx_tf32_kernel<NIG, NIG, CW>, cudaFuncAttributeMaxDynamicSharedMemorySize, MB_SMEM_BUDGET));
        attr_dev = ctx->device;
    }
    pqx_tf32_kernel<NIG, NIG, CW><<<grid, (CW + 1) * 32, rp.smem, ctx->stream>>>(L, N, rp, Si, Sd, Wm, (float2 *)Q, (const float2 *)P, (float2 *)Pn,
                                                                                X, fl);
    return bkr_check_launch(ctx);
}

// fp32 Q, P; N <= 16 (at 17-24 rhs the three coefficient sets and the fragments spill: 2.1 ms against 0.80 ms for the FP64
// tensor kernel on 32^4); BKR_EINVAL above
int launch_pqx_update_tf32(bkr_ctx *ctx, int N, const double2 *Sinv, const double2 *Sdag, const double2 *Wm, void *Q, const void *P, void *Pn,
                           double2 *X, const SolverFlags *flags)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    switch ((N + 7) / 8) {
    case 1: return pqx_tf32_go<1>(ctx, L, N, Sinv, Sdag, Wm, Q, P, Pn, X, flags);
    case 2: return pqx_tf32_go<2>(ctx, L, N, Sinv, Sdag, Wm, Q, P, Pn, X, flags);
    }
    return BKR_EINVAL;
}

// ------------------------------------------------------------------------------------------ fused update + aliased Gram
// update_gram_kernel of mblas.cu for fp32 blocks, N <= 16:  Z = C + W a  and  H = Z^dag Z  (Hermitian) in one pass.  Each warp
// writes its 16 finished rows of Z over the C rows it has consumed in the ring and reads them back as fragments of the
// reduction (two k-steps of 8 rows); the fp32 accumulators of H go into the fp64 ones after every unit.
template <int NT, int CW>
__global__ void __launch_bounds__((CW + 1) * 32, 1)
update_gram_tf32_kernel(size_t L, int N, RingPlan rp, uint32_t off_red, const double2 *__restrict__ a, const float2 *C,
                        const float2 *__restrict__ W, float2 *Z, double2 *__restrict__ partials, const int *done)
{
    extern __shared__ __align__(128) unsigned char dsm[];
    uint64_t *full = reinterpret_cast<uint64_t *>(dsm);
    uint64_t *empty = full + MB_MAX_STAGES;
    uint4 *coef = reinterpret_cast<uint4 *>(dsm + 128);
    double2 *red = reinterpret_cast<double2 *>(dsm + off_red); // [N * N]
    unsigned char *ring = dsm + rp.off_ring;
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        for (int s = 0; s < rp.nstg; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], CW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fill_coeff(coef, a, N, NT, NT);
    for (int o = threadIdx.x; o < N * N; o += blockDim.x) red[o] = make_double2(0.0, 0.0);
    __syncthreads();

    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const int my = (int)((ntiles > blockIdx.x) ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0);

    if (warp == CW) { // ---------------- producer
        const uint64_t pol = policy_evict_first();
        for (int it = 0; it < my; it++) {
            const int s = it % rp.nstg;
            if (it >= rp.nstg) mbar_wait(&empty[s], ((it / rp.nstg) - 1) & 1);
            const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
            const uint32_t rows = (uint32_t)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
            unsigned char *st = ring + (size_t)s * rp.stage_bytes;
            if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)N * rows * 16u);
            __syncwarp();
            if (lane < N) {
                tma_load_1d_hint(st + (size_t)lane * rp.rs_a, W + (size_t)lane * L + r0, rows * 8u, &full[s], pol);
                tma_load_1d_hint(st + rp.off_b + (size_t)lane * rp.rs_b, C + (size_t)lane * L + r0, rows * 8u, &full[s], pol);
            }
        }
        return;
    }

    // ---------------- consumers
    const int g = lane >> 2, t = lane & 3;
    constexpr int UG_FLUSH = 1; // units (16 rows) between flushes of the fp32 accumulators (more: the registers spill)
    float c[NT][4][4];          // [2] holds A = Zr^dag Zi, [3] is unused (cx_gram_tile_alias)
    double dre[NT][4], dim[NT][4];
#pragma unroll
    for (int nt = 0; nt < NT; nt++)
#pragma unroll
        for (int e = 0; e < 4; e++) dre[nt][e] = dim[nt][e] = 0.0;
    zero_z<NT>(c);
    auto flush = [&]() {
#pragma unroll
        for (int nt = 0; nt < NT; nt++)
#pragma unroll
            for (int e = 0; e < 4; e++) {
                dre[nt][e] += (double)(c[nt][0][e] + c[nt][1][e]);
                dim[nt][e] += (double)c[nt][2][e];
                c[nt][0][e] = c[nt][1][e] = c[nt][2][e] = 0.f;
            }
    };
    int units = 0;
    for (int it = 0; it < my; it++) {
        const int s = it % rp.nstg;
        const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
        const int rows = (int)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
        const unsigned char *stW = ring + (size_t)s * rp.stage_bytes;
        unsigned char *stC = ring + (size_t)s * rp.stage_bytes + rp.off_b;
        mbar_wait_acq(&full[s], (it / rp.nstg) & 1);
        for (int u = warp; u < (rows + 15) / 16; u += CW) {
            const int row_lo = 16 * u + g;
            float z[NT][4][4];
            zero_z<NT>(z);
#pragma unroll
            for (int ig = 0; ig < NT; ig++) {
                FragA wr, wi;
                load_rows_a(stW, rp.rs_a, N, ig, row_lo, t, wr, wi);
                cx_update_ig<NT>(z, wr, wi, coef, ig, lane, 0);
            }
#pragma unroll
            for (int tj = 0; tj < NT; tj++)
#pragma unroll
                for (int e = 0; e < 4; e++) {
                    const int j = 8 * tj + 2 * t + (e & 1), row = row_lo + 8 * (e >> 1);
                    if (j < N && row < rows) {
                        float2 *cp = reinterpret_cast<float2 *>(stC + (size_t)j * rp.rs_b + (size_t)row * 8);
                        const float2 c = *cp;
                        const float2 zv = make_float2(z[tj][0][e] + z[tj][1][e] + c.x, z[tj][2][e] + z[tj][3][e] + c.y);
                        *cp = zv; // H is the Gram matrix of what is stored
                        __stcs(Z + (size_t)j * L + r0 + row, zv);
                    }
                }
            __syncwarp();
            const int nk = (rows - 16 * u >= 16) ? 2 : 1; // the last unit of a ragged block has 8 rows
            for (int h = 0; h < nk; h++) {
                const unsigned char *px = stC + (size_t)(16 * u + 8 * h + t) * 8;
                const float2 z = make_float2(0.f, 0.f);
                const float2 x0 = g < N ? lds_f2(px + (size_t)g * rp.rs_b) : z, x1 = g + 8 < N ? lds_f2(px + (size_t)(g + 8) * rp.rs_b) : z;
                const float2 x2 = g < N ? lds_f2(px + (size_t)g * rp.rs_b + 32) : z, x3 = g + 8 < N ? lds_f2(px + (size_t)(g + 8) * rp.rs_b + 32) : z;
                FragA xr, xi;
                {
                    const float re[4] = {x0.x, x1.x, x2.x, x3.x}, im[4] = {x0.y, x1.y, x2.y, x3.y};
                    split_a(re, xr);
                    split_a(im, xi);
                }
#pragma unroll
                for (int nt = 0; nt < NT; nt++) {
                    FragB yr, yi;
                    yr.hi[0] = xr.hi[nt]; yr.hi[1] = xr.hi[nt + 2]; yr.lo[0] = xr.lo[nt]; yr.lo[1] = xr.lo[nt + 2];
                    yi.hi[0] = xi.hi[nt]; yi.hi[1] = xi.hi[nt + 2]; yi.lo[0] = xi.lo[nt]; yi.lo[1] = xi.lo[nt + 2];
                    cx_gram_tile_alias(c[nt], xr, xi, yr, yi);
                }
            }
            if ((++units & (UG_FLUSH - 1)) == 0) flush();
        }
        // generic-proxy writes to the stage before the async-proxy (TMA) refill of the same shared memory
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        uint32_t dep = 0; // everything read from the stage went into c (or, just flushed, into dre / dim)
#pragma unroll
        for (int nt = 0; nt < NT; nt++)
#pragma unroll
            for (int e = 0; e < 4; e++)
                dep |= (uint32_t)__double2loint(dre[nt][e]) | (uint32_t)__double2loint(dim[nt][e]) | __float_as_uint(c[nt][0][e]) |
                       __float_as_uint(c[nt][1][e]) | __float_as_uint(c[nt][2][e]);
        dep &= rp.zero;
        __syncwarp();
        if (lane == 0) mbar_arrive_rel(reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(&empty[s]) + dep));
    }
    flush();
    for (int w = 0; w < CW; w++) { // fixed-order reduction over the consumer warps (named barrier 1: the producer has left)
        if (warp == w) {
#pragma unroll
            for (int nt = 0; nt < NT; nt++)
#pragma unroll
                for (int e = 0; e < 4; e++) {
                    const int i = g + 8 * (e >> 1), j = 8 * nt + 2 * t + (e & 1);
                    if (i < N && j < N) {
                        double2 v = red[i * N + j];
                        v.x += dre[nt][e];
                        v.y += dim[nt][e];
                        red[i * N + j] = v;
                    }
                }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(CW * 32) : "memory");
    }
    // red.y holds A = Zr^dag Zi: Im H = A - A^T
    for (int o = threadIdx.x; o < N * N; o += CW * 32) {
        const int i = o / N, j = o % N;
        partials[(size_t)blockIdx.x * N * N + o] = make_double2(red[o].x, red[o].y - red[j * N + i].y);
    }
}

template <int NT>
static int update_gram_tf32_go(bkr_ctx *ctx, size_t L, int N, const double2 *a, const void *C, const void *W, void *Z, int *num_partials,
                               const int *done)
{
    constexpr int CW = TF_CW; // 10 warps: 0.196 ms against 0.184 (a stage is 16 units)
    const size_t off_red = (128 + (size_t)NT * NT * 2 * 32 * sizeof(uint4) + 127) / 128 * 128;
    const size_t fixed = off_red + (size_t)N * N * sizeof(double2);
    const RingPlan rp = plan_ring(L, fixed, 4, N, 8, 32, N, 8, 16);
    if (rp.nstg < 2) return BKR_EINVAL;
    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const unsigned grid = (unsigned)(ntiles < (size_t)BKR_NUM_SMS ? ntiles : (size_t)BKR_NUM_SMS);
    BKR_TRY(ensure_partials(ctx, (size_t)2 * BKR_NUM_SMS * BKR_MAX_N * BKR_MAX_N * sizeof(double2)));
    static int attr_dev = -1; // per instantiation: the opt-in is per device
    if (attr_dev != ctx->device) {
        BKR_CUDA(ctx, cudaFuncSetAttribute(update_gram_tf32_kernel<NT, CW>, cudaFuncAttributeMaxDynamicSharedMemorySize, MB_SMEM_BUDGET));
        attr_dev = ctx->device;
    }
    update_gram_tf32_kernel<NT, CW><<<grid, (CW + 1) * 32, rp.smem, ctx->stream>>>(L, N, rp, (uint32_t)off_red, a, (const float2 *)C,
                                                                                  (const float2 *)W, (float2 *)Z, ctx->partials, done);
    *num_partials = (int)grid;
    return bkr_check_launch(ctx);
}

// fp32 blocks, N <= 16; BKR_EINVAL above
int launch_update_gram_tf32(bkr_ctx *ctx, int N, const double2 *a, const void *C, const void *W, void *Z, int *num_partials, const int *done)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    if (N <= 8) return update_gram_tf32_go<1>(ctx, L, N, a, C, W, Z, num_partials, done);
    if (N <= 16) return update_gram_tf32_go<2>(ctx, L, N, a, C, W, Z, num_partials, done);
    return BKR_EINVAL;
}
