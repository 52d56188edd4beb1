// Multi-BLAS on native blocks v[j][k] (N vectors of L = 3 Vh complex, row index k contiguous):
//   reduction multi-BLAS  K = X^dag Y          PAPER.md:272-299 (eq. 4)
//   streaming multi-BLAS  Z = C + W a          PAPER.md:245-270 (eq. 3; Alg. 1 l.8, l.10, l.11, Alg. 2 l.4)
// Both stream every vector element once, so memory traffic is linear in N.
//
// Design.  These kernels are HBM streams with a small dense contraction attached, and the
// first version (one warp = 16 rows, loads -> DMMA -> loads -> stores in program order) was latency bound: ncu showed
// 48 of 56 cycles per issued instruction on the long scoreboard and 42 % of DRAM bandwidth, because a warp had at most
// 4 KB in flight.  Here the loads are taken off the warps altogether:
//  * persistent CTAs (one per SM) of one producer warp and CW consumer warps;
//  * the producer streams row tiles -- R rows of every vector of the block(s), one contiguous R x 16-byte chunk per
//    vector -- into a shared-memory ring with 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx, evict_first),
//    so ~150 KB per SM are in flight whatever the register budget;
//  * consumers read DMMA fragments from the ring with conflict-free 16-byte shared loads (the chunk stride is padded
//    so that the 8 lanes of a quarter warp hit 8 different 16-byte bank groups) and never wait on global memory.
// Arithmetic: both are tall-skinny complex GEMMs (inner or outer dimension N <= 32).  On B200 the FP64 tensor path
// (DMMA m8n8k4) runs at the same peak as DFMA (measured 36.8 vs 36.7 TFLOP/s), so it raises no ceiling; it is used
// because one DMMA replaces 8 DFMAs per lane and needs 2 operand registers for 8 FMAs.  A complex product is 4 real
// DMMAs.  All accumulation is fp64 whatever the storage precision.  Reductions finish in a fixed order (no
// floating-point atomics): results are bit-reproducible.
#include "mblas.cuh"

// The accumulator fragment of an 8 x 8 tile (lane 4 m + q holds row m, columns 2 q and 2 q + 1) -> the same entries of the
// TRANSPOSED tile, by shuffles.  For a diagonal tile of X^dag X the product Xi^dag Xr is the transpose of Xr^dag Xi
// (same products, same order of summation), so its DMMAs are not issued at all (the symmetry of the
// reduction used inside a tile as well).  All 32 lanes must call it.
__device__ __forceinline__ void frag_transpose(const double (&c)[2], double (&t)[2], int m, int q)
{
#pragma unroll
    for (int r = 0; r < 2; r++) {
        const int src = (2 * q + r) * 4 + (m >> 1);
        const double v0 = __shfl_sync(0xffffffffu, c[0], src), v1 = __shfl_sync(0xffffffffu, c[1], src);
        t[r] = (m & 1) ? v1 : v0;
    }
}

// ------------------------------------------------------------------------------------------ streaming update
// Z = C + W a  as  D(8 rows x 8 j) += A(8 rows x 4 i) B(4 i x 8 j) with DMMA m8n8k4:
//   A[m][q] = W[4 is + q][row m]      lane = 4 m + q reads one complex (Re and Im) from the ring,
//   B[q][n] = a[4 is + q][8 tj + n]   in fragment order (registers for N <= 16, shared memory above),
//   Re Z += Wr ar - Wi ai      Im Z += Wr ai + Wi ar.
// The accumulator fragment of lane (m, q) holds columns j = 8 tj + 2 q + r, r = 0, 1 of row m: C is read from the ring
// and Z written to global memory in that layout (8 consecutive rows of 4 vectors per instruction: full 128-byte
// segments).  Chunk strides: W = 32 (mod 128) bytes, C = 16 (mod 128): both fragment patterns are conflict-free.
// Z may alias C (the tile of C is in shared memory before the rows of Z are written); Z must not alias W.
template <typename RealZ, typename RealW, int NTJ, int NIS, bool HASC, int CW>
__global__ void __launch_bounds__((CW + 1) * 32, 1)
update_tma_kernel(size_t L, int N, RingPlan rp, const double2 *__restrict__ a, const typename CxT<RealZ>::type *C,
                  const typename CxT<RealW>::type *__restrict__ W, typename CxT<RealZ>::type *Z, const int *done, int tri)
{
    typedef typename CxT<RealZ>::type CxZ;
    typedef typename CxT<RealW>::type CxW;
    constexpr bool BREG = NIS * NTJ <= 8; // coefficient fragments in registers
    constexpr int NF = NIS * NTJ * 32;
    extern __shared__ __align__(128) unsigned char dsm[];
    uint64_t *full = reinterpret_cast<uint64_t *>(dsm);
    uint64_t *empty = full + MB_MAX_STAGES;
    double *bre = reinterpret_cast<double *>(dsm + 128), *bim = bre + NF;
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
    for (int idx = threadIdx.x; idx < NF; idx += blockDim.x) {
        const int ln = idx & 31, f = idx >> 5;
        const int is = f / NTJ, tj = f % NTJ;
        const int i = 4 * is + (ln & 3), j = 8 * tj + (ln >> 2);
        const double2 v = (i < N && j < N) ? a[i * N + j] : make_double2(0.0, 0.0);
        bre[idx] = v.x;
        bim[idx] = v.y;
    }
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
            if (lane == 0)
                mbar_expect_tx(&full[s], (uint32_t)N * rows * (uint32_t)(sizeof(CxW) + (HASC ? sizeof(CxZ) : 0)));
            __syncwarp();
            if (lane < N) {
                tma_load_1d_hint(st + (size_t)lane * rp.rs_a, W + (size_t)lane * L + r0, rows * (uint32_t)sizeof(CxW), &full[s], pol);
                if (HASC)
                    tma_load_1d_hint(st + rp.off_b + (size_t)lane * rp.rs_b, C + (size_t)lane * L + r0,
                                     rows * (uint32_t)sizeof(CxZ), &full[s], pol);
            }
        }
        return;
    }

    // ---------------- consumers
    const int m = lane >> 2, q = lane & 3;
    double ar[BREG ? NIS * NTJ : 1], ai[BREG ? NIS * NTJ : 1];
    if (BREG) {
#pragma unroll
        for (int f = 0; f < NIS * NTJ; f++) {
            ar[f] = bre[f * 32 + lane];
            ai[f] = bim[f * 32 + lane];
        }
    }
    for (int it = 0; it < my; it++) {
        const int s = it % rp.nstg;
        const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
        const int rows = (int)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
        const unsigned char *stW = ring + (size_t)s * rp.stage_bytes;
        const unsigned char *stC = stW + rp.off_b;
        mbar_wait_acq(&full[s], (it / rp.nstg) & 1);
        for (int u = warp; u < rows / 8; u += CW) {
            const int row = 8 * u + m;
            double2 wf[NIS];
#pragma unroll
            for (int is = 0; is < NIS; is++) {
                const int i = 4 * is + q;
                wf[is] = i < N ? sm_cx<CxW>(stW + (size_t)i * rp.rs_a + (size_t)row * sizeof(CxW)) : make_double2(0.0, 0.0);
            }
            double zre[NTJ][2], zim[NTJ][2];
#pragma unroll
            for (int tj = 0; tj < NTJ; tj++) zre[tj][0] = zre[tj][1] = zim[tj][0] = zim[tj][1] = 0.0;
#pragma unroll
            for (int is = 0; is < NIS; is++) {
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++) {
                    // triangular coefficients: fragments wholly on the zero side are skipped, not read
                    if ((tri == 1 && 4 * is > 8 * tj + 7) || (tri == 2 && 4 * is + 3 < 8 * tj)) continue;
                    const int f = is * NTJ + tj;
                    const double br = BREG ? ar[f] : bre[f * 32 + lane], bi = BREG ? ai[f] : bim[f * 32 + lane];
                    dmma(zre[tj], wf[is].x, br);
                    dmma(zre[tj], wf[is].y, -bi);
                    dmma(zim[tj], wf[is].x, bi);
                    dmma(zim[tj], wf[is].y, br);
                }
            }
#pragma unroll
            for (int tj = 0; tj < NTJ; tj++) {
#pragma unroll
                for (int r = 0; r < 2; r++) {
                    const int j = 8 * tj + 2 * q + r;
                    if (j < N) {
                        double re = zre[tj][r], im = zim[tj][r];
                        if (HASC) {
                            const double2 c = sm_cx<CxZ>(stC + (size_t)j * rp.rs_b + (size_t)row * sizeof(CxZ));
                            re += c.x;
                            im += c.y;
                        }
                        st_cx<CxZ>(Z + (size_t)j * L + r0 + row, re, im);
                    }
                }
            }
        }
        // (the stores above take their data from everything the stage was loaded for: a release cannot move above them,
        // so the loads have returned -- no fence needed here, dslash_win.cu has the story)
        __syncwarp();
        if (lane == 0) mbar_arrive_rel(&empty[s]);
    }
}

template <typename RealZ, typename RealW, int NTJ, int NIS>
static int update_go(bkr_ctx *ctx, size_t L, int N, const double2 *a, const void *C, const void *W, void *Z, const int *done, int tri)
{
    typedef typename CxT<RealZ>::type CxZ;
    typedef typename CxT<RealW>::type CxW;
    constexpr int CW = 8;
    const size_t fixed = 128 + (size_t)2 * NIS * NTJ * 32 * sizeof(double);
    const RingPlan rp = plan_ring(L, fixed, 4, N, (int)sizeof(CxW), 32, C ? N : 0, (int)sizeof(CxZ), 16);
    if (rp.nstg < 2) return BKR_EINVAL;
    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const unsigned grid = (unsigned)(ntiles < (size_t)BKR_NUM_SMS ? ntiles : (size_t)BKR_NUM_SMS);
    static int attr_dev = -1; // per instantiation: the opt-in is per device
    if (attr_dev != ctx->device) {
        BKR_CUDA(ctx, cudaFuncSetAttribute(update_tma_kernel<RealZ, RealW, NTJ, NIS, true, CW>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, MB_SMEM_BUDGET));
        BKR_CUDA(ctx, cudaFuncSetAttribute(update_tma_kernel<RealZ, RealW, NTJ, NIS, false, CW>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, MB_SMEM_BUDGET));
        attr_dev = ctx->device;
    }
    if (C)
        update_tma_kernel<RealZ, RealW, NTJ, NIS, true, CW><<<grid, (CW + 1) * 32, rp.smem, ctx->stream>>>(
            L, N, rp, a, (const CxZ *)C, (const CxW *)W, (CxZ *)Z, done, tri);
    else
        update_tma_kernel<RealZ, RealW, NTJ, NIS, false, CW><<<grid, (CW + 1) * 32, rp.smem, ctx->stream>>>(
            L, N, rp, a, nullptr, (const CxW *)W, (CxZ *)Z, done, tri);
    return bkr_check_launch(ctx);
}

template <typename RealZ, typename RealW>
static int launch_update_t(bkr_ctx *ctx, int N, const double2 *a, const void *C, const void *W, void *Z, const int *done, int tri)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    const int NIS = (N + 3) / 4;
#define UPD_GO(NTJ_, NIS_) return update_go<RealZ, RealW, NTJ_, NIS_>(ctx, L, N, a, C, W, Z, done, tri)
    switch (NIS) {
    case 1: UPD_GO(1, 1);
    case 2: UPD_GO(1, 2);
    case 3: UPD_GO(2, 3);
    case 4: UPD_GO(2, 4);
    case 5: UPD_GO(3, 5);
    case 6: UPD_GO(3, 6);
    case 7: UPD_GO(4, 7);
    default: UPD_GO(4, 8);
    }
#undef UPD_GO
}

// dense p x p copy of the sub-matrix a[i0 .. i0 + p)[j0 .. j0 + p) of an N x N coefficient matrix
__global__ void submatrix_kernel(int N, int p, int i0, int j0, const double2 *__restrict__ a, double2 *__restrict__ out, const int *done)
{
    if (done && *done) return;
    const int o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o < p * p) out[o] = a[(size_t)(i0 + o / p) * N + j0 + o % p];
}

int launch_block_update(bkr_ctx *ctx, int N, int precZ, int precW, const double2 *a, const void *C, const void *W, void *Z,
                        const int *done, int tri)
{
    if (N > 32) {
        // Blocks of 34..64 rhs (N even) as two panels of p = N / 2 columns: Z_J = C_J + W_0 a_0J + W_1 a_1J, one launch per
        // non-zero p x p block of the coefficient matrix (one level of the paper's recursive tiling; a
        // triangular a leaves three).  A panel is a contiguous view of the native block [rhs][colour][site].
        const int p = N / 2;
        const size_t L3 = (size_t)3 * ctx->g.Vh;
        const size_t cz = L3 * (precZ == BKR_F64 ? sizeof(double2) : sizeof(float2)), cw = L3 * (precW == BKR_F64 ? sizeof(double2) : sizeof(float2));
        if (!ctx->panel) BKR_CUDA(ctx, cudaMalloc((void **)&ctx->panel, (size_t)4 * 32 * 32 * sizeof(double2)));
        for (int J = 0; J < 2; J++) {
            bool first = true;
            for (int I = 0; I < 2; I++) {
                if ((tri == 1 && I > J) || (tri == 2 && I < J)) continue;
                double2 *sub = ctx->panel + (size_t)(2 * I + J) * 32 * 32;
                submatrix_kernel<<<(p * p + 127) / 128, 128, 0, ctx->stream>>>(N, p, I * p, J * p, a, sub, done);
                BKR_TRY(bkr_check_launch(ctx));
                char *zj = (char *)Z + (size_t)J * p * cz;
                const char *cj = first ? (C ? (const char *)C + (size_t)J * p * cz : nullptr) : (const char *)zj;
                BKR_TRY(launch_block_update(ctx, p, precZ, precW, sub, cj, (const char *)W + (size_t)I * p * cw, zj, done, I == J ? tri : 0));
                first = false;
            }
        }
        return BKR_OK;
    }
    if (precZ == BKR_F32 && precW == BKR_F32 && f32_tf32_update(ctx)) return launch_block_update_tf32(ctx, N, a, C, W, Z, done, tri);
    if (precZ == BKR_F64 && precW == BKR_F64) return launch_update_t<double, double>(ctx, N, a, C, W, Z, done, tri);
    if (precZ == BKR_F64 && precW == BKR_F32) return launch_update_t<double, float>(ctx, N, a, C, W, Z, done, tri);
    if (precZ == BKR_F32 && precW == BKR_F32) return launch_update_t<float, float>(ctx, N, a, C, W, Z, done, tri);
    // fp32 <- fp64: only Qhat = R C^-1 of the reliable update (Alg. 3 l.5), computed in fp64, rounded on store
    return launch_update_t<float, double>(ctx, N, a, C, W, Z, done, tri);
}

// ------------------------------------------------------------------------------------------ Gram, stage 1
// G = X^dag Y on 8 x 8 tiles of the N x N output, DMMA m8n8k4 over 4 rows at a time:
//   A[m][q] = X[8 ti + m][k + q] (8 x 4),  B[q][n] = Y[8 tj + n][k + q] (4 x 8), lane = 4 m + q reads one complex
//   of X (and of Y unless X == Y) from the ring with one 16-byte shared load, and
//   Re G += Xr Yr + Xi Yi     Im G += Xr Yi - Xi Yr      (four accumulators per tile pair, combined at the end).
// HERM: only pairs ti <= tj.  Otherwise blockIdx.y picks TIB i-tiles, all j-tiles.
// Chunk stride = 64 (mod 128) bytes for fp64 and 32 (mod 128) for fp32: conflict-free fragment loads.  Chunk slots of
// vectors >= N (padding of the last 8 x 8 tile) are never written by TMA; they are zeroed once, so no load in the loop
// is predicated.  Deterministic: fixed tile -> CTA -> warp assignment, fixed-order warp reduction through shared
// memory, one partial per CTA, fixed-order second stage.
template <typename Real, int NT, bool HERM, bool ALIAS, int TIB, int CW>
__global__ void __launch_bounds__((CW + 1) * 32, 1)
gram_tma_kernel(size_t L, int N, RingPlan rp, const typename CxT<Real>::type *__restrict__ X,
                const typename CxT<Real>::type *__restrict__ Y, double2 *__restrict__ partials, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int NXT = HERM ? NT : TIB;                    // i-tiles this CTA touches
    constexpr int NP = HERM ? NT * (NT + 1) / 2 : TIB * NT; // tile pairs this CTA accumulates
    extern __shared__ __align__(128) unsigned char dsm[];
    uint64_t *full = reinterpret_cast<uint64_t *>(dsm);
    uint64_t *empty = full + MB_MAX_STAGES;
    double2 *red = reinterpret_cast<double2 *>(dsm + 128); // [N * N]
    unsigned char *ring = dsm + rp.off_ring;
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ti0 = HERM ? 0 : blockIdx.y * TIB;
    const int i0 = 8 * ti0;                                  // first X vector of this CTA
    const int nxv = min(N - i0, 8 * NXT);                    // X vectors this CTA loads
    if (threadIdx.x == 0) {
        for (int s = 0; s < rp.nstg; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], CW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // zero the whole ring once (padding chunk slots stay zero; TMA overwrites the rest)
    {
        uint4 *z = reinterpret_cast<uint4 *>(ring);
        const size_t n16 = (size_t)rp.nstg * rp.stage_bytes / 16;
        for (size_t o = threadIdx.x; o < n16; o += blockDim.x) z[o] = make_uint4(0, 0, 0, 0);
    }
    for (int o = threadIdx.x; o < N * N; o += blockDim.x) red[o] = make_double2(0.0, 0.0);
    // generic-proxy writes (the zeroing) before async-proxy writes (TMA) to the same shared memory
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
            if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)(nxv + (ALIAS ? 0 : N)) * rows * (uint32_t)sizeof(Cx));
            __syncwarp();
            if (lane < nxv)
                tma_load_1d_hint(st + (size_t)lane * rp.rs_a, X + (size_t)(i0 + lane) * L + r0, rows * (uint32_t)sizeof(Cx), &full[s], pol);
            if (!ALIAS && lane < N)
                tma_load_1d_hint(st + rp.off_b + (size_t)lane * rp.rs_b, Y + (size_t)lane * L + r0, rows * (uint32_t)sizeof(Cx), &full[s], pol);
        }
        return;
    }

    // ---------------- consumers
    const int m = lane >> 2, q = lane & 3;
    double acc[NP][4][2]; // Xr Yr, Xr Yi, Xi Yr, Xi Yi: four independent DMMA chains per tile pair
#pragma unroll
    for (int p = 0; p < NP; p++)
#pragma unroll
        for (int c = 0; c < 4; c++) acc[p][c][0] = acc[p][c][1] = 0.0;

    for (int it = 0; it < my; it++) {
        const int s = it % rp.nstg;
        const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
        const int rows = (int)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
        const unsigned char *stX = ring + (size_t)s * rp.stage_bytes;
        const unsigned char *stY = ALIAS ? stX : stX + rp.off_b;
        const uint32_t rsy = ALIAS ? rp.rs_a : rp.rs_b;
        mbar_wait_acq(&full[s], (it / rp.nstg) & 1);
        // a k-step = 4 rows; two k-steps per iteration (fragments of both loaded before the first DMMA) so that the
        // shared-memory latency of one hides behind the tensor work of the other even with one warp per scheduler
        const int nks = rows / 4;
        for (int ks = warp; ks < nks; ks += 2 * CW) {
            const bool two = ks + CW < nks;
            double2 xf[2][NXT], yf[2][ALIAS ? 1 : NT];
#pragma unroll
            for (int h = 0; h < 2; h++) {
                const size_t ro = (size_t)(4 * (ks + (h && two ? CW : 0)) + q) * sizeof(Cx);
#pragma unroll
                for (int t = 0; t < NXT; t++) xf[h][t] = sm_cx<Cx>(stX + (size_t)(8 * t + m) * rp.rs_a + ro);
                if (!ALIAS) {
#pragma unroll
                    for (int t = 0; t < NT; t++) yf[h][t] = sm_cx<Cx>(stY + (size_t)(8 * t + m) * rsy + ro);
                }
            }
            if (!two) { // odd tail: the second k-step contributes nothing
#pragma unroll
                for (int t = 0; t < NXT; t++) xf[1][t] = make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int h = 0; h < 2; h++) {
                int p = 0;
#pragma unroll
                for (int ti = 0; ti < NXT; ti++) {
#pragma unroll
                    for (int tj = HERM ? ti : 0; tj < NT; tj++, p++) {
                        const double2 a = xf[h][ti];
                        const double2 b = ALIAS ? xf[h][tj] : yf[h][tj];
                        dmma(acc[p][0], a.x, b.x);
                        dmma(acc[p][1], a.x, b.y);
                        if (!(ALIAS && ti == tj)) dmma(acc[p][2], a.y, b.x); // diagonal tile of X^dag X: the transpose of [1]
                        dmma(acc[p][3], a.y, b.y);
                    }
                }
            }
        }
        // The stage goes back when its fragments have been consumed: the barrier address depends on every accumulator (all
        // of them took a DMMA from the last k-step), so the arrive cannot issue before those loads have returned
        // (dslash_win.cu has the story; a CTA-scope fence here cost 7 %).
        uint32_t dep = 0;
#pragma unroll
        for (int p = 0; p < NP; p++)
#pragma unroll
            for (int c = 0; c < 4; c++) dep |= (uint32_t)__double2loint(acc[p][c][0]) | (uint32_t)__double2loint(acc[p][c][1]);
        dep &= rp.zero;
        __syncwarp();
        if (lane == 0) mbar_arrive_rel(reinterpret_cast<uint64_t *>(reinterpret_cast<unsigned char *>(&empty[s]) + dep));
    }

    // fixed-order reduction over the consumer warps of the CTA, then one partial per CTA.  Named barrier 1 over the
    // consumer warps only (the producer warp has returned).
    for (int w = 0; w < CW; w++) {
        if (warp == w) {
            int p = 0;
#pragma unroll
            for (int ti = 0; ti < NXT; ti++) {
#pragma unroll
                for (int tj = HERM ? ti : 0; tj < NT; tj++, p++) {
                    if (ALIAS && ti == tj) frag_transpose(acc[p][1], acc[p][2], m, q);
#pragma unroll
                    for (int r = 0; r < 2; r++) {
                        const int i = 8 * (ti0 + ti) + m, j = 8 * tj + 2 * q + r;
                        if (i < N && j < N) {
                            double2 v = red[i * N + j];
                            v.x += acc[p][0][r] + acc[p][3][r];
                            v.y += acc[p][1][r] - acc[p][2][r];
                            red[i * N + j] = v;
                        }
                    }
                }
            }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(CW * 32) : "memory");
    }
    const int row0 = 8 * ti0, row1 = HERM ? N : min(N, 8 * (ti0 + TIB));
    for (int o = row0 * N + threadIdx.x; o < row1 * N; o += CW * 32)
        partials[(size_t)blockIdx.x * N * N + o] = red[o];
}

static const int GRAM_MAX_GRID = BKR_NUM_SMS;

template <typename Real, int NT>
static int gram_go(bkr_ctx *ctx, size_t L, int N, const void *X, const void *Y, int hermitian, int *num_partials, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int TIB = NT > 2 ? 2 : NT;
    constexpr int CW = NT > 2 ? 4 : 8; // above two tiles the accumulators need the 255-register budget of 160 threads
    const Cx *x = (const Cx *)X, *y = (const Cx *)Y;
    const bool alias = hermitian && X == Y;
    const int pad = sizeof(Real) == 8 ? 64 : 32;
    const size_t fixed = 128 + (size_t)N * N * sizeof(double2);
    const int nxs = hermitian ? 8 * NT : 8 * TIB; // X chunk slots (vectors >= N: zero padding)
    const RingPlan rp = plan_ring(L, fixed, 3, nxs, (int)sizeof(Cx), pad, alias ? 0 : 8 * NT, (int)sizeof(Cx), pad);
    if (rp.nstg < 2) return BKR_EINVAL;
    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const unsigned gx = (unsigned)(ntiles < (size_t)GRAM_MAX_GRID ? ntiles : (size_t)GRAM_MAX_GRID);
#define GRAM_LAUNCH(H_, A_, TIB_, GRID_)                                                                               \
    do {                                                                                                               \
        static int attr_dev = -1; /* per instantiation: the opt-in is per device */                                   \
        if (attr_dev != ctx->device) {                                                                                              \
            BKR_CUDA(ctx, cudaFuncSetAttribute(gram_tma_kernel<Real, NT, H_, A_, TIB_, CW>,                            \
                                               cudaFuncAttributeMaxDynamicSharedMemorySize, MB_SMEM_BUDGET));          \
            attr_dev = ctx->device;                                                                                          \
        }                                                                                                              \
        gram_tma_kernel<Real, NT, H_, A_, TIB_, CW><<<GRID_, (CW + 1) * 32, rp.smem, ctx->stream>>>(L, N, rp, x, y,     \
                                                                                                   ctx->partials, done); \
    } while (0)
    if (hermitian) {
        if (alias) GRAM_LAUNCH(true, true, NT, gx);
        else GRAM_LAUNCH(true, false, NT, gx);
    } else {
        dim3 g2(gx, (NT + TIB - 1) / TIB);
        GRAM_LAUNCH(false, false, TIB, g2);
    }
#undef GRAM_LAUNCH
    *num_partials = (int)gx;
    return bkr_check_launch(ctx);
}

int launch_gram_partials(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, int *num_partials,
                         const int *done)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    if (prec == BKR_F32 && f32_tf32_gram(ctx)) return launch_gram_partials_tf32(ctx, N, X, Y, hermitian, num_partials, done);
    BKR_TRY(ensure_partials(ctx, (size_t)2 * BKR_NUM_SMS * BKR_MAX_N * BKR_MAX_N * sizeof(double2)));
    const int NT = (N + 7) / 8;
#define GRAM_NT(Real)                                                                    \
    switch (NT) {                                                                        \
    case 1: return gram_go<Real, 1>(ctx, L, N, X, Y, hermitian, num_partials, done);     \
    case 2: return gram_go<Real, 2>(ctx, L, N, X, Y, hermitian, num_partials, done);     \
    case 3: return gram_go<Real, 3>(ctx, L, N, X, Y, hermitian, num_partials, done);     \
    default: return gram_go<Real, 4>(ctx, L, N, X, Y, hermitian, num_partials, done);    \
    }
    if (prec == BKR_F64) {
        GRAM_NT(double)
    }
    GRAM_NT(float)
#undef GRAM_NT
}

// ------------------------------------------------------------------------------------------ fused Q / P / X update
// Alg. 2 l.4 of the previous iteration, Alg. 1 l.8 of this one and l.10 of the previous one in one pass over Q', P, X
// (the deferral of PAPER.md:243):
//     Q   = Q' Si     if !flags->done   (Si = S^-1 upper triangular; in place)
//     Pn  = Q + P Sd  if !flags->done   (Sd = S^dag lower triangular)
//     X  += P Wm      if flags->xpend   (Wm = beta C of the previous l.9; X fp64, in place)
// 6 block passes.  Same ring, fragment layouts and DMMA tiles as update_tma_kernel; a stage holds R rows of Q' and P
// (A-fragment layout) and of X (accumulator layout).
template <typename RealP, int NTJ, int NIS, int CW>
__global__ void __launch_bounds__((CW + 1) * 32, 1)
pqx_update_kernel(size_t L, int N, Ring3 rp, const double2 *__restrict__ Si, const double2 *__restrict__ Sd,
                  const double2 *__restrict__ Wm,
                  typename CxT<RealP>::type *Q, const typename CxT<RealP>::type *__restrict__ P,
                  typename CxT<RealP>::type *__restrict__ Pn, double2 *X, const SolverFlags *fl)
{
    typedef typename CxT<RealP>::type CxP;
    constexpr int NF = NIS * NTJ * 32;
    extern __shared__ __align__(128) unsigned char dsm[];
    uint64_t *full = reinterpret_cast<uint64_t *>(dsm);
    uint64_t *empty = full + MB_MAX_STAGES;
    double *b1r = reinterpret_cast<double *>(dsm + 128), *b1i = b1r + NF, *b2r = b1i + NF, *b2i = b2r + NF, *b0r = b2i + NF,
           *b0i = b0r + NF;
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
    for (int idx = threadIdx.x; idx < NF; idx += blockDim.x) {
        const int ln = idx & 31, f = idx >> 5;
        const int is = f / NTJ, tj = f % NTJ;
        const int i = 4 * is + (ln & 3), j = 8 * tj + (ln >> 2);
        const bool in = i < N && j < N;
        const double2 v1 = in ? Sd[i * N + j] : make_double2(0.0, 0.0), v2 = in ? Wm[i * N + j] : make_double2(0.0, 0.0);
        const double2 v0 = in ? Si[i * N + j] : make_double2(0.0, 0.0);
        b0r[idx] = v0.x;
        b0i[idx] = v0.y;
        b1r[idx] = v1.x;
        b1i[idx] = v1.y;
        b2r[idx] = v2.x;
        b2i[idx] = v2.y;
    }
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
            if (lane == 0)
                mbar_expect_tx(&full[s], (uint32_t)N * rows *
                                             (uint32_t)(sizeof(CxP) + (doP ? sizeof(CxP) : 0) + (doX ? sizeof(double2) : 0)));
            __syncwarp();
            if (lane < N) {
                tma_load_1d_hint(st + (size_t)lane * rp.rs_p, P + (size_t)lane * L + r0, rows * (uint32_t)sizeof(CxP), &full[s], pol);
                if (doP)
                    tma_load_1d_hint(st + rp.off_q + (size_t)lane * rp.rs_q, Q + (size_t)lane * L + r0,
                                     rows * (uint32_t)sizeof(CxP), &full[s], pol);
                if (doX)
                    tma_load_1d_hint(st + rp.off_x + (size_t)lane * rp.rs_x, X + (size_t)lane * L + r0,
                                     rows * (uint32_t)sizeof(double2), &full[s], pol);
            }
        }
        return;
    }

    // ---------------- consumers
    const int m = lane >> 2, q = lane & 3;
    for (int it = 0; it < my; it++) {
        const int s = it % rp.nstg;
        const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
        const int rows = (int)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
        const unsigned char *stP = ring + (size_t)s * rp.stage_bytes;
        const unsigned char *stQ = stP + rp.off_q, *stX = stP + rp.off_x;
        mbar_wait_acq(&full[s], (it / rp.nstg) & 1);
        for (int u = warp; u < rows / 8; u += CW) {
            const int row = 8 * u + m;
            double2 wf[NIS];
#pragma unroll
            for (int is = 0; is < NIS; is++) {
                const int i = 4 * is + q;
                wf[is] = i < N ? sm_cx<CxP>(stP + (size_t)i * rp.rs_p + (size_t)row * sizeof(CxP)) : make_double2(0.0, 0.0);
            }
            if (doP) {
                // Qn = Q' Si (Si = S^-1 upper triangular: fragments with 4 is > 8 tj + 7 are zero and skipped), then
                // Pn = Qn + P Sd (Sd = S^dag lower triangular: fragments with 4 is + 3 < 8 tj skipped)
                double2 wq[NIS];
#pragma unroll
                for (int is = 0; is < NIS; is++) {
                    const int i = 4 * is + q;
                    wq[is] = i < N ? sm_cx<CxP>(stQ + (size_t)i * rp.rs_q + (size_t)row * sizeof(CxP)) : make_double2(0.0, 0.0);
                }
                double zre[NTJ][2], zim[NTJ][2];
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++) zre[tj][0] = zre[tj][1] = zim[tj][0] = zim[tj][1] = 0.0;
#pragma unroll
                for (int is = 0; is < NIS; is++)
#pragma unroll
                    for (int tj = 0; tj < NTJ; tj++) {
                        if (4 * is <= 8 * tj + 7) {
                            const int f = (is * NTJ + tj) * 32 + lane;
                            const double br = b0r[f], bi = b0i[f];
                            dmma(zre[tj], wq[is].x, br);
                            dmma(zre[tj], wq[is].y, -bi);
                            dmma(zim[tj], wq[is].x, bi);
                            dmma(zim[tj], wq[is].y, br);
                        }
                    }
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++)
#pragma unroll
                    for (int r = 0; r < 2; r++) {
                        const int j = 8 * tj + 2 * q + r;
                        if (j < N) st_cx<CxP>(Q + (size_t)j * L + r0 + row, zre[tj][r], zim[tj][r]);
                    }
#pragma unroll
                for (int is = 0; is < NIS; is++)
#pragma unroll
                    for (int tj = 0; tj < NTJ; tj++) {
                        if (4 * is + 3 >= 8 * tj) {
                            const int f = (is * NTJ + tj) * 32 + lane;
                            const double br = b1r[f], bi = b1i[f];
                            dmma(zre[tj], wf[is].x, br);
                            dmma(zre[tj], wf[is].y, -bi);
                            dmma(zim[tj], wf[is].x, bi);
                            dmma(zim[tj], wf[is].y, br);
                        }
                    }
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++)
#pragma unroll
                    for (int r = 0; r < 2; r++) {
                        const int j = 8 * tj + 2 * q + r;
                        if (j < N) st_cx<CxP>(Pn + (size_t)j * L + r0 + row, zre[tj][r], zim[tj][r]);
                    }
            }
            if (doX) {
                double zre[NTJ][2], zim[NTJ][2];
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++) zre[tj][0] = zre[tj][1] = zim[tj][0] = zim[tj][1] = 0.0;
#pragma unroll
                for (int is = 0; is < NIS; is++)
#pragma unroll
                    for (int tj = 0; tj < NTJ; tj++) {
                        const int f = (is * NTJ + tj) * 32 + lane;
                        const double br = b2r[f], bi = b2i[f];
                        dmma(zre[tj], wf[is].x, br);
                        dmma(zre[tj], wf[is].y, -bi);
                        dmma(zim[tj], wf[is].x, bi);
                        dmma(zim[tj], wf[is].y, br);
                    }
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++)
#pragma unroll
                    for (int r = 0; r < 2; r++) {
                        const int j = 8 * tj + 2 * q + r;
                        if (j < N) {
                            const double2 c = sm_cx<double2>(stX + (size_t)j * rp.rs_x + (size_t)row * sizeof(double2));
                            st_cx<double2>(X + (size_t)j * L + r0 + row, zre[tj][r] + c.x, zim[tj][r] + c.y);
                        }
                    }
            }
        }
        // (the stores above take their data from everything the stage was loaded for: a release cannot move above them,
        // so the loads have returned -- no fence needed here, dslash_win.cu has the story)
        __syncwarp();
        if (lane == 0) mbar_arrive_rel(&empty[s]);
    }
}

template <typename RealP, int NTJ, int NIS>
static int pqx_go(bkr_ctx *ctx, size_t L, int N, const double2 *Si, const double2 *Sd, const double2 *Wm, void *Q, const void *P, void *Pn,
                 double2 *X, const SolverFlags *fl)
{
    typedef typename CxT<RealP>::type CxP;
    // 9 warps get the register budget of 12 (168 per thread); with 4 column tiles the fragments and accumulators need more:
    // 7 consumer warps + the producer = 8 warps = 255 registers per thread, no spills (32^4, N = 32: 1.50 -> 1.25 ms; with
    // 3 tiles nothing spills at 168 and 8 warps are faster: 0.78 against 0.79 ms at N = 24)
    constexpr int CW = NTJ >= 4 ? 7 : 8;
    const size_t fixed = (128 + (size_t)6 * NIS * NTJ * 32 * sizeof(double) + 127) / 128 * 128;
    const Ring3 rp = plan_ring3(L, N, fixed, (int)sizeof(CxP));
    if (rp.nstg < 2) return BKR_EINVAL;
    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const unsigned grid = (unsigned)(ntiles < (size_t)BKR_NUM_SMS ? ntiles : (size_t)BKR_NUM_SMS);
    static int attr_dev = -1; // per instantiation: the opt-in is per device
    if (attr_dev != ctx->device) {
        BKR_CUDA(ctx, cudaFuncSetAttribute(pqx_update_kernel<RealP, NTJ, NIS, CW>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           MB_SMEM_BUDGET));
        attr_dev = ctx->device;
    }
    pqx_update_kernel<RealP, NTJ, NIS, CW><<<grid, (CW + 1) * 32, rp.smem, ctx->stream>>>(
        L, N, rp, Si, Sd, Wm, (CxP *)Q, (const CxP *)P, (CxP *)Pn, X, fl);
    return bkr_check_launch(ctx);
}

template <typename RealP>
static int launch_pqx_t(bkr_ctx *ctx, int N, const double2 *Si, const double2 *Sd, const double2 *Wm, void *Q, const void *P, void *Pn,
                       double2 *X, const SolverFlags *fl)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
#define PQX_GO(NTJ_, NIS_) return pqx_go<RealP, NTJ_, NIS_>(ctx, L, N, Si, Sd, Wm, Q, P, Pn, X, fl)
    switch ((N + 3) / 4) {
    case 1: PQX_GO(1, 1);
    case 2: PQX_GO(1, 2);
    case 3: PQX_GO(2, 3);
    case 4: PQX_GO(2, 4);
    case 5: PQX_GO(3, 5);
    case 6: PQX_GO(3, 6);
    case 7: PQX_GO(4, 7);
    default: PQX_GO(4, 8);
    }
#undef PQX_GO
}


int launch_pqx_update(bkr_ctx *ctx, int N, int prec, const double2 *Sinv, const double2 *Sdag, const double2 *Wm, void *Q,
                      const void *P, void *Pn, double2 *X, const SolverFlags *flags)
{
    if (prec == BKR_F64) return launch_pqx_t<double>(ctx, N, Sinv, Sdag, Wm, Q, P, Pn, X, flags);
    if (N <= 16 && f32_tf32_update(ctx)) return launch_pqx_update_tf32(ctx, N, Sinv, Sdag, Wm, Q, P, Pn, X, flags);
    return launch_pqx_t<float>(ctx, N, Sinv, Sdag, Wm, Q, P, Pn, X, flags);
}

// ------------------------------------------------------------------------------------------ fused update + aliased Gram
// Alg. 1 l.11 / Alg. 2 l.2 in one pass:  Z = C + W a  (Q' = Q - MP beta)  and  H = Z^dag Z  (Hermitian, upper
// tile pairs).  The update part is update_tma_kernel's; each warp then writes its 8 finished rows of Z -- rounded to the
// storage precision, so that H is the Gram matrix of what is stored -- over the C rows it has just consumed in the ring
// and feeds them back as DMMA fragments of the reduction (gram_tma_kernel's tiles, accumulators and fixed-order
// two-stage reduction).  Saves the separate read of Z.
template <typename Real, int NT, int NIS, int CW>
__global__ void __launch_bounds__((CW + 1) * 32, 1)
update_gram_kernel(size_t L, int N, RingPlan rp, uint32_t off_red, const double2 *__restrict__ a,
                   const typename CxT<Real>::type *C, const typename CxT<Real>::type *__restrict__ W,
                   typename CxT<Real>::type *Z, double2 *__restrict__ partials, const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int NTJ = NT;
    constexpr int NF = NIS * NTJ * 32;
    constexpr int NP = NT * (NT + 1) / 2;
    extern __shared__ __align__(128) unsigned char dsm[];
    uint64_t *full = reinterpret_cast<uint64_t *>(dsm);
    uint64_t *empty = full + MB_MAX_STAGES;
    double *bre = reinterpret_cast<double *>(dsm + 128), *bim = bre + NF;
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
    for (int idx = threadIdx.x; idx < NF; idx += blockDim.x) {
        const int ln = idx & 31, f = idx >> 5;
        const int is = f / NTJ, tj = f % NTJ;
        const int i = 4 * is + (ln & 3), j = 8 * tj + (ln >> 2);
        const double2 v = (i < N && j < N) ? a[i * N + j] : make_double2(0.0, 0.0);
        bre[idx] = v.x;
        bim[idx] = v.y;
    }
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
            if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)N * rows * 2u * (uint32_t)sizeof(Cx));
            __syncwarp();
            if (lane < N) {
                tma_load_1d_hint(st + (size_t)lane * rp.rs_a, W + (size_t)lane * L + r0, rows * (uint32_t)sizeof(Cx), &full[s], pol);
                tma_load_1d_hint(st + rp.off_b + (size_t)lane * rp.rs_b, C + (size_t)lane * L + r0, rows * (uint32_t)sizeof(Cx),
                                 &full[s], pol);
            }
        }
        return;
    }

    // ---------------- consumers
    const int m = lane >> 2, q = lane & 3;
    double acc[NP][4][2]; // Zr Zr, Zr Zi, Zi Zr, Zi Zi per tile pair
#pragma unroll
    for (int p = 0; p < NP; p++)
#pragma unroll
        for (int c = 0; c < 4; c++) acc[p][c][0] = acc[p][c][1] = 0.0;
    for (int it = 0; it < my; it++) {
        const int s = it % rp.nstg;
        const size_t r0 = ((size_t)blockIdx.x + (size_t)it * gridDim.x) * rp.R;
        const int rows = (int)((L - r0 < (size_t)rp.R) ? L - r0 : rp.R);
        const unsigned char *stW = ring + (size_t)s * rp.stage_bytes;
        unsigned char *stC = ring + (size_t)s * rp.stage_bytes + rp.off_b;
        mbar_wait_acq(&full[s], (it / rp.nstg) & 1);
        for (int u = warp; u < rows / 8; u += CW) {
            const int row = 8 * u + m;
            double2 wf[NIS];
#pragma unroll
            for (int is = 0; is < NIS; is++) {
                const int i = 4 * is + q;
                wf[is] = i < N ? sm_cx<Cx>(stW + (size_t)i * rp.rs_a + (size_t)row * sizeof(Cx)) : make_double2(0.0, 0.0);
            }
            double zre[NTJ][2], zim[NTJ][2];
#pragma unroll
            for (int tj = 0; tj < NTJ; tj++) zre[tj][0] = zre[tj][1] = zim[tj][0] = zim[tj][1] = 0.0;
#pragma unroll
            for (int is = 0; is < NIS; is++)
#pragma unroll
                for (int tj = 0; tj < NTJ; tj++) {
                    const int f = (is * NTJ + tj) * 32 + lane;
                    const double br = bre[f], bi = bim[f];
                    dmma(zre[tj], wf[is].x, br);
                    dmma(zre[tj], wf[is].y, -bi);
                    dmma(zim[tj], wf[is].x, bi);
                    dmma(zim[tj], wf[is].y, br);
                }
#pragma unroll
            for (int tj = 0; tj < NTJ; tj++)
#pragma unroll
                for (int r = 0; r < 2; r++) {
                    const int j = 8 * tj + 2 * q + r;
                    if (j < N) {
                        Cx *cp = reinterpret_cast<Cx *>(stC + (size_t)j * rp.rs_b + (size_t)row * sizeof(Cx));
                        const Cx c = *cp;
                        Cx zv; // rounded to the storage precision: H is the Gram matrix of what is stored
                        zv.x = (Real)(zre[tj][r] + (double)c.x);
                        zv.y = (Real)(zim[tj][r] + (double)c.y);
                        *cp = zv;
                        __stcs(Z + (size_t)j * L + r0 + row, zv);
                    }
                }
            __syncwarp();
#pragma unroll
            for (int h = 0; h < 2; h++) {
                double2 xf[NT];
#pragma unroll
                for (int t = 0; t < NT; t++)
                    xf[t] = (8 * t + m) < N
                                ? sm_cx<Cx>(stC + (size_t)(8 * t + m) * rp.rs_b + (size_t)(8 * u + 4 * h + q) * sizeof(Cx))
                                : make_double2(0.0, 0.0);
                int p = 0;
#pragma unroll
                for (int ti = 0; ti < NT; ti++)
#pragma unroll
                    for (int tj = ti; tj < NT; tj++, p++) {
                        dmma(acc[p][0], xf[ti].x, xf[tj].x);
                        dmma(acc[p][1], xf[ti].x, xf[tj].y);
                        if (ti != tj) dmma(acc[p][2], xf[ti].y, xf[tj].x); // diagonal tile: the transpose of [1] (frag_transpose)
                        dmma(acc[p][3], xf[ti].y, xf[tj].y);
                    }
            }
        }
        // generic-proxy writes to the stage before the async-proxy (TMA) refill of the same shared memory
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        // (the stores above take their data from everything the stage was loaded for: a release cannot move above them,
        // so the loads have returned -- no fence needed here, dslash_win.cu has the story)
        __syncwarp();
        if (lane == 0) mbar_arrive_rel(&empty[s]);
    }
    for (int w = 0; w < CW; w++) { // fixed-order reduction over the consumer warps (named barrier 1: the producer has left)
        if (warp == w) {
            int p = 0;
#pragma unroll
            for (int ti = 0; ti < NT; ti++)
#pragma unroll
                for (int tj = ti; tj < NT; tj++, p++) {
                    if (ti == tj) frag_transpose(acc[p][1], acc[p][2], m, q);
#pragma unroll
                    for (int r = 0; r < 2; r++) {
                        const int i = 8 * ti + m, j = 8 * tj + 2 * q + r;
                        if (i < N && j < N) {
                            double2 v = red[i * N + j];
                            v.x += acc[p][0][r] + acc[p][3][r];
                            v.y += acc[p][1][r] - acc[p][2][r];
                            red[i * N + j] = v;
                        }
                    }
                }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(CW * 32) : "memory");
    }
    for (int o = threadIdx.x; o < N * N; o += CW * 32) partials[(size_t)blockIdx.x * N * N + o] = red[o];
}

template <typename Real, int NT, int NIS>
static int update_gram_go(bkr_ctx *ctx, size_t L, int N, const double2 *a, const void *C, const void *W, void *Z, int *num_partials,
                          const int *done)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int CW = 8; // (7 warps at 255 registers end the spills of the 3-4 tile instances but are slower: 0.65 / 1.12 ms
                          // against 0.55 / 0.83 ms at N = 24 / 32 on 32^4; the solver fuses this pair only up to 16 rhs)
    const size_t off_red = (128 + (size_t)2 * NIS * NT * 32 * sizeof(double) + 127) / 128 * 128;
    const size_t fixed = off_red + (size_t)N * N * sizeof(double2);
    const RingPlan rp = plan_ring(L, fixed, 4, N, (int)sizeof(Cx), 32, N, (int)sizeof(Cx), 16);
    if (rp.nstg < 2) return BKR_EINVAL;
    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const unsigned grid = (unsigned)(ntiles < (size_t)BKR_NUM_SMS ? ntiles : (size_t)BKR_NUM_SMS);
    BKR_TRY(ensure_partials(ctx, (size_t)2 * BKR_NUM_SMS * BKR_MAX_N * BKR_MAX_N * sizeof(double2)));
    static int attr_dev = -1; // per instantiation: the opt-in is per device
    if (attr_dev != ctx->device) {
        BKR_CUDA(ctx, cudaFuncSetAttribute(update_gram_kernel<Real, NT, NIS, CW>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           MB_SMEM_BUDGET));
        attr_dev = ctx->device;
    }
    update_gram_kernel<Real, NT, NIS, CW><<<grid, (CW + 1) * 32, rp.smem, ctx->stream>>>(
        L, N, rp, (uint32_t)off_red, a, (const Cx *)C, (const Cx *)W, (Cx *)Z, ctx->partials, done);
    *num_partials = (int)grid;
    return bkr_check_launch(ctx);
}

// Z = C + W a (Z may alias C) and per-CTA partials of the Hermitian Gram matrix Z^dag Z in ctx->partials (second stage:
// small_kernel or launch_gram_finish, as after launch_gram_partials).  All blocks in precision prec.
int launch_update_gram(bkr_ctx *ctx, int N, int prec, const double2 *a, const void *C, const void *W, void *Z, int *num_partials,
                       const int *done)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    if (prec == BKR_F32 && N <= 16 && f32_tf32_update(ctx)) return launch_update_gram_tf32(ctx, N, a, C, W, Z, num_partials, done);
#define UG_GO(Real, NT_, NIS_) return update_gram_go<Real, NT_, NIS_>(ctx, L, N, a, C, W, Z, num_partials, done)
#define UG_SW(Real)                  \
    switch ((N + 3) / 4) {           \
    case 1: UG_GO(Real, 1, 1);       \
    case 2: UG_GO(Real, 1, 2);       \
    case 3: UG_GO(Real, 2, 3);       \
    case 4: UG_GO(Real, 2, 4);       \
    case 5: UG_GO(Real, 3, 5);       \
    case 6: UG_GO(Real, 3, 6);       \
    case 7: UG_GO(Real, 4, 7);       \
    default: UG_GO(Real, 4, 8);      \
    }
    if (prec == BKR_F64) {
        UG_SW(double)
    }
    UG_SW(float)
#undef UG_SW
#undef UG_GO
}

// ------------------------------------------------------------------------------------------ Gram without allocation
// bkr_gram_static (bkr.h): K = X^dag Y with the per-CTA partials of stage 1 in a file-scope device array instead of
// ctx->partials, for callers that must not reach cudaMalloc (stream capture, serving loops).  Same kernels, same tile ->
// CTA -> warp assignment and the same fixed-order second stage as launch_gram_partials + launch_gram_finish on the FP64
// tensor path, so the result is bit-identical to bkr_gram's default path.
//  * Capacity: one partial per SM for blocks of up to BKR_STATIC_MAX_N = 32 rhs: 148 x 32 x 32 x 16 B = 2.3 MB, held by
//    every GPU that loads the library until the process exits.
//  * The array is shared by all contexts and streams of a device and keeps the last call's contents.  Nothing in it has
//    to start at zero: stage 1 writes every entry stage 2 reads (each CTA stores its whole N x N partial, or its rows
//    of it when the block is split over blockIdx.y), so there is no clearing pass.  Two calls that overlap on the GPU
//    (different streams, or two contexts on one device) race on it: callers serialise.
//  * In host code `gram_static_scratch` is a host-side stand-in, not a device address; the kernels get the address
//    cudaGetSymbolAddress returns, looked up once per device with that device current.
static __device__ __align__(256) double2 gram_static_scratch[(size_t)BKR_NUM_SMS * BKR_STATIC_MAX_N * BKR_STATIC_MAX_N];

static const int STATIC_MAX_DEVICES = 64;
static double2 *gram_static_ptr[STATIC_MAX_DEVICES]; // device address of the array on each device (0 = not looked up)

static int gram_static_address(bkr_ctx *ctx, double2 **ptr)
{
    if (ctx->device < 0 || ctx->device >= STATIC_MAX_DEVICES) return BKR_EINVAL;
    if (!gram_static_ptr[ctx->device]) { // the caller (BKR_ENTER) has made ctx->device current
        double2 *p = nullptr;
        BKR_CUDA(ctx, cudaGetSymbolAddress((void **)&p, gram_static_scratch));
        gram_static_ptr[ctx->device] = p;
    }
    *ptr = gram_static_ptr[ctx->device];
    return BKR_OK;
}

// stage 2 (gram_finish_kernel of blas.cu on an explicit partials pointer: same order of summation)
__global__ void __launch_bounds__(128)
gram_static_finish_kernel(int N, int num_partials, int hermitian, const double2 *__restrict__ partials, double2 *__restrict__ K)
{
    const int w = (blockIdx.x * 128 + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 1, o = 2 * w + (lane & 1);
    const bool act = o < N * N;
    const int i = act ? o / N : 0, j = act ? o % N : 0;
    const bool lower = hermitian && i > j;
    const int src = lower ? j * N + i : i * N + j;
    double2 s = sum_partials_16(partials + src, (size_t)N * N, num_partials, g, act);
    if (act && g == 0) {
        if (lower) s.y = -s.y;
        if (hermitian && i == j) s.y = 0.0;
        K[o] = s;
    }
}

template <typename Real, int NT>
static int gram_static_go(bkr_ctx *ctx, size_t L, int N, const void *X, const void *Y, int hermitian, double2 *scratch, double2 *K)
{
    typedef typename CxT<Real>::type Cx;
    constexpr int TIB = NT > 2 ? 2 : NT; // the launch geometry of gram_go
    constexpr int CW = NT > 2 ? 4 : 8;
    const Cx *x = (const Cx *)X, *y = (const Cx *)Y;
    const bool alias = hermitian && X == Y;
    const int pad = sizeof(Real) == 8 ? 64 : 32;
    const size_t fixed = 128 + (size_t)N * N * sizeof(double2);
    const int nxs = hermitian ? 8 * NT : 8 * TIB;
    const RingPlan rp = plan_ring(L, fixed, 3, nxs, (int)sizeof(Cx), pad, alias ? 0 : 8 * NT, (int)sizeof(Cx), pad);
    if (rp.nstg < 2) return BKR_EINVAL;
    const size_t ntiles = (L + rp.R - 1) / rp.R;
    const unsigned gx = (unsigned)(ntiles < (size_t)GRAM_MAX_GRID ? ntiles : (size_t)GRAM_MAX_GRID);
#define GRAM_STATIC_LAUNCH(H_, A_, TIB_, GRID_)                                                                        \
    do {                                                                                                               \
        static int attr_dev = -1; /* cudaFuncSetAttribute allocates nothing */                                         \
        if (attr_dev != ctx->device) {                                                                                 \
            BKR_CUDA(ctx, cudaFuncSetAttribute(gram_tma_kernel<Real, NT, H_, A_, TIB_, CW>,                            \
                                               cudaFuncAttributeMaxDynamicSharedMemorySize, MB_SMEM_BUDGET));          \
            attr_dev = ctx->device;                                                                                    \
        }                                                                                                              \
        gram_tma_kernel<Real, NT, H_, A_, TIB_, CW><<<GRID_, (CW + 1) * 32, rp.smem, ctx->stream>>>(L, N, rp, x, y,     \
                                                                                                   scratch, nullptr);  \
    } while (0)
    if (hermitian) {
        if (alias) GRAM_STATIC_LAUNCH(true, true, NT, gx);
        else GRAM_STATIC_LAUNCH(true, false, NT, gx);
    } else {
        dim3 g2(gx, (NT + TIB - 1) / TIB);
        GRAM_STATIC_LAUNCH(false, false, TIB, g2);
    }
#undef GRAM_STATIC_LAUNCH
    BKR_TRY(bkr_check_launch(ctx));
    gram_static_finish_kernel<<<(N * N * 16 + 127) / 128, 128, 0, ctx->stream>>>(N, (int)gx, hermitian, scratch, K);
    return bkr_check_launch(ctx);
}

// N <= BKR_STATIC_MAX_N (checked by the caller, bkr_gram_static); no cudaMalloc / cudaFree on this path
int launch_gram_static(bkr_ctx *ctx, int N, int prec, const void *X, const void *Y, int hermitian, double2 *K)
{
    const size_t L = (size_t)ctx->g.Vh * 3;
    double2 *scratch = nullptr;
    BKR_TRY(gram_static_address(ctx, &scratch));
#define GRAM_STATIC_NT(Real)                                                                 \
    switch ((N + 7) / 8) {                                                                   \
    case 1: return gram_static_go<Real, 1>(ctx, L, N, X, Y, hermitian, scratch, K);          \
    case 2: return gram_static_go<Real, 2>(ctx, L, N, X, Y, hermitian, scratch, K);          \
    case 3: return gram_static_go<Real, 3>(ctx, L, N, X, Y, hermitian, scratch, K);          \
    default: return gram_static_go<Real, 4>(ctx, L, N, X, Y, hermitian, scratch, K);         \
    }
    if (prec == BKR_F64) {
        GRAM_STATIC_NT(double)
    }
    GRAM_STATIC_NT(float)
#undef GRAM_STATIC_NT
}
