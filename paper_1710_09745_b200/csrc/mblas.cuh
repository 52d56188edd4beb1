// Pieces shared by the multi-BLAS kernel files (mblas.cu: FP64 tensor path; mblas_tf32.cu: split-TF32 path for fp32
// blocks): ring geometry, barrier helpers, shared-memory / store helpers.
#pragma once
#include "common.cuh"
#include "tma.cuh"

#include <stdlib.h>
#include <string.h>

static const int MB_SMEM_BUDGET = 216 * 1024; // of the 227 KB a CTA may opt in to
static const int MB_MAX_STAGES = 8;

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1])
        : "d"(a), "d"(b));
}

// mbarrier wait that is also a compiler barrier for memory: the plain shared-memory reads of a stage must not move
// above it
__device__ __forceinline__ void mbar_wait_acq(uint64_t *bar, uint32_t parity)
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
__device__ __forceinline__ void mbar_arrive_rel(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}

template <typename Cx> __device__ __forceinline__ double2 sm_cx(const unsigned char *p)
{
    const Cx v = *reinterpret_cast<const Cx *>(p);
    return make_double2((double)v.x, (double)v.y);
}
template <typename Cx> __device__ __forceinline__ void st_cx(Cx *p, double re, double im);
template <> __device__ __forceinline__ void st_cx<double2>(double2 *p, double re, double im)
{
    __stcs(p, make_double2(re, im));
}
template <> __device__ __forceinline__ void st_cx<float2>(float2 *p, double re, double im)
{
    __stcs(p, make_float2((float)re, (float)im));
}

// Ring geometry shared by host and device.  A stage holds `nchunk_a` chunks of stride rs_a and `nchunk_b` chunks of
// stride rs_b (bytes); a chunk is R consecutive rows of one vector.
struct RingPlan {
    int R, nstg;
    uint32_t rs_a, rs_b, off_b, stage_bytes, off_ring; // off_ring: start of the ring in dynamic shared memory
    size_t smem;
    uint32_t zero; // 0 at run time, unknown to the compiler (ties a barrier arrival to registers, gram_tma_kernel)
};

// pad: the residue (mod 128 bytes) the chunk stride must have so that fragment loads are conflict-free
// Policy (measured, 32^4): a stage costs ~600 cycles of fixed overhead plus ~40 per bulk copy,
// so R is the largest power of two that still leaves `min_stages` stages in the ring (3 for the reductions, 4 for the
// updates, whose consumers also write) and gives every SM at least two row tiles.
static inline RingPlan plan_ring(size_t L, size_t fixed, int min_stages, int nchunk_a, int esize_a, int pad_a, int nchunk_b,
                          int esize_b, int pad_b)
{
    RingPlan best;
    memset(&best, 0, sizeof(best));
    fixed = (fixed + 127) / 128 * 128;
    for (int R = 1024; R >= 64; R /= 2) {
        RingPlan p;
        p.zero = 0;
        p.R = R;
        p.rs_a = (uint32_t)(R * esize_a + pad_a);
        p.rs_b = (uint32_t)(R * esize_b + pad_b);
        p.off_b = ((uint32_t)nchunk_a * p.rs_a + 127) / 128 * 128;
        p.stage_bytes = (p.off_b + (uint32_t)nchunk_b * p.rs_b + 127) / 128 * 128;
        p.off_ring = (uint32_t)fixed;
        int n = (int)((MB_SMEM_BUDGET - fixed) / p.stage_bytes);
        if (n > MB_MAX_STAGES) n = MB_MAX_STAGES;
        p.nstg = n;
        p.smem = fixed + (size_t)n * p.stage_bytes;
        bool ok = n >= min_stages && (L + R - 1) / R >= (size_t)2 * BKR_NUM_SMS;
        if (ok || R == 64) {
            if (n < 2) p.nstg = 0; // does not fit at all (cannot happen for N <= 32)
            best = p;
            break;
        }
    }
    return best;
}

struct Ring3 {
    int R, nstg;
    uint32_t rs_p, rs_q, rs_x, off_q, off_x, stage_bytes, off_ring;
    size_t smem;
};

// ring of the fused Q / P / X update: R rows of P and Q' (A-fragment layout, element size esize_p) and of X (fp64,
// accumulator layout); `fixed` = bytes in front of the ring
static inline Ring3 plan_ring3(size_t L, int N, size_t fixed, int esize_p)
{
    Ring3 rp;
    memset(&rp, 0, sizeof(rp));
    for (int R = 512; R >= 32; R /= 2) {
        rp.R = R;
        rp.rs_p = (uint32_t)(R * esize_p + 32);
        rp.rs_q = (uint32_t)(R * esize_p + 32); // Q' is an A operand here
        rp.rs_x = (uint32_t)(R * sizeof(double2) + 16);
        rp.off_q = ((uint32_t)N * rp.rs_p + 127) / 128 * 128;
        rp.off_x = (rp.off_q + (uint32_t)N * rp.rs_q + 127) / 128 * 128;
        rp.stage_bytes = (rp.off_x + (uint32_t)N * rp.rs_x + 127) / 128 * 128;
        rp.off_ring = (uint32_t)fixed;
        int n = (int)((MB_SMEM_BUDGET - fixed) / rp.stage_bytes);
        if (n > MB_MAX_STAGES) n = MB_MAX_STAGES;
        rp.nstg = n;
        rp.smem = fixed + (size_t)n * rp.stage_bytes;
        if ((n >= 4 && (L + R - 1) / R >= (size_t)2 * BKR_NUM_SMS) || R == 32) break;
    }
    return rp;
}

// fp32 blocks: FP64 DMMA path of mblas.cu (default) or the split-TF32 tensor path of mblas_tf32.cu.  BKR_TUNE_F32_MATH:
// 0 = FP64 DMMA (products of fp32 numbers exact, every sum fp64, one rounding on store), 1 = split-TF32 wherever it exists,
// 2 = split-TF32 updates only, 3 = split-TF32 reductions only.  TF32 is faster per call (32^4, N = 16: update 0.168 -> 0.117 ms,
// fused update + Gram 0.227 -> 0.184, Gram 0.108 -> 0.098) but its ~3e-7 errors cost the fp32-inner blockCGrQ 25-30 %
// more iterations at config 3, tol 1e-10 (529 -> 663-686 with either the updates or the reductions on TF32), so the solver
// stays on FP64 tensor products.
static inline bool f32_tf32_update(const bkr_ctx *ctx) { const int m = ctx->tune[BKR_TUNE_F32_MATH]; return m == 1 || m == 2; }
static inline bool f32_tf32_gram(const bkr_ctx *ctx) { const int m = ctx->tune[BKR_TUNE_F32_MATH]; return m == 1 || m == 3; }
int launch_block_update_tf32(bkr_ctx *ctx, int N, const double2 *a, const void *C, const void *W, void *Z, const int *done, int tri);
int launch_gram_partials_tf32(bkr_ctx *ctx, int N, const void *X, const void *Y, int hermitian, int *num_partials, const int *done);
int launch_pqx_update_tf32(bkr_ctx *ctx, int N, const double2 *Sinv, const double2 *Sdag, const double2 *Wm, void *Q, const void *P, void *Pn,
                           double2 *X, const SolverFlags *flags);
int launch_update_gram_tf32(bkr_ctx *ctx, int N, const double2 *a, const void *C, const void *W, void *Z, int *num_partials, const int *done);
