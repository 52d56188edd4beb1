// Small dense N x N algebra on the device (PAPER.md:178 does it on the host with Eigen; north_star moves it
// into a device-side kernel so that no Gram matrix or coefficient matrix ever crosses to the host).
//
// One CTA.  All threads: the deterministic second stage of the Gram reduction (fixed-order sum of the per-CTA
// partials, Hermitised from the upper triangle) and the N x N products.  Warp 0 alone: the
// Cholesky factorisation H = R^dag R (Algorithm 2 l.3) and the triangular inverse, matrices in shared memory.
//
// Modes (Algorithm 1 / 2 / 3 line numbers as reconstructed in DESIGN.md U7):
//   SMALL_CHOL    API: R = chol(in), Rinv
//   SMALL_HPDINV  API: out0 = in^-1
//   SMALL_BETA    l.9/l.10: G = sum partials; beta = G^-1; negbeta = -beta; W = beta C
//   SMALL_QR      l.11/l.12: H = sum partials; S = chol(H); Sinv; Sdag; Cprev = C; C = S C; residuals, flags
//   SMALL_INIT    l.4-l.5:  H = sum partials; C = chol(H); Sinv = C^-1 (to form Q = R C^-1); Sdag = 1
//   SMALL_RELUPD  Alg. 3 l.5-l.6: C_new = chol(H); Sinv = C_new^-1; Sdag = (C_new Cprev^-1)^dag; C = C_new
//   SMALL_RQ1     two-pass QR of an ill-conditioned residual block (refs [43, 44] of PAPER.md:184-186), pass 1:
//                 H = sum partials; R1 = chol(H + 1e-12 max_i H_ii); W = R1 (scratch); Sinv = R1^-1
//   SMALL_RQ2     pass 2: H2 = sum partials; R2 = chol(H2), breakdown when a pivot is below 1e-8 (no full rank);
//                 C = R2 R1; Sinv = R2^-1; then as SMALL_INIT
#include "common.cuh"

#define SMALL_THREADS 1024
#define SMALL_SMEM4_MAX_N 56 /* 4 x 56^2 x 16 = 196 KB of shared memory; 3 x 64^2 x 16 = 192 KB */

__device__ __forceinline__ double2 cmul(double2 a, double2 b)
{
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) // conj(a) * b
{
    return make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x);
}

// In-place upper Cholesky of the Hermitian matrix whose upper triangle is in A (row-major, shared memory).
// On return A = R (upper triangular, real positive diagonal, zeros below).  Whole CTA, right-looking: per column j one
// pivot test, the scaling of row j and the rank-1 update of the trailing triangle spread over all threads, three
// barriers (round 1 did this in one warp, a column per lane: 57 us per call at N = 16, most of it dependent
// shared-memory round trips).  Per element the operations and their order are those of the column version.
//
// Breakdown (U15): a pivot that is non-finite, non-positive, or has lost more than 13
// digits against the diagonal entry it started from (d <= 1e-13 h_jj: the column is linearly dependent on the
// previous ones to working precision, and only rounding noise decides the sign of the pivot).
// rel_tol / abs_tol: a pivot must exceed rel_tol * h_jj and abs_tol.  *finite_out: no NaN / Inf was met.  The return
// value and *finite_out are the same in every thread (they depend on shared-memory values read after a barrier).
__device__ bool cta_cholesky_upper(int N, double2 *A, double rel_tol, double abs_tol, bool *finite_out, double *h0)
{
    const int tid = threadIdx.x, nt = blockDim.x;
    for (int c = tid; c < N; c += nt) h0[c] = A[c * N + c].x;
    __syncthreads();
    *finite_out = true;
    for (int j = 0; j < N; j++) {
        const double d = A[j * N + j].x, hjj = h0[j];
        if (!isfinite(d) || !isfinite(hjj)) {
            *finite_out = false;
            return false;
        }
        if (!(d > rel_tol * hjj) || !(d > abs_tol)) return false;
        const double rjj = sqrt(d);
        __syncthreads(); // everyone has read the pivot
        for (int c = tid; c < N; c += nt) {
            if (c == j) A[j * N + j] = make_double2(rjj, 0.0);
            else if (c > j) {
                double2 v = A[j * N + c];
                A[j * N + c] = make_double2(v.x / rjj, v.y / rjj);
            } else A[j * N + c] = make_double2(0.0, 0.0);
        }
        __syncthreads();
        const int m = N - j - 1; // trailing block: rows / columns j + 1 .. N - 1, upper triangle
        for (int o = tid; o < m * m; o += nt) {
            const int i = j + 1 + o / m, c = j + 1 + o % m;
            if (c < i) continue;
            const double2 t = cmulc(A[j * N + i], A[j * N + c]);
            const double2 v = A[i * N + c];
            A[i * N + c] = make_double2(v.x - t.x, v.y - t.y);
        }
        __syncthreads();
    }
    return true;
}

// Ri = R^-1 for upper-triangular R with real diagonal, whole CTA: the entries at distance d = c - i from the diagonal
// depend only on those at smaller distances, so each distance is one parallel step (a dot product of length d per entry,
// summed in the order of the column-wise back substitution).
__device__ void cta_upper_inverse(int N, const double2 *R, double2 *Ri)
{
    const int tid = threadIdx.x, nt = blockDim.x;
    for (int o = tid; o < N * N; o += nt) {
        const int i = o / N, c = o % N;
        if (i > c) Ri[o] = make_double2(0.0, 0.0);
        else if (i == c) Ri[o] = make_double2(1.0 / R[o].x, 0.0);
    }
    __syncthreads();
    for (int d = 1; d < N; d++) {
        for (int i = tid; i + d < N; i += nt) {
            const int c = i + d;
            double2 s = make_double2(0.0, 0.0);
            for (int k = i + 1; k <= c; k++) {
                double2 t = cmul(R[i * N + k], Ri[k * N + c]);
                s.x += t.x;
                s.y += t.y;
            }
            const double dd = R[i * N + i].x;
            Ri[i * N + c] = make_double2(-s.x / dd, -s.y / dd);
        }
        __syncthreads();
    }
}

__device__ void load_hermitian(const SmallArgs &p, double2 *A)
{
    const int N = p.N;
    if (p.num_partials > 0) {
        // Second stage of the Gram reduction, fixed order, hence deterministic (P12): the partials q = 0, 1, 2, ... go to
        // four running sums by q mod 4, combined as (s0 + s1) + (s2 + s3).  Four adjacent lanes hold the four sums of
        // one matrix element (eight loads in flight each) and meet through shuffles: one serial chain of ~148 dependent
        // L2 loads cost 54 us per call, four interleaved chains in one thread ~10 us.
        const int g = threadIdx.x & 3, lane = threadIdx.x & 31, per = blockDim.x >> 2;
        const size_t stride = (size_t)N * N;
        for (int o0 = 0; o0 < N * N; o0 += per) {
            const int o = o0 + (threadIdx.x >> 2);
            const bool act = o < N * N;
            const int i = act ? o / N : 0, j = act ? o % N : 0;
            const int src = i <= j ? i * N + j : j * N + i;
            double2 acc = make_double2(0.0, 0.0);
            if (act) {
                const double2 *pp = p.partials + src;
                int q = g;
                for (; q + 28 < p.num_partials; q += 32) {
                    double2 v[8];
#pragma unroll
                    for (int c = 0; c < 8; c++) v[c] = pp[(size_t)(q + 4 * c) * stride];
#pragma unroll
                    for (int c = 0; c < 8; c++) {
                        acc.x += v[c].x;
                        acc.y += v[c].y;
                    }
                }
                for (; q < p.num_partials; q += 4) {
                    const double2 v = pp[(size_t)q * stride];
                    acc.x += v.x;
                    acc.y += v.y;
                }
            }
            const int b0 = lane & ~3;
            const double x0 = __shfl_sync(0xffffffffu, acc.x, b0), x1 = __shfl_sync(0xffffffffu, acc.x, b0 + 1),
                         x2 = __shfl_sync(0xffffffffu, acc.x, b0 + 2), x3 = __shfl_sync(0xffffffffu, acc.x, b0 + 3);
            const double y0 = __shfl_sync(0xffffffffu, acc.y, b0), y1 = __shfl_sync(0xffffffffu, acc.y, b0 + 1),
                         y2 = __shfl_sync(0xffffffffu, acc.y, b0 + 2), y3 = __shfl_sync(0xffffffffu, acc.y, b0 + 3);
            if (act && g == 0) {
                double2 s = make_double2((x0 + x1) + (x2 + x3), (y0 + y1) + (y2 + y3));
                if (i > j) s.y = -s.y;
                if (i == j) s.y = 0.0;
                A[o] = s;
            }
        }
    } else {
        for (int o = threadIdx.x; o < N * N; o += blockDim.x) {
            const int i = o / N, j = o % N;
            double2 s = p.in[i <= j ? o : j * N + i];
            if (i > j) s.y = -s.y;
            if (i == j) s.y = 0.0;
            A[o] = s;
        }
    }
    __syncthreads();
}

// residual norms from C (PAPER.md:208 with the index fix U11): r_i = ||C[:,i]|| / ||b_i||
__device__ double max_relres(int N, const double2 *C, const double *bnorm2, double *scratch)
{
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        double s = 0.0;
        for (int j = 0; j < N; j++) {
            double2 v = C[j * N + i];
            s += v.x * v.x + v.y * v.y;
        }
        scratch[i] = sqrt(s / bnorm2[i]);
    }
    __syncthreads();
    double m = 0.0;
    for (int i = 0; i < N; i++) m = fmax(m, scratch[i]);
    __syncthreads();
    return m;
}

__global__ void __launch_bounds__(SMALL_THREADS) small_kernel(SmallArgs p)
{
    extern __shared__ double2 sm[];
    const int N = p.N, NN = N * N;
    // four N x N matrices; above N = 56 the fourth (a read-mostly copy) lives in global memory: 4 x 64^2 x 16 bytes do not fit
    double2 *A = sm, *B = sm + NN, *Cm = sm + 2 * NN, *Dm = N > SMALL_SMEM4_MAX_N ? p.scratch : sm + 3 * NN;
    __shared__ int ok_s, finite_s;
    __shared__ double scratch[BKR_MAX_N], h0s[BKR_MAX_N];
    SolverFlags *fl = p.flags;
    if (p.mode >= SMALL_BETA && p.mode <= SMALL_QR && fl->done) {
        if (p.mode == SMALL_BETA && threadIdx.x == 0) { // no new W: nothing left to apply to X after this iteration
            fl->xpend = 0;
            fl->xidle = 1;
        }
        return;
    }

    load_hermitian(p, A);
    if (p.mode == SMALL_RQ1) { // shifted Cholesky QR: H + s 1, s = 1e-12 max_i H_ii
        double hmax = 0.0;
        for (int i = 0; i < N; i++) hmax = fmax(hmax, A[i * N + i].x);
        __syncthreads();
        if (threadIdx.x < N) A[threadIdx.x * N + threadIdx.x].x += 1e-12 * hmax;
        __syncthreads();
    }
    {
        // Breakdown thresholds (U15): 13 digits lost against the diagonal entry for Gram matrices of fp64 blocks;
        // fp32 blocks carry rounding noise of ~1e-7 h_jj, so a rank-deficient one would pass that test with a noise pivot:
        // the caller passes pivot_tol = 4e-6 there.  Pass 2 of the two-pass QR: columns have norm <= 1 after pass 1, a
        // pivot below 1e-8 is the image of rounding noise (no full rank).
        const double rel = p.pivot_tol > 0.0 ? p.pivot_tol : 1e-13;
        bool fin = true;
        bool ok = cta_cholesky_upper(N, A, rel, p.mode == SMALL_RQ2 ? 1e-8 : 0.0, &fin, h0s); // A = R
        if (ok) cta_upper_inverse(N, A, B); // B = R^-1
        if (threadIdx.x == 0) {
            ok_s = ok ? 1 : 0;
            finite_s = fin ? 1 : 0;
        }
    }
    __syncthreads();
    const bool ok = ok_s != 0;
    if (!ok) {
        if (threadIdx.x == 0) {
            if (p.status) *p.status = BKR_EBREAKDOWN;
            if (fl) {
                fl->breakdown = 1;
                fl->illcond = (finite_s && p.mode != SMALL_RQ2) ? 1 : 0;
                fl->done = 1;
                if (p.mode == SMALL_BETA) {
                    fl->xpend = 0;
                    fl->xidle = 1;
                }
            }
        }
        return;
    }
    if (threadIdx.x == 0 && p.status) *p.status = BKR_OK;

    switch (p.mode) {
    case SMALL_CHOL:
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            p.out0[o] = A[o];
            if (p.out1) p.out1[o] = B[o];
        }
        break;
    case SMALL_HPDINV:
    case SMALL_BETA: {
        // beta = R^-1 R^-dag : beta_ij = sum_k Ri_ik conj(Ri_jk), k >= max(i,j)
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            int i = o / N, j = o % N;
            double2 s = make_double2(0.0, 0.0);
            for (int k = (i > j ? i : j); k < N; k++) {
                double2 t = cmulc(B[j * N + k], B[i * N + k]);
                s.x += t.x;
                s.y += t.y;
            }
            Cm[o] = s;
        }
        __syncthreads();
        if (p.mode == SMALL_HPDINV) {
            for (int o = threadIdx.x; o < NN; o += blockDim.x) p.out0[o] = Cm[o];
            break;
        }
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            Dm[o] = p.C[o];
            p.negbeta[o] = make_double2(-Cm[o].x, -Cm[o].y);
        }
        __syncthreads();
        for (int o = threadIdx.x; o < NN; o += blockDim.x) { // W = beta C, C upper triangular
            int i = o / N, j = o % N;
            double2 s = make_double2(0.0, 0.0);
            for (int k = 0; k <= j; k++) {
                double2 t = cmul(Cm[i * N + k], Dm[k * N + j]);
                s.x += t.x;
                s.y += t.y;
            }
            p.W[o] = s;
        }
        if (threadIdx.x == 0 && fl) { // W is valid and not yet applied to X
            fl->xpend = 1;
            fl->xidle = 0;
        }
        break;
    }
    case SMALL_QR: {
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            int i = o / N, j = o % N;
            double2 c = p.C[o];
            Dm[o] = c;
            p.Cprev[o] = c;
            p.Sinv[o] = B[o];
            double2 s = A[j * N + i]; // S^dag_ij = conj(S_ji)
            p.Sdag[o] = make_double2(s.x, -s.y);
        }
        __syncthreads();
        for (int o = threadIdx.x; o < NN; o += blockDim.x) { // C = S C, both upper triangular
            int i = o / N, j = o % N;
            double2 s = make_double2(0.0, 0.0);
            for (int k = i; k <= j; k++) {
                double2 t = cmul(A[i * N + k], Dm[k * N + j]);
                s.x += t.x;
                s.y += t.y;
            }
            Cm[o] = s;
            p.C[o] = s;
        }
        __syncthreads();
        double r = max_relres(N, Cm, p.bnorm2, scratch);
        if (threadIdx.x == 0) {
            fl->iters += 1;
            fl->relres_max = r;
            if (!p.mixed) {
                if (r <= p.tol) fl->done = 1;
            } else if (r < p.delta * fl->relres_last_update || r <= p.tol) fl->want_update = 1;
        }
        break;
    }
    case SMALL_RQ1:
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            p.W[o] = A[o];    // R1, kept for pass 2
            p.Sinv[o] = B[o]; // Q1 = R R1^-1
        }
        break;
    case SMALL_RQ2: // C = R2 R1 (both upper triangular), then as SMALL_INIT with A = C
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            Dm[o] = p.W[o];
            Cm[o] = A[o];
        }
        __syncthreads();
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            int i = o / N, j = o % N;
            double2 s = make_double2(0.0, 0.0);
            for (int k = i; k <= j; k++) {
                double2 t = cmul(Cm[i * N + k], Dm[k * N + j]);
                s.x += t.x;
                s.y += t.y;
            }
            A[o] = s;
        }
        __syncthreads();
        // fall through
    case SMALL_INIT: {
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            int i = o / N, j = o % N;
            p.C[o] = A[o];
            p.Cprev[o] = A[o];
            p.Sinv[o] = B[o];
            p.Sdag[o] = make_double2(i == j ? 1.0 : 0.0, 0.0);
        }
        double r = max_relres(N, A, p.bnorm2, scratch);
        if (threadIdx.x == 0) {
            fl->relres_max = r;
            fl->relres_last_update = r;
            fl->want_update = 0;
            if (r <= p.tol) fl->done = 1;
        }
        break;
    }
    case SMALL_RELUPD: {
        // A = C_new, B = C_new^-1.  S = C_new Cprev^-1 (Alg. 3 l.6, C_old = C before this iteration's l.12: U12)
        for (int o = threadIdx.x; o < NN; o += blockDim.x) Dm[o] = p.Cprev[o];
        __syncthreads();
        cta_upper_inverse(N, Dm, Cm); // Cm = Cprev^-1
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            int i = o / N, j = o % N;
            double2 s = make_double2(0.0, 0.0);
            for (int k = i; k <= j; k++) {
                double2 t = cmul(A[i * N + k], Cm[k * N + j]);
                s.x += t.x;
                s.y += t.y;
            }
            Dm[o] = s; // S_ij
        }
        __syncthreads();
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            int i = o / N, j = o % N;
            double2 s = Dm[j * N + i];
            p.Sdag[o] = make_double2(s.x, -s.y);
            p.Sinv[o] = B[o];
            p.C[o] = A[o];
        }
        double r = max_relres(N, A, p.bnorm2, scratch);
        if (threadIdx.x == 0) {
            fl->relres_max = r;
            fl->relres_last_update = r;
            fl->want_update = 0;
            if (r <= p.tol) fl->done = 1;
        }
        break;
    }
    }
}

int launch_small(bkr_ctx *ctx, const SmallArgs &args_in)
{
    SmallArgs args = args_in;
    args.scratch = ctx->small + (size_t)4 * BKR_MAX_N * BKR_MAX_N;
    const size_t nmat = args.N > SMALL_SMEM4_MAX_N ? 3 : 4;
    size_t smem = nmat * args.N * args.N * sizeof(double2);
    static int attr_dev = -1; // the opt-in is per device
    if (attr_dev != ctx->device) {
        cudaFuncSetAttribute(small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)(4 * SMALL_SMEM4_MAX_N * SMALL_SMEM4_MAX_N * sizeof(double2)));
        attr_dev = ctx->device;
    }
    small_kernel<<<1, SMALL_THREADS, smem, ctx->stream>>>(args);
    return bkr_check_launch(ctx);
}

// Scalars of the CG baseline (ref. [40]): step 0: alpha = rho / pAp; step 1: beta = rho'/rho,
// convergence per rhs, rho = rho'.  A converged rhs keeps alpha = 0 so that its x no longer changes.
__global__ void cg_scalar_kernel(int N, int step, double tol, CgScalars *s, SolverFlags *fl)
{
    if (fl->done) return;
    int j = threadIdx.x;
    __shared__ int all_conv;
    if (j == 0) all_conv = 1;
    __syncthreads();
    if (j < N) {
        if (step == 2) { // initial residual already below tol?
            if (sqrt(s->rho[j] / s->bb[j]) <= tol) s->conv[j] = 1;
            else all_conv = 0;
        } else if (step == 0) {
            s->alpha[j] = s->conv[j] ? 0.0 : s->rho[j] / s->pAp[j];
        } else {
            if (!s->conv[j]) {
                s->iters[j] += 1;
                double rn = s->rho_new[j];
                s->beta[j] = rn / s->rho[j];
                s->rho[j] = rn;
                if (sqrt(rn / s->bb[j]) <= tol) s->conv[j] = 1;
            } else s->beta[j] = 0.0;
            if (!s->conv[j]) all_conv = 0;
        }
    }
    __syncthreads();
    if (j == 0 && step != 0) {
        if (step == 1) fl->iters += 1;
        if (all_conv) fl->done = 1;
    }
}

int launch_cg_scalar(bkr_ctx *ctx, int N, int step, double tol, CgScalars *s, SolverFlags *flags)
{
    cg_scalar_kernel<<<1, BKR_MAX_N, 0, ctx->stream>>>(N, step, tol, s, flags);
    return bkr_check_launch(ctx);
}
