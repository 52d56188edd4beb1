// Small dense N x N algebra on the device (PAPER.md:178 does it on the host with Eigen; north_star moves it
// into a device-side kernel so that no Gram matrix or coefficient matrix ever crosses to the host).
//
// A cluster of SMALL_CLUSTER CTAs of 1024 threads.  All of them: the deterministic second stage of the Gram reduction
// (fixed-order sum of the per-CTA partials, Hermitised from the upper triangle), each a slice of the matrix,
// stored into rank 0's shared memory.  Rank 0 alone: the Cholesky factorisation H = R^dag R (Algorithm 2 l.3), the
// triangular inverse and the N x N products, matrices in shared memory; up to 32 rhs a thread per matrix element with the
// element in a register and one barrier per column (16 us per call at N = 16; 43 us before, 57 us in round 1).
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

#include <cooperative_groups.h>
namespace cg = cooperative_groups;

#define SMALL_THREADS 1024
#define SMALL_CLUSTER 8 /* CTAs that share the second stage of the Gram reduction (load_hermitian); rank 0 does the rest */
#define SMALL_SMEM4_MAX_N 56 /* 4 x 56^2 x 16 = 196 KB of shared memory; 3 x 64^2 x 16 = 192 KB */

__device__ __forceinline__ double2 cmul(double2 a, double2 b)
{
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) // conj(a) * b
{
    return make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x);
}

// Named barrier 1 over the first nth threads of the CTA (nth a multiple of 32): the factorisation and the triangular
// inverse run on 32 x clamp(N, 8, 32) threads -- a barrier over all 32 warps costs twice one over 8.
__device__ __forceinline__ void bar_part(int nth) { asm volatile("bar.sync 1, %0;" ::"r"(nth) : "memory"); }
__device__ __forceinline__ int small_part_threads(int N) { return 32 * (N < 8 ? 8 : N > 32 ? 32 : N); }

// N <= 32: thread (warp i, lane c) of the 1024 owns matrix element (i, c) and keeps it in a register; one CTA barrier per
// column.  A single warp issues one dependent instruction every ~5 cycles, so what counts is the number of instructions on
// the chain from one pivot to the next, not their latencies (measured on this GPU: DFMA 8, shuffle 9, 1/x 81, rsqrt 74,
// a 1024-thread barrier 76 cycles): here the chain is a row store, the barrier, three shared-memory reads, a reciprocal
// and one complex multiply-add, ~220 cycles per column.  Versions tried before it, at N = 16: one warp through shared
// memory 57 us (round 1); CTA-wide with three barriers and two divisions per column 27 k cycles; one barrier and a warp per
// trailing row 16 k; one warp with the pivot row in shuffles 32 k (a warp alone is issue bound); this one 3.5 k.
//
// Column j: warp j stores its (final, still unscaled) row into R; after the barrier every thread below it subtracts
// conj(a_ji) a_jc / d, d = a_jj.  At the end row i is scaled by rsqrt(d_i).  Pivot tests as in part_cholesky_upper.
// Called by ALL threads (the return value is the same in each); the caller puts a barrier behind it.
__device__ bool reg_cholesky_upper(int N, const double2 *A, double2 *R, double rel_tol, double abs_tol, bool *finite_out, double *h0)
{
    const int i = threadIdx.x >> 5, c = threadIdx.x & 31;
    const bool own = i < N && c < N && c >= i;
    double2 v = own ? A[i * N + c] : make_double2(0.0, 0.0);
    if (own && i == c) h0[i] = v.x;
    *finite_out = true;
    for (int j = 0; j < N; j++) {
        if (i == j && c < N) R[j * N + c] = v; // zeros left of the diagonal
        __syncthreads();
        const double d = R[j * N + j].x, hjj = h0[j];
        if (!isfinite(d) || !isfinite(hjj)) {
            *finite_out = false;
            return false;
        }
        if (!(d > rel_tol * hjj) || !(d > abs_tol)) return false;
        if (own && i > j) {
            const double dinv = 1.0 / d;
            const double2 t = cmulc(R[j * N + i], R[j * N + c]);
            v.x -= t.x * dinv;
            v.y -= t.y * dinv;
        }
    }
    __syncthreads(); // the last pivot has been read by everyone
    if (i < N) { // every row is in R and nobody reads another warp's row any more: scale row i in place
        const double di = R[i * N + i].x, rin = rsqrt(di);
        __syncwarp();
        if (c < N && c >= i) R[i * N + c] = c == i ? make_double2(di * rin, 0.0) : make_double2(v.x * rin, v.y * rin);
    }
    return true;
}

// Ri = R^-1 for N <= 32 in the same layout: thread (i, c) accumulates s_ic = sum_{k > i} R_ik X_kc in a register while the
// rows of X = R^-1 become final from the bottom up (row k = (e_k - s_k) / R_kk), one CTA barrier per row.  Called by all
// threads; Ri is complete and visible when it returns.
__device__ void reg_upper_inverse(int N, const double2 *R, double2 *Ri)
{
    const int i = threadIdx.x >> 5, c = threadIdx.x & 31;
    const bool own = i < N && c < N && c >= i;
    const double rinv = i < N ? 1.0 / R[i * N + i].x : 0.0;
    double2 s = make_double2(0.0, 0.0);
    for (int k = N - 1; k >= 0; k--) {
        if (i == k && c < N)
            Ri[k * N + c] = c > k ? make_double2(-s.x * rinv, -s.y * rinv) : c == k ? make_double2(rinv, 0.0) : make_double2(0.0, 0.0);
        __syncthreads();
        if (own && i < k && c >= k) {
            const double2 t = cmul(R[i * N + k], Ri[k * N + c]);
            s.x += t.x;
            s.y += t.y;
        }
    }
}

// Upper Cholesky factor of the Hermitian matrix in A (row-major, shared memory; upper triangle read, trailing part
// overwritten): R (upper triangular, real positive diagonal, zeros below) goes to a second matrix, so that a column step
// needs ONE barrier: everyone reads the pivot d and the still unscaled row j, writes r_jc = a_jc / sqrt(d) to R and updates
// the trailing triangle with conj(a_ji) a_jc / d (= conj(r_ji) r_jc).  A warp per trailing row, lanes across its columns.
// Round 1 did this in one warp through shared memory (57 us at N = 16); the first CTA-wide version took three barriers over
// 1024 threads and two dependent fp64 divisions per column (27 k cycles at N = 16); this one ~7 k.
// Called by threads 0 .. nth - 1 only.
//
// Breakdown (U15): a pivot that is non-finite, non-positive, or has lost more than 13
// digits against the diagonal entry it started from (d <= 1e-13 h_jj: the column is linearly dependent on the
// previous ones to working precision, and only rounding noise decides the sign of the pivot).
// rel_tol / abs_tol: a pivot must exceed rel_tol * h_jj and abs_tol.  *finite_out: no NaN / Inf was met.  The return
// value and *finite_out are the same in every calling thread (shared-memory values read after a barrier).
__device__ bool part_cholesky_upper(int N, double2 *A, double2 *R, double rel_tol, double abs_tol, bool *finite_out, double *h0,
                                    int nth)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = nth >> 5;
    for (int c = tid; c < N; c += nth) h0[c] = A[c * N + c].x;
    for (int i = 1 + warp; i < N; i += nwarp)
        for (int c = lane; c < i; c += 32) R[i * N + c] = make_double2(0.0, 0.0);
    bar_part(nth);
    *finite_out = true;
    for (int j = 0; j < N; j++) {
        const double d = A[j * N + j].x, hjj = h0[j];
        if (!isfinite(d) || !isfinite(hjj)) {
            *finite_out = false;
            return false;
        }
        if (!(d > rel_tol * hjj) || !(d > abs_tol)) return false;
        const double rjj = sqrt(d), rinv = 1.0 / rjj, dinv = 1.0 / d;
        for (int c = j + tid; c < N; c += nth) {
            const double2 v = A[j * N + c];
            R[j * N + c] = c == j ? make_double2(rjj, 0.0) : make_double2(v.x * rinv, v.y * rinv);
        }
        for (int i = j + 1 + warp; i < N; i += nwarp) { // trailing block, upper triangle
            const double2 aji = A[j * N + i];
            for (int c = i + lane; c < N; c += 32) {
                const double2 t = cmulc(aji, A[j * N + c]);
                const double2 v = A[i * N + c];
                A[i * N + c] = make_double2(v.x - t.x * dinv, v.y - t.y * dinv);
            }
        }
        bar_part(nth);
    }
    return true;
}

// Ri = R^-1 for upper-triangular R with real diagonal, 32 < N <= 64, whole CTA, no barrier inside: a warp per column c of Ri,
// which is the back substitution R x = e_c.  Lane k keeps the running sums s_k = sum_{m > k} R_km x_m of rows k and k + 32;
// x_i = -s_i / R_ii is formed in the lane that owns row i, broadcast by a shuffle, and every lane above adds R_ki x_i.  The
// chain per entry is a multiply, a shuffle and a multiply-add.  Called by all threads; ends with a CTA barrier.
__device__ void cta_upper_inverse(int N, const double2 *R, double2 *Ri)
{
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const double rinv0 = lane < N ? 1.0 / R[lane * N + lane].x : 0.0;
    const double rinv1 = lane + 32 < N ? 1.0 / R[(lane + 32) * N + lane + 32].x : 0.0;
    for (int c = warp; c < N; c += nwarp) {
        double2 s0 = make_double2(0.0, 0.0), s1 = make_double2(0.0, 0.0);
        for (int i = c; i >= 0; i--) {
            const bool hi = i >= 32;
            const double2 s = hi ? s1 : s0;
            const double ri = hi ? rinv1 : rinv0;
            double2 xi = i == c ? make_double2(ri, 0.0) : make_double2(-s.x * ri, -s.y * ri);
            xi.x = __shfl_sync(full, xi.x, i & 31);
            xi.y = __shfl_sync(full, xi.y, i & 31);
            if (lane < i) {
                const double2 t = cmul(R[lane * N + i], xi);
                s0.x += t.x;
                s0.y += t.y;
            }
            if (lane + 32 < i) {
                const double2 t = cmul(R[(lane + 32) * N + i], xi);
                s1.x += t.x;
                s1.y += t.y;
            }
            if (lane == (i & 31)) Ri[i * N + c] = xi;
        }
        for (int i = c + 1 + lane; i < N; i += 32) Ri[i * N + c] = make_double2(0.0, 0.0);
    }
    __syncthreads();
}

__device__ void upper_inverse(int N, const double2 *R, double2 *Ri)
{
    if (N <= 32) reg_upper_inverse(N, R, Ri);
    else cta_upper_inverse(N, R, Ri);
}

// H (N x N, into A0 = the A matrix of cluster rank 0, through distributed shared memory for the other ranks) = the
// fixed-order sum of the per-CTA partials of the Gram reduction, Hermitised from the upper triangle, or the
// caller's matrix `in`.  The partials are 148 x N^2 x 16 bytes (0.6 MB at N = 16, 2.4 MB at N = 32): one SM pulls them from
// L2 at ~20 B/clk, which was 30 k of the kernel's 82 k cycles at N = 16 and 110 k of 240 k at N = 32.  So the kernel runs as
// a cluster of SMALL_CLUSTER CTAs: rank r sums a contiguous slice of the matrix elements and stores them into rank 0's shared
// memory; after a cluster barrier rank 0 goes on alone.  Per element, fixed order hence deterministic (P12): 16 lanes take the
// partials q = g, g + 16, g + 32, ... (all loads of a lane in flight at once), a butterfly over the 16 lanes adds them up; two
// adjacent elements per warp so that every load instruction reads whole 32-byte sectors.
__device__ void load_hermitian(const SmallArgs &p, double2 *A0, int rank, int nrank)
{
    const int N = p.N, NN = N * N;
    if (p.num_partials > 0) {
        const int per = ((NN + nrank - 1) / nrank + 1) & ~1; // elements per rank, even
        const int o_lo = rank * per, o_hi = min(NN, o_lo + per);
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
        const int g = lane >> 1, e = lane & 1;
        const size_t stride = (size_t)NN;
        for (int ob = o_lo + 2 * warp; ob < o_hi; ob += 2 * nwarp) { // warp-uniform
            const int o = ob + e;
            const bool act = o < o_hi;
            const int i = act ? o / N : 0, j = act ? o % N : 0;
            const int src = i <= j ? i * N + j : j * N + i;
            double2 acc = sum_partials_16(p.partials + src, stride, p.num_partials, g, act);
            if (act && g == 0) {
                if (i > j) acc.y = -acc.y;
                if (i == j) acc.y = 0.0;
                A0[o] = acc;
            }
        }
    } else if (rank == 0) {
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            const int i = o / N, j = o % N;
            double2 s = p.in[i <= j ? o : j * N + i];
            if (i > j) s.y = -s.y;
            if (i == j) s.y = 0.0;
            A0[o] = s;
        }
    }
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

__global__ void __cluster_dims__(SMALL_CLUSTER, 1, 1) __launch_bounds__(SMALL_THREADS) small_kernel(SmallArgs p)
{
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    extern __shared__ double2 sm[];
    const int N = p.N, NN = N * N;
    // four N x N matrices; above N = 56 the fourth (a read-mostly copy) lives in global memory: 4 x 64^2 x 16 bytes do not fit
    double2 *A = sm, *B = sm + NN, *Cm = sm + 2 * NN, *Dm = N > SMALL_SMEM4_MAX_N ? p.scratch : sm + 3 * NN;
    __shared__ int ok_s, finite_s;
    __shared__ double scratch[BKR_MAX_N], h0s[BKR_MAX_N];
    SolverFlags *fl = p.flags;
    if (p.mode >= SMALL_BETA && p.mode <= SMALL_QR && fl->done) { // the same in every CTA of the cluster
        if (p.mode == SMALL_BETA && threadIdx.x == 0 && rank == 0) { // no new W: nothing left to apply to X after this iteration
            fl->xpend = 0;
            fl->xidle = 1;
        }
        return;
    }

    cluster.sync(); // every CTA of the cluster runs: its shared memory may be written from the others
    load_hermitian(p, cluster.map_shared_rank(A, 0), rank, SMALL_CLUSTER);
    cluster.sync();
    if (rank != 0) return;
    if (p.mode == SMALL_RQ1) { // shifted Cholesky QR: H + s 1, s = 1e-12 max_i H_ii
        double hmax = 0.0;
        for (int i = 0; i < N; i++) hmax = fmax(hmax, A[i * N + i].x);
        __syncthreads();
        if (threadIdx.x < N) A[threadIdx.x * N + threadIdx.x].x += 1e-12 * hmax;
        __syncthreads();
    }
    const int nth = small_part_threads(N);
    {
        // Breakdown thresholds (U15): 13 digits lost against the diagonal entry for Gram matrices of fp64 blocks;
        // fp32 blocks carry rounding noise of ~1e-7 h_jj, so a rank-deficient one would pass that test with a noise pivot:
        // the caller passes pivot_tol = 4e-6 there.  Pass 2 of the two-pass QR: columns have norm <= 1 after pass 1, a
        // pivot below 1e-8 is the image of rounding noise (no full rank).
        const double rel = p.pivot_tol > 0.0 ? p.pivot_tol : 1e-13;
        bool fin = true, okc = true;
        if (N <= 32) {
            okc = reg_cholesky_upper(N, A, Cm, rel, p.mode == SMALL_RQ2 ? 1e-8 : 0.0, &fin, h0s); // Cm = R
        } else if ((int)threadIdx.x < nth) {
            okc = part_cholesky_upper(N, A, Cm, rel, p.mode == SMALL_RQ2 ? 1e-8 : 0.0, &fin, h0s, nth);
        }
        if (threadIdx.x == 0) {
            ok_s = okc ? 1 : 0;
            finite_s = fin ? 1 : 0;
        }
    }
    __syncthreads();
    if (ok_s) upper_inverse(N, Cm, B); // B = R^-1 (uniform branch; complete and visible on return)
    {
        double2 *t = A; // from here on A = R; the matrix the factorisation worked in is scratch
        A = Cm;
        Cm = t;
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
        // beta = R^-1 R^-dag : beta_ij = sum_k Ri_ik conj(Ri_jk), k >= max(i,j).  The lanes of a warp run over j: Ri_jk is read
        // from a transposed copy (in A: R is not needed any more), else every lane hits the same bank (21 k cycles at N = 32)
        for (int o = threadIdx.x; o < NN; o += blockDim.x) A[(o % N) * N + o / N] = B[o];
        __syncthreads();
        for (int o = threadIdx.x; o < NN; o += blockDim.x) {
            int i = o / N, j = o % N;
            double2 s = make_double2(0.0, 0.0);
            for (int k = (i > j ? i : j); k < N; k++) {
                double2 t = cmulc(A[k * N + j], B[i * N + k]);
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
        upper_inverse(N, Dm, Cm); // Cm = Cprev^-1
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
    small_kernel<<<SMALL_CLUSTER, SMALL_THREADS, smem, ctx->stream>>>(args); // one cluster (__cluster_dims__)
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
