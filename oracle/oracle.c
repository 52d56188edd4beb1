/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 *
 * A plain, slow, fp64 CPU statement of what the hot path of arXiv:1710.09745 computes:
 * the improved-staggered hop operator, the even-odd normal operator, the block BLAS
 * (eq. 3, eq. 4), thin QR (Algorithm 2), CG, blockCGrQ (Algorithm 1) and blockCGrQ with
 * block reliable updates (Algorithm 3).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this file.  It shares no code,
 * header, table or helper with the CUDA library under paper_1710_09745_b200/csrc.
 *
 * Citations are "PAPER.md:<line>" (the paper text under /root/reference) plus the reading
 * of DESIGN.md ("U<n>") where the extracted text is silent or garbled.
 *
 * Pins (tests/test_oracle_pins.py, all CPU): anti-Hermiticity of D, Hermitian positive
 * definiteness of M, the free-field closed-form spectrum (4^4 worked example and plane
 * waves at other sizes), gauge covariance, dense brute force on 4^4 assembled independently
 * in numpy, N=1 == CG, finite termination on the 5-eigenvalue free field, thin-QR
 * identities (also for the two-pass QR on nearly dependent columns), numpy.linalg for the small matrices.  Nothing here is "parity unpinned"
 * except iteration counts on the synthetic configs (no published value exists).
 *
 * Layouts (canonical, host memory, complex = (re, im) fp64):
 *   links  U[mu][s][a][b],  mu = 0..3 (x,y,z,t), s = x + X(y + Y(z + Z t)) lexicographic,
 *          staggered phases / boundary signs / coefficients already folded in;
 *   vector v[rhs][e][a],    e = s div 2 = even-odd index of a site of the field's parity
 *          (all extents even), a = colour 0..2;  one parity has Vh = V/2 sites;
 *   block  as L x N with L = 3 Vh rows k = 3 e + a, stored column by column: v[j*L + k];
 *   small  N x N matrices row-major: a[i*N + j].
 *
 * The only concession to speed is "#pragma omp parallel for" over sites / rows / (i,j);
 * every sum over the long index k runs in index order in fp64.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

/* ---------------------------------------------------------------- geometry (U6) */

static long lexidx(const int D[4], const int c[4])
{
    return c[0] + (long)D[0] * (c[1] + (long)D[1] * (c[2] + (long)D[2] * c[3]));
}

/* coordinates of the site with even-odd index e and parity p = (x+y+z+t) mod 2 */
static void coords_of(const int D[4], int parity, long e, int c[4])
{
    long s0 = 2 * e; /* the pair {s0, s0+1} lies in one x-row because X is even */
    int x0 = (int)(s0 % D[0]);
    long r = s0 / D[0];
    c[1] = (int)(r % D[1]);
    r /= D[1];
    c[2] = (int)(r % D[2]);
    c[3] = (int)(r / D[2]);
    c[0] = x0 + ((c[1] + c[2] + c[3] + parity) & 1);
}

static int dims_ok(const int D[4])
{
    for (int mu = 0; mu < 4; mu++)
        if (D[mu] < 4 || (D[mu] & 1)) return 0;
    return 1;
}

/* ------------------------------------------------ hop operator, PAPER.md:95-101 (eq. 2), U1/U2
 * (D psi)(x) = sum_mu [ F_mu(x) psi(x+mu) - F_mu(x-mu)^dag psi(x-mu)
 *                     + K_mu(x) psi(x+3mu) - K_mu(x-3mu)^dag psi(x-3mu) ]
 * F = fat (one hop), K = long (three hops).  `in` is one rhs of the opposite parity. */
static void hop_site(const int D[4], long V, const cplx *fat, const cplx *lng,
                     const int c[4], const cplx *in, cplx out[3])
{
    long s = lexidx(D, c);
    out[0] = out[1] = out[2] = 0.0;
    for (int mu = 0; mu < 4; mu++) {
        for (int h = 1; h <= 3; h += 2) {
            const cplx *U = (h == 1) ? fat : lng;
            int cf[4] = {c[0], c[1], c[2], c[3]};
            int cb[4] = {c[0], c[1], c[2], c[3]};
            cf[mu] = (c[mu] + h) % D[mu];
            cb[mu] = (c[mu] - h + D[mu]) % D[mu];
            long sf = lexidx(D, cf), sb = lexidx(D, cb);
            const cplx *Uf = U + ((long)mu * V + s) * 9;  /* link leaving x            */
            const cplx *Ub = U + ((long)mu * V + sb) * 9; /* link leaving x - h mu     */
            const cplx *pf = in + (sf / 2) * 3;
            const cplx *pb = in + (sb / 2) * 3;
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++)
                    out[a] += Uf[a * 3 + b] * pf[b] - conj(Ub[b * 3 + a]) * pb[b];
        }
    }
}

/* out[rhs][e][a] (parity out_parity) = D_{out_parity, 1-out_parity} in[rhs][e][a] */
int orc_dslash(const int D[4], const cplx *fat, const cplx *lng, int out_parity, int N,
               const cplx *in, cplx *out)
{
    if (!dims_ok(D) || N < 1) return -1;
    long V = (long)D[0] * D[1] * D[2] * D[3], Vh = V / 2;
    for (int j = 0; j < N; j++) {
#pragma omp parallel for schedule(static)
        for (long e = 0; e < Vh; e++) {
            int c[4];
            coords_of(D, out_parity, e, c);
            hop_site(D, V, fat, lng, c, in + (long)j * Vh * 3, out + ((long)j * Vh + e) * 3);
        }
    }
    return 0;
}

/* the same at a list of output sites only: out[rhs][i][a] for e = e_idx[i] */
int orc_dslash_sites(const int D[4], const cplx *fat, const cplx *lng, int out_parity, int N,
                     const cplx *in, long nsites, const long *e_idx, cplx *out)
{
    if (!dims_ok(D) || N < 1) return -1;
    long V = (long)D[0] * D[1] * D[2] * D[3], Vh = V / 2;
    for (int j = 0; j < N; j++)
        for (long i = 0; i < nsites; i++) {
            int c[4];
            coords_of(D, out_parity, e_idx[i], c);
            hop_site(D, V, fat, lng, c, in + (long)j * Vh * 3, out + ((long)j * nsites + i) * 3);
        }
    return 0;
}

/* M psi_e = 4 m^2 psi_e - D_eo (D_oe psi_e), PAPER.md:103 ("Schur decomposed"), U3.
 * tmp_odd: caller's scratch of N*Vh*3 complex. */
int orc_apply_M(const int D[4], const cplx *fat, const cplx *lng, double mass, int N,
                const cplx *in, cplx *out, cplx *tmp_odd)
{
    if (!dims_ok(D) || N < 1) return -1;
    long Vh = (long)D[0] * D[1] * D[2] * D[3] / 2, n = (long)N * Vh * 3;
    orc_dslash(D, fat, lng, 1, N, in, tmp_odd);
    orc_dslash(D, fat, lng, 0, N, tmp_odd, out);
    double m2 = 4.0 * mass * mass;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; i++) out[i] = m2 * in[i] - out[i];
    return 0;
}

/* ------------------------------------------------------------------ block BLAS (eq. 3, eq. 4) */

/* K = X^dag Y, k_ij = sum_k conj(x_ki) y_kj, PAPER.md:274-277 (eq. 4) */
void orc_gram(long L, int N, const cplx *X, const cplx *Y, cplx *K)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int i = 0; i < N; i++)
        for (int j = 0; j < N; j++) {
            cplx s = 0.0;
            for (long k = 0; k < L; k++) s += conj(X[(long)i * L + k]) * Y[(long)j * L + k];
            K[i * N + j] = s;
        }
}

/* Y <- Y + X a, y_kj += sum_i x_ki a_ij, PAPER.md:249-252 (eq. 3) */
void orc_block_axpy(long L, int N, const cplx *a, const cplx *X, cplx *Y)
{
#pragma omp parallel for schedule(static)
    for (long k = 0; k < L; k++)
        for (int j = 0; j < N; j++) {
            cplx s = 0.0;
            for (int i = 0; i < N; i++) s += X[(long)i * L + k] * a[i * N + j];
            Y[(long)j * L + k] += s;
        }
}

/* --------------------------------------------------------------------- small dense N x N */

/* use the upper triangle, real diagonal (U9) */
static void hermitise(int N, cplx *H)
{
    for (int i = 0; i < N; i++) {
        H[i * N + i] = creal(H[i * N + i]);
        for (int j = i + 1; j < N; j++) H[j * N + i] = conj(H[i * N + j]);
    }
}

/* H = R^dag R, R upper triangular with real positive diagonal, PAPER.md:169 (Alg. 2 l.3), U8.
 * returns -5 on a non-positive or non-finite pivot (U15). */
int orc_cholesky_upper(int N, const cplx *H, cplx *R)
{
    memset(R, 0, sizeof(cplx) * N * N);
    for (int j = 0; j < N; j++) {
        double d = creal(H[j * N + j]);
        for (int k = 0; k < j; k++) d -= creal(R[k * N + j] * conj(R[k * N + j]));
        if (!(d > 0.0) || !isfinite(d)) return -5;
        double rjj = sqrt(d);
        R[j * N + j] = rjj;
        for (int i = j + 1; i < N; i++) {
            cplx s = H[j * N + i];
            for (int k = 0; k < j; k++) s -= conj(R[k * N + j]) * R[k * N + i];
            R[j * N + i] = s / rjj;
        }
    }
    return 0;
}

/* inverse of an upper-triangular matrix by back substitution, column by column */
void orc_upper_inverse(int N, const cplx *R, cplx *Ri)
{
    memset(Ri, 0, sizeof(cplx) * N * N);
    for (int j = 0; j < N; j++) {
        Ri[j * N + j] = 1.0 / R[j * N + j];
        for (int i = j - 1; i >= 0; i--) {
            cplx s = 0.0;
            for (int k = i + 1; k <= j; k++) s += R[i * N + k] * Ri[k * N + j];
            Ri[i * N + j] = -s / R[i * N + i];
        }
    }
}

static void matmul(int N, const cplx *A, const cplx *B, cplx *C)
{
    for (int i = 0; i < N; i++)
        for (int j = 0; j < N; j++) {
            cplx s = 0.0;
            for (int k = 0; k < N; k++) s += A[i * N + k] * B[k * N + j];
            C[i * N + j] = s;
        }
}

/* G^-1 for Hermitian positive-definite G = U^dag U:  G^-1 = U^-1 U^-dag  (U9) */
int orc_hpd_inverse(int N, const cplx *G, cplx *Gi)
{
    cplx *U = malloc(sizeof(cplx) * N * N), *Ui = malloc(sizeof(cplx) * N * N);
    int rc = orc_cholesky_upper(N, G, U);
    if (rc == 0) {
        orc_upper_inverse(N, U, Ui);
        for (int i = 0; i < N; i++)
            for (int j = 0; j < N; j++) {
                cplx s = 0.0;
                for (int k = 0; k < N; k++) s += Ui[i * N + k] * conj(Ui[j * N + k]);
                Gi[i * N + j] = s;
            }
    }
    free(U);
    free(Ui);
    return rc;
}

/* thin QR, PAPER.md:164-172 (Algorithm 2): H = Z^dag Z ; R^dag R = H ; Q = Z R^-1.
 * Z (L x N, column-major) is overwritten by Q; Q R = Z is solved column by column
 * (q_j = (z_j - sum_{i<j} q_i R_ij) / R_jj). */
int orc_thin_qr(long L, int N, cplx *Z, cplx *R)
{
    cplx *H = malloc(sizeof(cplx) * N * N);
    orc_gram(L, N, Z, Z, H);
    hermitise(N, H);
    int rc = orc_cholesky_upper(N, H, R);
    free(H);
    if (rc) return rc;
    for (int j = 0; j < N; j++) {
        cplx *qj = Z + (long)j * L;
        for (int i = 0; i < j; i++) {
            const cplx *qi = Z + (long)i * L;
            cplx r = R[i * N + j];
#pragma omp parallel for schedule(static)
            for (long k = 0; k < L; k++) qj[k] -= qi[k] * r;
        }
        double inv = 1.0 / creal(R[j * N + j]);
#pragma omp parallel for schedule(static)
        for (long k = 0; k < L; k++) qj[k] *= inv;
    }
    return 0;
}

/* thin QR by TWO Cholesky-QR passes (the remedy of the paper's refs [43, 44], PAPER.md:184-186 footnote, for the
 * squared condition number of Algorithm 2; U24):
 *   pass 1  H = Z^dag Z ; R1^dag R1 = H, or = H + s 1 with s = 1e-12 max_i H_ii when a pivot of H is not positive
 *           ("shifted" Cholesky QR) ; Q1 = Z R1^-1
 *   pass 2  H2 = Q1^dag Q1 ; R2^dag R2 = H2 ; Q = Q1 R2^-1 ; R = R2 R1
 * The factorisation Z = Q R with R upper triangular and a positive diagonal is unique, so for a well conditioned Z this
 * returns what orc_thin_qr returns up to rounding.  -5 if a pivot of pass 2 is below 1e-8 (Z has no full rank to
 * working precision). */
int orc_thin_qr2(long L, int N, cplx *Z, cplx *R)
{
    cplx *H = malloc(sizeof(cplx) * N * N), *R1 = malloc(sizeof(cplx) * N * N), *R2 = malloc(sizeof(cplx) * N * N);
    int rc;
    orc_gram(L, N, Z, Z, H);
    hermitise(N, H);
    rc = orc_cholesky_upper(N, H, R1);
    if (rc) {
        double hmax = 0.0;
        for (int i = 0; i < N; i++) hmax = fmax(hmax, creal(H[i * N + i]));
        for (int i = 0; i < N; i++) H[i * N + i] += 1e-12 * hmax;
        rc = orc_cholesky_upper(N, H, R1);
    }
    free(H);
    if (rc) { free(R1); free(R2); return rc; }
    for (int pass = 0; pass < 2; pass++) {
        const cplx *Rp = pass == 0 ? R1 : R2;
        if (pass == 1) {
            cplx *H2 = malloc(sizeof(cplx) * N * N);
            orc_gram(L, N, Z, Z, H2);
            hermitise(N, H2);
            rc = orc_cholesky_upper(N, H2, R2);
            /* after pass 1 the columns have norm <= 1 and are orthonormal up to kappa(Z)^2 u (or up to the shift: a direction
             * with singular value sigma keeps sigma^2 / (sigma^2 + s)); a pivot below 1e-8 means Z has no full rank to
             * working precision (its image under pass 1 is rounding noise) */
            for (int j = 0; j < N && !rc; j++)
                if (!(creal(R2[j * N + j]) * creal(R2[j * N + j]) > 1e-8)) rc = -5;
            free(H2);
            if (rc) { free(R1); free(R2); return rc; }
        }
        for (int j = 0; j < N; j++) { /* Z <- Z Rp^-1, column by column as in orc_thin_qr */
            cplx *qj = Z + (long)j * L;
            for (int i = 0; i < j; i++) {
                const cplx *qi = Z + (long)i * L;
                cplx r = Rp[i * N + j];
#pragma omp parallel for schedule(static)
                for (long k = 0; k < L; k++) qj[k] -= qi[k] * r;
            }
            double inv = 1.0 / creal(Rp[j * N + j]);
#pragma omp parallel for schedule(static)
            for (long k = 0; k < L; k++) qj[k] *= inv;
        }
    }
    matmul(N, R2, R1, R);
    free(R1); free(R2);
    return 0;
}

/* ------------------------------------------------------------------------------ solvers */

static double norm2(long n, const cplx *v)
{
    double s = 0.0;
    for (long i = 0; i < n; i++) s += creal(v[i]) * creal(v[i]) + cimag(v[i]) * cimag(v[i]);
    return s;
}

static cplx cdot(long n, const cplx *a, const cplx *b)
{
    cplx s = 0.0;
    for (long i = 0; i < n; i++) s += conj(a[i]) * b[i];
    return s;
}

/* Conjugate gradients on M x = b for one rhs (ref. [40] of the paper).
 * x holds the initial guess on entry.  hist (may be NULL) receives the relative iterated
 * residual after every iteration, hist[0] = initial.  Returns 0, or -6 at maxiter.
 * iteration count = number of applications of M inside the loop. */
int orc_cg(const int D[4], const cplx *fat, const cplx *lng, double mass, const cplx *b, cplx *x,
           double tol, int maxiter, int *iters, double *hist)
{
    if (!dims_ok(D)) return -1;
    long L = (long)D[0] * D[1] * D[2] * D[3] / 2 * 3;
    cplx *r = malloc(sizeof(cplx) * L), *p = malloc(sizeof(cplx) * L);
    cplx *q = malloc(sizeof(cplx) * L), *t = malloc(sizeof(cplx) * L);
    double bb = norm2(L, b);
    orc_apply_M(D, fat, lng, mass, 1, x, r, t);
    for (long k = 0; k < L; k++) r[k] = b[k] - r[k];
    memcpy(p, r, sizeof(cplx) * L);
    double rho = norm2(L, r);
    int it = 0, rc = -6;
    if (hist) hist[0] = sqrt(rho / bb);
    if (sqrt(rho / bb) <= tol) rc = 0;
    while (rc != 0 && it < maxiter) {
        orc_apply_M(D, fat, lng, mass, 1, p, q, t);
        it++;
        double alpha = rho / creal(cdot(L, p, q));
        for (long k = 0; k < L; k++) x[k] += alpha * p[k];
        for (long k = 0; k < L; k++) r[k] -= alpha * q[k];
        double rho1 = norm2(L, r);
        if (hist) hist[it] = sqrt(rho1 / bb);
        if (sqrt(rho1 / bb) <= tol) { rc = 0; break; }
        double bet = rho1 / rho;
        for (long k = 0; k < L; k++) p[k] = r[k] + bet * p[k];
        rho = rho1;
    }
    *iters = it;
    free(r); free(p); free(q); free(t);
    return rc;
}

static double max_relres_from_C(int N, const cplx *C, const double *bnorm)
{
    /* ||R[:,i]||^2 = sum_j |C_ji|^2 : column i of C (PAPER.md:208 with the index fix U11) */
    double m = 0.0;
    for (int i = 0; i < N; i++) {
        double s = 0.0;
        for (int j = 0; j < N; j++) s += creal(C[j * N + i] * conj(C[j * N + i]));
        double r = sqrt(s) / bnorm[i];
        if (r > m) m = r;
    }
    return m;
}

/* storage rounding to fp32 and back (mixed-precision emulation, U13) */
static void round_f32(long n, cplx *v)
{
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; i++) v[i] = (double)(float)creal(v[i]) + I * (double)(float)cimag(v[i]);
}

/* blockCGrQ, PAPER.md:113-138 (Algorithm 1) in the reconstruction U7, with optional block
 * reliable updates, PAPER.md:190-210 (Algorithm 3) in the reading U12-U14.
 *
 *   l.3  R = B - M X        l.4  Q C = R (thin QR)     l.5  S = I      l.6  P = 0
 *   l.7  while max_i ||C[:,i]|| / ||b_i|| > tol:
 *   l.8     P = Q + P S^dag
 *   l.9     beta = (P^dag M P)^-1
 *   l.10    X = X + P beta C
 *   l.11    Q S = Q - (M P) beta   (thin QR)
 *   l.12    C = S C
 *
 * mixed = 0: everything fp64, delta ignored, converged on the iterated residual (U10).
 * mixed = 1: P, Q, MP, the odd temporary and the inner operator's links are rounded to fp32
 *            after every step that writes them; after l.12, with r = max relative iterated
 *            residual: if r < delta * r_last or r <= tol, do Algorithm 3:
 *              Y += X ; X = 0 ; R = B - M Y (fp64 links) ; Qhat C_new = R ;
 *              S = C_new C_prev^-1, C_prev = C before this iteration's l.12 ; C = C_new.
 *            Converged only on a residual computed by an update (U14).  Result in X (= Y + X).
 * hist (may be NULL): max relative iterated residual, hist[0] initial, hist[it] after it.
 * trace_G / trace_C (may be NULL): G = P^dag M P and C (after l.12) of the first `ntrace`
 * iterations, N*N each, for comparing intermediates (U16).
 * trace_QP (may be NULL): Q^dag P right after l.8 of the first `ntrace` iterations, Q being the
 * block that entered l.8 ("Q_old" of PAPER.md:210, whose identity (Q_old)^dag P = 1 pins the
 * driver, with and without reliable updates).  A trace only: no arithmetic of the solve uses it.
 * Returns 0, -5 on a Cholesky breakdown (U15), -6 at maxiter. */
static int block_cg_impl(const int D[4], const cplx *fat, const cplx *lng, double mass, int N,
                         const cplx *B, cplx *X, double tol, int maxiter, int mixed, double delta,
                         int *iters, int *nupdates, double *hist, int ntrace, cplx *trace_G,
                         cplx *trace_C, cplx *trace_QP, int reorth)
{
    int (*const thin_qr)(long, int, cplx *, cplx *) = reorth ? orc_thin_qr2 : orc_thin_qr;
    if (!dims_ok(D) || N < 1) return -1;
    long V = (long)D[0] * D[1] * D[2] * D[3], Vh = V / 2, L = 3 * Vh, n = L * N;
    size_t nn = sizeof(cplx) * N * N;
    cplx *Q = malloc(sizeof(cplx) * n), *P = calloc(n, sizeof(cplx)), *AP = malloc(sizeof(cplx) * n);
    cplx *T = malloc(sizeof(cplx) * n), *Pn = malloc(sizeof(cplx) * n);
    cplx *Y = NULL, *fat32 = NULL, *lng32 = NULL;
    cplx *C = malloc(nn), *S = malloc(nn), *G = malloc(nn), *beta = malloc(nn), *W = malloc(nn);
    cplx *Sd = malloc(nn), *Cprev = malloc(nn), *tmp = malloc(nn), *Ci = malloc(nn);
    double *bnorm = malloc(sizeof(double) * N);
    const cplx *fin = fat, *lin = lng; /* links of the inner operator */
    int rc = -6, it = 0, nup = 0;

    for (int i = 0; i < N; i++) bnorm[i] = sqrt(norm2(L, B + (long)i * L));
    if (mixed) {
        fat32 = malloc(sizeof(cplx) * 36 * V);
        lng32 = malloc(sizeof(cplx) * 36 * V);
        memcpy(fat32, fat, sizeof(cplx) * 36 * V);
        memcpy(lng32, lng, sizeof(cplx) * 36 * V);
        round_f32(36 * V, fat32);
        round_f32(36 * V, lng32);
        fin = fat32;
        lin = lng32;
        Y = malloc(sizeof(cplx) * n);
        memcpy(Y, X, sizeof(cplx) * n);          /* Y accumulates, X restarts from 0 */
        memset(X, 0, sizeof(cplx) * n);
        orc_apply_M(D, fat, lng, mass, N, Y, Q, T); /* l.3 with the fp64 operator */
    } else {
        orc_apply_M(D, fat, lng, mass, N, X, Q, T); /* l.3 */
    }
    for (long k = 0; k < n; k++) Q[k] = B[k] - Q[k];
    if (thin_qr(L, N, Q, C)) { rc = -5; goto done; } /* l.4 */
    if (mixed) round_f32(n, Q);
    memset(S, 0, nn);
    for (int i = 0; i < N; i++) S[i * N + i] = 1.0; /* l.5 ; P = 0 from calloc (l.6) */
    double r = max_relres_from_C(N, C, bnorm), r_last = r;
    if (hist) hist[0] = r;
    if (r <= tol) rc = 0;

    while (rc == -6 && it < maxiter) {
        /* l.8  P = Q + P S^dag */
        for (int i = 0; i < N; i++)
            for (int j = 0; j < N; j++) Sd[i * N + j] = conj(S[j * N + i]);
        memcpy(Pn, Q, sizeof(cplx) * n);
        orc_block_axpy(L, N, Sd, P, Pn);
        memcpy(P, Pn, sizeof(cplx) * n);
        if (mixed) round_f32(n, P);
        if (it < ntrace && trace_QP) orc_gram(L, N, Q, P, trace_QP + (long)it * N * N);
        /* l.9  beta = (P^dag M P)^-1 */
        orc_apply_M(D, fin, lin, mass, N, P, AP, T);
        if (mixed) round_f32(n, AP);
        it++;
        orc_gram(L, N, P, AP, G);
        hermitise(N, G);
        if (it <= ntrace && trace_G) memcpy(trace_G + (long)(it - 1) * N * N, G, nn);
        if (orc_hpd_inverse(N, G, beta)) { rc = -5; break; }
        /* l.10 X = X + P beta C */
        matmul(N, beta, C, W);
        orc_block_axpy(L, N, W, P, X);
        /* l.11 Q S = Q - (M P) beta */
        for (int i = 0; i < N * N; i++) tmp[i] = -beta[i];
        orc_block_axpy(L, N, tmp, AP, Q);
        if (thin_qr(L, N, Q, S)) { rc = -5; break; }
        if (mixed) round_f32(n, Q);
        /* l.12 C = S C */
        memcpy(Cprev, C, nn);
        matmul(N, S, Cprev, C);
        if (it <= ntrace && trace_C) memcpy(trace_C + (long)(it - 1) * N * N, C, nn);
        r = max_relres_from_C(N, C, bnorm);
        if (!mixed) {
            if (hist) hist[it] = r;
            if (r <= tol) rc = 0;
            continue;
        }
        if (r < delta * r_last || r <= tol) { /* Algorithm 3 */
            for (long k = 0; k < n; k++) Y[k] += X[k];           /* l.2 */
            memset(X, 0, sizeof(cplx) * n);                      /* l.3 */
            orc_apply_M(D, fat, lng, mass, N, Y, Q, T);          /* l.4, fp64 operator */
            for (long k = 0; k < n; k++) Q[k] = B[k] - Q[k];
            if (thin_qr(L, N, Q, C)) { rc = -5; break; }      /* l.5, C = C_new */
            round_f32(n, Q);
            orc_upper_inverse(N, Cprev, Ci);                     /* l.6 S = C_new C_prev^-1 */
            matmul(N, C, Ci, S);
            nup++;
            r = max_relres_from_C(N, C, bnorm);
            r_last = r;
            if (r <= tol) rc = 0;
        }
        if (hist) hist[it] = r;
    }
    if (mixed)
        for (long k = 0; k < n; k++) X[k] += Y[k];
done:
    *iters = it;
    if (nupdates) *nupdates = nup;
    free(Q); free(P); free(AP); free(T); free(Pn); free(Y); free(fat32); free(lng32);
    free(C); free(S); free(G); free(beta); free(W); free(Sd); free(Cprev); free(tmp); free(Ci);
    free(bnorm);
    return rc;
}

int orc_block_cg(const int D[4], const cplx *fat, const cplx *lng, double mass, int N,
                 const cplx *B, cplx *X, double tol, int maxiter, int mixed, double delta,
                 int *iters, int *nupdates, double *hist, int ntrace, cplx *trace_G,
                 cplx *trace_C, cplx *trace_QP)
{
    return block_cg_impl(D, fat, lng, mass, N, B, X, tol, maxiter, mixed, delta, iters, nupdates, hist, ntrace, trace_G,
                         trace_C, trace_QP, 0);
}

/* the same with every thin QR (l.4, l.11, Alg. 3 l.5) done by orc_thin_qr2: the comparison solver for blocks whose
 * residuals are ill conditioned (nearly dependent right-hand sides), where Algorithm 2 as printed breaks down */
int orc_block_cg_reorth(const int D[4], const cplx *fat, const cplx *lng, double mass, int N,
                        const cplx *B, cplx *X, double tol, int maxiter, int mixed, double delta,
                        int *iters, int *nupdates, double *hist, int ntrace, cplx *trace_G,
                        cplx *trace_C, cplx *trace_QP)
{
    return block_cg_impl(D, fat, lng, mass, N, B, X, tol, maxiter, mixed, delta, iters, nupdates, hist, ntrace, trace_G,
                         trace_C, trace_QP, 1);
}

/* true relative residuals ||b_i - M x_i|| / ||b_i|| */
int orc_true_relres(const int D[4], const cplx *fat, const cplx *lng, double mass, int N,
                    const cplx *B, const cplx *X, double *relres)
{
    if (!dims_ok(D) || N < 1) return -1;
    long L = (long)D[0] * D[1] * D[2] * D[3] / 2 * 3, n = L * N;
    cplx *R = malloc(sizeof(cplx) * n), *T = malloc(sizeof(cplx) * n);
    orc_apply_M(D, fat, lng, mass, N, X, R, T);
    for (int i = 0; i < N; i++) {
        cplx *ri = R + (long)i * L;
        const cplx *bi = B + (long)i * L;
        for (long k = 0; k < L; k++) ri[k] = bi[k] - ri[k];
        relres[i] = sqrt(norm2(L, ri) / norm2(L, bi));
    }
    free(R);
    free(T);
    return 0;
}
