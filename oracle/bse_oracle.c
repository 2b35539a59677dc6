/*
 * oracle/bse_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU implementation of what the hot path of arXiv 2504.10096
 * computes (structured BSE operator x block of vectors, basis orthogonalisation, Lanczos
 * eigenpairs).  Written from PAPER.md only; shares no code with the CUDA library.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Conventions: all matrices are DENSE, ROW-MAJOR, complex128 (C99 `double complex`);
 * vector blocks X, Y are ROW-MAJOR n_rows x k.  Accumulation is in `long double` so that the
 * oracle's own rounding (~N 2^-64) is negligible against the 1e-12 parity budget.
 *
 * Pins (tests/test_oracle_*.py): identity / diagonal / unit-impulse operators, numpy matmul of
 * the unpacked operator, the paper's identity Q^H H Q = -i J M_r (Eq. 2-3), prescribed spectra
 * Q diag(lambda) Q^H, +-omega pairing, omega^2 = eig((R-C)(R+C)) for real R, C,
 * sum omega^2 = |R|_F^2 - |C|_F^2, residuals.  The paper prints no eigenvalue, residual or
 * vector of its own: parity against the paper's own outputs is UNPINNED.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>

typedef double complex zc;
typedef long double ld;

/* ------------------------------------------------------------------------------------------
 * Operator entries.  PAPER.md:18 (Eq. 1): H = [[R, C], [-C^dagger, -A]], R = R^dagger.
 * optical case A = R^*, C = C^T.  PAPER.md:24: TDA sets C = 0 => R x = w x.
 * Only the LOWER triangle (j <= i) of the stored R and C is read; the rest follows from
 * R_ij = conj(R_ji) and C_ij = C_ji.  The diagonal of R is real (imaginary part ignored).
 * ------------------------------------------------------------------------------------------ */
static inline zc R_at(const zc *R, int64_t N, int64_t i, int64_t j)
{
    if (i == j) return creal(R[i * N + i]);
    return (j < i) ? R[i * N + j] : conj(R[j * N + i]);
}
static inline zc C_at(const zc *C, int64_t N, int64_t i, int64_t j)
{
    return (j <= i) ? C[i * N + j] : C[j * N + i];
}
/* entry (i, j) of the full 2N x 2N operator of Eq. (1) with A = R^*, C^dagger = conj(C^T) */
static inline zc H_at(const zc *R, const zc *C, int64_t N, int64_t i, int64_t j)
{
    if (i < N) {
        return (j < N) ? R_at(R, N, i, j) : C_at(C, N, i, j - N);
    } else {
        int64_t ii = i - N;
        if (j < N) return -conj(C_at(C, N, j, ii));          /* -(C^dagger)_{ii,j} = -conj(C_{j,ii}) */
        return -conj(R_at(R, N, ii, j - N));                  /* -A = -R^*                            */
    }
}

/* Y = R X, rows r0 <= i < r1 of Y only (TDA).  Triple loop. */
void orc_apply_tda_rows(int64_t N, int64_t k, const zc *R, const zc *X, zc *Y, int64_t r0, int64_t r1)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t i = r0; i < r1; ++i) {
        for (int64_t c = 0; c < k; ++c) {
            ld ar = 0.0L, ai = 0.0L;
            for (int64_t j = 0; j < N; ++j) {
                zc h = R_at(R, N, i, j);
                zc x = X[j * k + c];
                ar += (ld)creal(h) * (ld)creal(x) - (ld)cimag(h) * (ld)cimag(x);
                ai += (ld)creal(h) * (ld)cimag(x) + (ld)cimag(h) * (ld)creal(x);
            }
            Y[i * k + c] = (double)ar + I * (double)ai;
        }
    }
}
void orc_apply_tda(int64_t N, int64_t k, const zc *R, const zc *X, zc *Y)
{
    orc_apply_tda_rows(N, k, R, X, Y, 0, N);
}

/* [Y1;Y2] = H [X1;X2], X and Y are 2N x k (Eq. 1).  Rows r0 <= i < r1 only. */
void orc_apply_full_rows(int64_t N, int64_t k, const zc *R, const zc *C, const zc *X, zc *Y,
                         int64_t r0, int64_t r1)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t i = r0; i < r1; ++i) {
        for (int64_t c = 0; c < k; ++c) {
            ld ar = 0.0L, ai = 0.0L;
            for (int64_t j = 0; j < 2 * N; ++j) {
                zc h = H_at(R, C, N, i, j);
                zc x = X[j * k + c];
                ar += (ld)creal(h) * (ld)creal(x) - (ld)cimag(h) * (ld)cimag(x);
                ai += (ld)creal(h) * (ld)cimag(x) + (ld)cimag(h) * (ld)creal(x);
            }
            Y[i * k + c] = (double)ar + I * (double)ai;
        }
    }
}
void orc_apply_full(int64_t N, int64_t k, const zc *R, const zc *C, const zc *X, zc *Y)
{
    orc_apply_full_rows(N, k, R, C, X, Y, 0, 2 * N);
}

/* Structured half-apply (reading S4, derived from Eq. 1): for u = [x; sign*conj(x)],
 * the upper half of H u is  R x + sign * C conj(x).  sign=+1: P(x); sign=-1: M(x). */
void orc_apply_half(int64_t N, int64_t k, int sign, const zc *R, const zc *C, const zc *X, zc *Y)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t i = 0; i < N; ++i) {
        for (int64_t c = 0; c < k; ++c) {
            ld ar = 0.0L, ai = 0.0L;
            for (int64_t j = 0; j < N; ++j) {
                zc r = R_at(R, N, i, j);
                zc cc = C_at(C, N, i, j);
                zc x = X[j * k + c];
                zc xc = conj(x);
                ar += (ld)creal(r) * (ld)creal(x) - (ld)cimag(r) * (ld)cimag(x);
                ai += (ld)creal(r) * (ld)cimag(x) + (ld)cimag(r) * (ld)creal(x);
                ar += sign * ((ld)creal(cc) * (ld)creal(xc) - (ld)cimag(cc) * (ld)cimag(xc));
                ai += sign * ((ld)creal(cc) * (ld)cimag(xc) + (ld)cimag(cc) * (ld)creal(xc));
            }
            Y[i * k + c] = (double)ar + I * (double)ai;
        }
    }
}

/* Generic dense row panel times block: Y (nr x k) = Hrows (nr x n) X (n x k).  Used for sampled-row
 * parity at sizes where the dense operator does not fit the host (rows come from bse_inputs). */
void orc_rows_times_block(int64_t nr, int64_t n, int64_t k, const zc *Hrows, const zc *X, zc *Y)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < nr; ++i) {
        for (int64_t c = 0; c < k; ++c) {
            ld ar = 0.0L, ai = 0.0L;
            for (int64_t j = 0; j < n; ++j) {
                zc h = Hrows[i * n + j];
                zc x = X[j * k + c];
                ar += (ld)creal(h) * (ld)creal(x) - (ld)cimag(h) * (ld)cimag(x);
                ai += (ld)creal(h) * (ld)cimag(x) + (ld)cimag(h) * (ld)creal(x);
            }
            Y[i * k + c] = (double)ar + I * (double)ai;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Cyclic Jacobi for a Hermitian n x n matrix (textbook; north_star asks for it at tiny sizes).
 * A (row-major) is overwritten; w gets the eigenvalues ascending, V (row-major, columns are
 * eigenvectors) the eigenvectors.  Returns the number of sweeps, or -1 if not converged.
 * Rotation: a_pq = |a_pq| e^{i phi}; U = D J, D = diag(1, e^{-i phi}), J = [[c, s], [-s, c]],
 * t = sgn(th)/(|th| + sqrt(th^2+1)), th = (a_qq - a_pp) / (2 |a_pq|);  A <- U^H A U.
 * ------------------------------------------------------------------------------------------ */
int orc_jacobi_herm(int64_t n, zc *A, double *w, zc *V)
{
    for (int64_t i = 0; i < n; ++i)
        for (int64_t j = 0; j < n; ++j) V[i * n + j] = (i == j) ? 1.0 : 0.0;
    double fro = 0.0;
    for (int64_t i = 0; i < n * n; ++i) fro += creal(A[i]) * creal(A[i]) + cimag(A[i]) * cimag(A[i]);
    fro = sqrt(fro);
    int sweep;
    int converged = 0;
    for (sweep = 0; sweep < 100; ++sweep) {
        double off = 0.0;
        for (int64_t i = 0; i < n; ++i)
            for (int64_t j = 0; j < n; ++j)
                if (i != j) off += creal(A[i * n + j]) * creal(A[i * n + j]) + cimag(A[i * n + j]) * cimag(A[i * n + j]);
        if (sqrt(off) <= 1e-15 * fro || fro == 0.0) { converged = 1; break; }
        for (int64_t p = 0; p < n - 1; ++p) {
            for (int64_t q = p + 1; q < n; ++q) {
                zc apq = A[p * n + q];
                double g = cabs(apq);
                if (g == 0.0) continue;
                double app = creal(A[p * n + p]), aqq = creal(A[q * n + q]);
                if (g < 1e-300) continue;
                double th = (aqq - app) / (2.0 * g);
                double t = ((th >= 0.0) ? 1.0 : -1.0) / (fabs(th) + sqrt(th * th + 1.0));
                double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
                zc e = conj(apq) / g;                       /* e^{-i phi} */
                zc Upp = c, Upq = s, Uqp = -s * e, Uqq = c * e;
                for (int64_t r = 0; r < n; ++r) {           /* A <- A U */
                    zc arp = A[r * n + p], arq = A[r * n + q];
                    A[r * n + p] = arp * Upp + arq * Uqp;
                    A[r * n + q] = arp * Upq + arq * Uqq;
                }
                for (int64_t r = 0; r < n; ++r) {           /* A <- U^H A */
                    zc apr = A[p * n + r], aqr = A[q * n + r];
                    A[p * n + r] = conj(Upp) * apr + conj(Uqp) * aqr;
                    A[q * n + r] = conj(Upq) * apr + conj(Uqq) * aqr;
                }
                A[p * n + q] = 0.0; A[q * n + p] = 0.0;
                A[p * n + p] = creal(A[p * n + p]); A[q * n + q] = creal(A[q * n + q]);
                for (int64_t r = 0; r < n; ++r) {           /* V <- V U */
                    zc vrp = V[r * n + p], vrq = V[r * n + q];
                    V[r * n + p] = vrp * Upp + vrq * Uqp;
                    V[r * n + q] = vrp * Upq + vrq * Uqq;
                }
            }
        }
    }
    /* sort ascending (selection sort, swapping eigenvector columns) */
    for (int64_t i = 0; i < n; ++i) w[i] = creal(A[i * n + i]);
    for (int64_t i = 0; i < n - 1; ++i) {
        int64_t m = i;
        for (int64_t j = i + 1; j < n; ++j) if (w[j] < w[m]) m = j;
        if (m != i) {
            double tw = w[i]; w[i] = w[m]; w[m] = tw;
            for (int64_t r = 0; r < n; ++r) { zc tv = V[r * n + i]; V[r * n + i] = V[r * n + m]; V[r * n + m] = tv; }
        }
    }
    return converged ? sweep : -1;
}

/* ------------------------------------------------------------------------------------------
 * The paper's direct route for the full problem, PAPER.md:40-53 (section 2.1, Eq. 2-4):
 *   M_r = [[Re(R+C), Im(R-C)], [-Im(R+C), Re(R-C)]]          (Eq. 3)
 *   M_r = L L^T (real Cholesky; fails iff M_r -- equivalently Omega -- is not positive definite)
 *   W = L^T J L,  J = [[0, I], [-I, 0]]  (Eq. 2);  -iW Hermitian with the eigenvalues of H
 *   eigenvector of H:  v = Q L^-T z,   Q = (1/sqrt 2) [[I, -iI], [I, iI]]  (Eq. 2, reading S1)
 * Outputs: Mr (2N x 2N real, row-major; may be NULL), omega (2N ascending: -w ... +w),
 * V (2N x 2N complex row-major, columns = right eigenvectors of H; may be NULL).
 * Returns 0, or 1 if the Cholesky factorisation met a non-positive pivot, or 2 if Jacobi failed.
 * ------------------------------------------------------------------------------------------ */
void orc_build_Mr(int64_t N, const zc *R, const zc *C, double *Mr)
{
    int64_t n2 = 2 * N;
    for (int64_t i = 0; i < N; ++i)
        for (int64_t j = 0; j < N; ++j) {
            zc r = R_at(R, N, i, j), c = C_at(C, N, i, j);
            Mr[i * n2 + j] = creal(r + c);
            Mr[i * n2 + (j + N)] = cimag(r - c);
            Mr[(i + N) * n2 + j] = -cimag(r + c);
            Mr[(i + N) * n2 + (j + N)] = creal(r - c);
        }
}

int orc_cholesky_real(int64_t n, const double *A, double *L)
{
    memset(L, 0, sizeof(double) * n * n);
    for (int64_t j = 0; j < n; ++j) {
        ld d = A[j * n + j];
        for (int64_t p = 0; p < j; ++p) d -= (ld)L[j * n + p] * (ld)L[j * n + p];
        if (!(d > 0.0L)) return 1;
        double ljj = sqrt((double)d);
        L[j * n + j] = ljj;
        for (int64_t i = j + 1; i < n; ++i) {
            ld s = A[i * n + j];
            for (int64_t p = 0; p < j; ++p) s -= (ld)L[i * n + p] * (ld)L[j * n + p];
            L[i * n + j] = (double)(s / ljj);
        }
    }
    return 0;
}

int orc_bse_direct(int64_t N, const zc *R, const zc *C, double *Mr_out, double *omega, zc *V)
{
    int64_t n2 = 2 * N;
    double *Mr = (double *)malloc(sizeof(double) * n2 * n2);
    double *L = (double *)malloc(sizeof(double) * n2 * n2);
    double *JL = (double *)malloc(sizeof(double) * n2 * n2);
    zc *Hm = (zc *)malloc(sizeof(zc) * n2 * n2);
    zc *Z = (zc *)malloc(sizeof(zc) * n2 * n2);
    int rc = 0;
    orc_build_Mr(N, R, C, Mr);
    if (Mr_out) memcpy(Mr_out, Mr, sizeof(double) * n2 * n2);
    if (orc_cholesky_real(n2, Mr, L)) { rc = 1; goto done; }
    /* JL = J L : rows 0..N-1 of JL are rows N..2N-1 of L; rows N..2N-1 are minus rows 0..N-1 */
    for (int64_t i = 0; i < N; ++i)
        for (int64_t j = 0; j < n2; ++j) {
            JL[i * n2 + j] = L[(i + N) * n2 + j];
            JL[(i + N) * n2 + j] = -L[i * n2 + j];
        }
    /* W = L^T (J L);  Hm = -i W */
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n2; ++i)
        for (int64_t j = 0; j < n2; ++j) {
            ld s = 0.0L;
            for (int64_t p = 0; p < n2; ++p) s += (ld)L[p * n2 + i] * (ld)JL[p * n2 + j];
            Hm[i * n2 + j] = -I * (double)s;
        }
    /* enforce exact Hermitian symmetry of -iW against rounding (W is skew by construction) */
    for (int64_t i = 0; i < n2; ++i) {
        Hm[i * n2 + i] = 0.0;
        for (int64_t j = i + 1; j < n2; ++j) {
            zc a = 0.5 * (Hm[i * n2 + j] + conj(Hm[j * n2 + i]));
            Hm[i * n2 + j] = a; Hm[j * n2 + i] = conj(a);
        }
    }
    if (orc_jacobi_herm(n2, Hm, omega, Z) < 0) { rc = 2; goto done; }
    if (V) {
        /* vbar = L^-T z (back substitution with the upper triangular L^T), then v = Q vbar */
        double isq2 = 1.0 / sqrt(2.0);
        zc *vb = (zc *)malloc(sizeof(zc) * n2);
        for (int64_t c = 0; c < n2; ++c) {
            for (int64_t i = n2 - 1; i >= 0; --i) {
                zc s = Z[i * n2 + c];
                for (int64_t p = i + 1; p < n2; ++p) s -= L[p * n2 + i] * vb[p];
                vb[i] = s / L[i * n2 + i];
            }
            for (int64_t i = 0; i < N; ++i) {
                V[i * n2 + c] = isq2 * (vb[i] - I * vb[i + N]);
                V[(i + N) * n2 + c] = isq2 * (vb[i] + I * vb[i + N]);
            }
        }
        free(vb);
    }
done:
    free(Mr); free(L); free(JL); free(Hm); free(Z);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Real symmetric tridiagonal eigenproblem by the implicit-shift QR iteration with Wilkinson's shift
 * (textbook: Golub & Van Loan, "Matrix Computations", symmetric QR step on a tridiagonal matrix).
 * 8(c) step 4 allows "the oracle's own tridiagonal QL" for the projected matrix T of the Lanczos routines
 * below ("projected into a smaller structured problem"); the dense Jacobi routine above costs
 * O(m^3) per sweep and took more than an hour at m = 1500.
 * In:  m, d[0..m) diagonal, e[0..m-1) off-diagonal (both untouched).
 * Out: w[0..m) eigenvalues ascending; Z (m x m row-major, may be NULL) with eigenvector i in COLUMN i.
 * One step on the unreduced block lo..hi: mu = Wilkinson shift from the trailing 2 x 2 block; x = d_lo - mu,
 * z = e_lo; for k = lo..hi-1: c = x/r, s = z/r, r = hypot(x, z), G = [[c, -s], [s, c]] acting on (k, k+1),
 * T <- G^T T G (which moves the bulge z = s e_{k+1} one position down), Z <- Z G, x = e_k.
 * Returns 0, or 1 if some eigenvalue needed more than 60 steps.
 * Pins (tests/test_oracle_eig.py): the Toeplitz matrix tridiag(b, a, b) with eigenvalues a + 2 b cos(j pi/(m+1)) and
 * eigenvectors sin(i j pi/(m+1)); the Jacobi routine on random tridiagonals; Z^T T Z = diag(w), Z^T Z = I.
 * ------------------------------------------------------------------------------------------ */
int orc_tridiag_ql(int64_t m, const double *d_in, const double *e_in, double *w, double *Z)
{
    double *d = (double *)malloc(sizeof(double) * m), *e = (double *)calloc(m, sizeof(double));
    const double eps = 2.220446049250313e-16;
    int rc = 0;
    for (int64_t i = 0; i < m; ++i) d[i] = d_in[i];
    for (int64_t i = 0; i + 1 < m; ++i) e[i] = e_in[i];
    if (Z) for (int64_t i = 0; i < m; ++i) for (int64_t j = 0; j < m; ++j) Z[i * m + j] = (i == j) ? 1.0 : 0.0;
    int64_t hi = m - 1;
    int64_t steps = 0;
    while (hi > 0) {
        if (fabs(e[hi - 1]) <= eps * (fabs(d[hi - 1]) + fabs(d[hi]))) { e[hi - 1] = 0.0; --hi; steps = 0; continue; }
        if (++steps > 60) { rc = 1; break; }
        int64_t lo = hi - 1;
        while (lo > 0 && fabs(e[lo - 1]) > eps * (fabs(d[lo - 1]) + fabs(d[lo]))) --lo;
        double delta = 0.5 * (d[hi - 1] - d[hi]), b2 = e[hi - 1] * e[hi - 1];
        double mu = d[hi] - b2 / (delta + ((delta >= 0.0) ? 1.0 : -1.0) * sqrt(delta * delta + b2));
        double x = d[lo] - mu, z = e[lo];
        for (int64_t k = lo; k < hi; ++k) {
            double r = hypot(x, z);
            double c = (r > 0.0) ? x / r : 1.0, s = (r > 0.0) ? z / r : 0.0;
            if (k > lo) e[k - 1] = r;
            double a = d[k], b = e[k], g = d[k + 1];
            d[k] = c * c * a + 2.0 * c * s * b + s * s * g;
            d[k + 1] = s * s * a - 2.0 * c * s * b + c * c * g;
            e[k] = c * s * (g - a) + (c * c - s * s) * b;
            x = e[k];
            if (k + 1 < hi) { z = s * e[k + 1]; e[k + 1] = c * e[k + 1]; }
            if (Z) {                                                  /* Z <- Z G; Z is held transposed while iterating */
                double *zk = Z + k * m, *zk1 = zk + m;
                for (int64_t i = 0; i < m; ++i) {
                    double u = zk[i], v = zk1[i];
                    zk[i] = c * u + s * v;
                    zk1[i] = -s * u + c * v;
                }
            }
        }
    }
    /* sort ascending (selection sort, swapping eigenvectors), then transpose: eigenvector i into column i */
    for (int64_t i = 0; i < m; ++i) w[i] = d[i];
    for (int64_t i = 0; i + 1 < m; ++i) {
        int64_t p = i;
        for (int64_t j = i + 1; j < m; ++j) if (w[j] < w[p]) p = j;
        if (p != i) {
            double t = w[i]; w[i] = w[p]; w[p] = t;
            if (Z) for (int64_t r = 0; r < m; ++r) { double tv = Z[i * m + r]; Z[i * m + r] = Z[p * m + r]; Z[p * m + r] = tv; }
        }
    }
    if (Z)
        for (int64_t i = 0; i < m; ++i)
            for (int64_t j = i + 1; j < m; ++j) { double tv = Z[i * m + j]; Z[i * m + j] = Z[j * m + i]; Z[j * m + i] = tv; }
    free(d); free(e);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Block classical Gram-Schmidt with one reorthogonalisation (new vectors "have to
 * be orthogonalized against the previous ones"), followed by a column-by-column QR of the block.
 * In:  V (N x m, orthonormal columns, row-major), W (N x k row-major).
 * Out: Q (N x k), h (m x k), B (k x k upper triangular, positive real diagonal) with
 *      W = V h + Q B,  V^H Q = 0,  Q^H Q = I.  Returns the numerical rank of the block.
 * ------------------------------------------------------------------------------------------ */
static zc dotc_col(int64_t N, const zc *A, int64_t lda, int64_t ca, const zc *B, int64_t ldb, int64_t cb)
{
    ld sr = 0.0L, si = 0.0L;
    for (int64_t i = 0; i < N; ++i) {
        zc a = A[i * lda + ca], b = B[i * ldb + cb];
        sr += (ld)creal(a) * (ld)creal(b) + (ld)cimag(a) * (ld)cimag(b);
        si += (ld)creal(a) * (ld)cimag(b) - (ld)cimag(a) * (ld)creal(b);
    }
    return (double)sr + I * (double)si;
}

int orc_block_cgs2(int64_t N, int64_t m, int64_t k, const zc *V, const zc *W, zc *Q, zc *h, zc *B)
{
    memcpy(Q, W, sizeof(zc) * N * k);
    for (int64_t i = 0; i < m * k; ++i) h[i] = 0.0;
    for (int64_t i = 0; i < k * k; ++i) B[i] = 0.0;
    zc *c = (zc *)malloc(sizeof(zc) * (m > k ? m : k) * k);
    for (int pass = 0; pass < 2; ++pass) {
        for (int64_t a = 0; a < m; ++a)
            for (int64_t b = 0; b < k; ++b) c[a * k + b] = dotc_col(N, V, m, a, Q, k, b);   /* c = V^H Q */
        for (int64_t i = 0; i < N; ++i)
            for (int64_t b = 0; b < k; ++b) {
                zc s = 0.0;
                for (int64_t a = 0; a < m; ++a) s += V[i * m + a] * c[a * k + b];
                Q[i * k + b] -= s;
            }
        for (int64_t i = 0; i < m * k; ++i) h[i] += c[i];
    }
    int rank = 0;
    double scale = 0.0;
    for (int64_t b = 0; b < k; ++b) { double nb = sqrt(creal(dotc_col(N, W, k, b, W, k, b))); if (nb > scale) scale = nb; }
    for (int64_t b = 0; b < k; ++b) {
        for (int pass = 0; pass < 2; ++pass)
            for (int64_t a = 0; a < b; ++a) {
                zc r = dotc_col(N, Q, k, a, Q, k, b);
                for (int64_t i = 0; i < N; ++i) Q[i * k + b] -= Q[i * k + a] * r;
                B[a * k + b] += r;
            }
        double nb = sqrt(creal(dotc_col(N, Q, k, b, Q, k, b)));
        B[b * k + b] = nb;
        if (nb > 1e-14 * scale && nb > 0.0) {
            ++rank;
            for (int64_t i = 0; i < N; ++i) Q[i * k + b] /= nb;
        } else {
            B[b * k + b] = 0.0;
            for (int64_t i = 0; i < N; ++i) Q[i * k + b] = 0.0;
        }
    }
    free(c);
    return rank;
}

/* ------------------------------------------------------------------------------------------
 * Textbook Lanczos, TDA (Hermitian R), single vector, full reorthogonalisation (classical
 * Gram-Schmidt twice) -- PAPER.md:65-71: vectors generated one by one, each orthogonalised
 * against the previous ones and stored.  No restart (the basis fits at the sizes the oracle runs).
 * The projected tridiagonal T is diagonalised by orc_tridiag_ql every `check` steps.
 * Converged when the nev lowest Ritz pairs have |beta_{m+1} s_{m,i}| <= tol * max|theta|.
 * Out: w (nev ascending), Vec (N x nev row-major), res (nev), returns number of steps (<0: failed).
 * ------------------------------------------------------------------------------------------ */
static double nrm2(int64_t n, const zc *x)
{
    ld s = 0.0L;
    for (int64_t i = 0; i < n; ++i) s += (ld)creal(x[i]) * (ld)creal(x[i]) + (ld)cimag(x[i]) * (ld)cimag(x[i]);
    return sqrt((double)s);
}

int orc_lanczos_tda(int64_t N, const zc *R, int nev, double tol, int maxit, int check, const zc *v0,
                    double *w, zc *Vec, double *res)
{
    if (maxit > N) maxit = (int)N;
    zc *Vb = (zc *)malloc(sizeof(zc) * (size_t)N * (maxit + 1));      /* basis, vector j at Vb + j*N */
    double *alpha = (double *)calloc(maxit + 1, sizeof(double));
    double *beta = (double *)calloc(maxit + 2, sizeof(double));        /* beta[j] couples j-1 and j */
    zc *wv = (zc *)malloc(sizeof(zc) * N);
    double *S = NULL, *th = NULL;
    int m = 0, result = -1;
    double n0 = nrm2(N, v0);
    for (int64_t i = 0; i < N; ++i) Vb[i] = v0[i] / n0;
    for (int j = 0; j < maxit; ++j) {
        orc_apply_tda(N, 1, R, Vb + (size_t)j * N, wv);                  /* w = R v_j */
        ld a = 0.0L;
        for (int64_t i = 0; i < N; ++i) {
            zc v = Vb[(size_t)j * N + i];
            a += (ld)creal(v) * (ld)creal(wv[i]) + (ld)cimag(v) * (ld)cimag(wv[i]);
        }
        alpha[j] = (double)a;
        for (int pass = 0; pass < 2; ++pass)                              /* full reorthogonalisation */
            for (int p = 0; p <= j; ++p) {
                const zc *vp = Vb + (size_t)p * N;
                ld sr = 0.0L, si = 0.0L;
                for (int64_t i = 0; i < N; ++i) {
                    sr += (ld)creal(vp[i]) * (ld)creal(wv[i]) + (ld)cimag(vp[i]) * (ld)cimag(wv[i]);
                    si += (ld)creal(vp[i]) * (ld)cimag(wv[i]) - (ld)cimag(vp[i]) * (ld)creal(wv[i]);
                }
                zc cf = (double)sr + I * (double)si;
                for (int64_t i = 0; i < N; ++i) wv[i] -= cf * vp[i];
            }
        double b = nrm2(N, wv);
        beta[j + 1] = b;
        m = j + 1;
        int last = (m == maxit) || (b <= 1e-300);
        if (b > 1e-300) for (int64_t i = 0; i < N; ++i) Vb[(size_t)(j + 1) * N + i] = wv[i] / b;
        if (m >= nev && (m % check == 0 || last)) {
            S = (double *)realloc(S, sizeof(double) * m * m);
            th = (double *)realloc(th, sizeof(double) * m);
            if (orc_tridiag_ql(m, alpha, beta + 1, th, S)) break;        /* T = tridiag(beta, alpha, beta) */
            double hn = fmax(fabs(th[0]), fabs(th[m - 1]));
            int ok = 1;
            for (int i = 0; i < nev; ++i) {
                res[i] = fabs(b) * fabs(S[(m - 1) * m + i]);
                if (res[i] > tol * hn) ok = 0;
            }
            if (ok || last) {
                for (int i = 0; i < nev; ++i) {
                    w[i] = th[i];
                    for (int64_t r = 0; r < N; ++r) {
                        zc s = 0.0;
                        for (int p = 0; p < m; ++p) s += Vb[(size_t)p * N + r] * S[p * m + i];
                        Vec[r * nev + i] = s;
                    }
                }
                result = ok ? m : -m;
                break;
            }
        }
        if (last) break;
    }
    free(Vb); free(alpha); free(beta); free(wv); free(S); free(th);
    return result;
}

/* ------------------------------------------------------------------------------------------
 * Textbook structure-preserving Lanczos, full mode -- DESIGN.md reading S4 of PAPER.md:65-69
 * (basis with block structure from the start vector, lower blocks implicit, works on H^2, last
 * step recovers +omega and eigenvectors).  With P(x) = R x + C conj(x), M(y) = R y - C conj(y):
 *   x_1 random, p_1 = P(x_1), both scaled by 1/sqrt(Re(x_1^H p_1));
 *   w = M(p_j); alpha_j = Re(p_j^H w); w -= X c, c = Re(PX^H w) (real, twice);
 *   pw = P(w); beta_{j+1} = sqrt(Re(w^H pw)) (<= 0: Omega not positive definite, return -1000000);
 *   x_{j+1} = w / beta, p_{j+1} = pw / beta.   T = tridiag(beta, alpha, beta) real symmetric,
 *   theta_i, s_i its eigenpairs; omega_i = sqrt(theta_i); x = X s_i, y = (PX s_i)/omega_i;
 *   v_i = [x + y; conj(x - y)] sqrt(omega_i)/2   (then v^H Sigma v = 1).
 * Residual estimate |H v - omega v| = sqrt(2) beta_{m+1} |s_{m,i}| |x_{m+1}|_2 / omega * (sqrt(omega)/2).
 *
 * Multiplicity (reading R1): on C^N = R^2N every omega^2 is a DOUBLE eigenvalue of G = M o P, with
 * eigenvectors x and K x, K(x) = i P(x) (K^2 = -G, K commutes with G); both give the same eigenvector of H up to
 * the phase i:  v(K x / omega) = i v(x).  In exact arithmetic the Krylov space of one start vector is P-orthogonal
 * to its image under K, so the iteration sees one copy; the second copy grows out of rounding noise after the first
 * has converged (like the "ghosts" of Lanczos without reorthogonalisation, except that it is a genuine eigenvector
 * of G).  "The nev lowest positive omega of H" therefore counts eigenvectors of H, not Ritz
 * values of G: the leading converged Ritz pairs are turned into vectors v_i of H, each is Sigma-orthogonalised
 * (complex coefficients a^H Sigma v) against the ones already accepted, and it is a NEW eigenpair iff what is left
 * has v^H Sigma v > 1e-4 (a copy leaves the square of the eigenvector error, ~1e-16; a distinct eigenvector of H is
 * exactly Sigma-orthogonal to the others and leaves 1).  The iteration stops when nev eigenpairs have been accepted,
 * every Ritz value below the last of them is converged, and at least `minit` steps were done (minit lets a test run
 * the iteration far past first convergence, where the copies are present).
 * Out: omega (nev ascending), Vec (2N x nev row-major, Sigma-orthonormal), res (nev).  Returns steps (<0: failed).
 * ------------------------------------------------------------------------------------------ */
/* v^H Sigma w for 2N-vectors stored with stride ld (column c of a row-major 2N x ld array) */
static zc sigma_dot(int64_t N, const zc *v, int64_t ldv, const zc *w, int64_t ldw)
{
    ld sr = 0.0L, si = 0.0L;
    for (int64_t i = 0; i < 2 * N; ++i) {
        zc a = v[i * ldv], b = w[i * ldw];
        ld pr = (ld)creal(a) * (ld)creal(b) + (ld)cimag(a) * (ld)cimag(b);
        ld pi = (ld)creal(a) * (ld)cimag(b) - (ld)cimag(a) * (ld)creal(b);
        if (i < N) { sr += pr; si += pi; } else { sr -= pr; si -= pi; }
    }
    return (double)sr + I * (double)si;
}

int orc_lanczos_full(int64_t N, const zc *R, const zc *C, int nev, double tol, int maxit, int check, int minit,
                     const zc *x0, double *omega, zc *Vec, double *res)
{
    if (maxit > 2 * N) maxit = (int)(2 * N);
    zc *Xb = (zc *)malloc(sizeof(zc) * (size_t)N * (maxit + 1));
    zc *Pb = (zc *)malloc(sizeof(zc) * (size_t)N * (maxit + 1));
    double *alpha = (double *)calloc(maxit + 1, sizeof(double));
    double *beta = (double *)calloc(maxit + 2, sizeof(double));
    zc *wv = (zc *)malloc(sizeof(zc) * N), *pw = (zc *)malloc(sizeof(zc) * N);
    zc *cand = (zc *)malloc(sizeof(zc) * 2 * (size_t)N);
    double *S = NULL, *th = NULL;
    int m = 0, result = -1;
    memcpy(Xb, x0, sizeof(zc) * N);
    orc_apply_half(N, 1, +1, R, C, Xb, Pb);
    {
        ld s = 0.0L;
        for (int64_t i = 0; i < N; ++i) s += (ld)creal(Xb[i]) * (ld)creal(Pb[i]) + (ld)cimag(Xb[i]) * (ld)cimag(Pb[i]);
        if (!(s > 0.0L)) { result = -1000000; goto done; }
        double sc = 1.0 / sqrt((double)s);
        for (int64_t i = 0; i < N; ++i) { Xb[i] *= sc; Pb[i] *= sc; }
    }
    for (int j = 0; j < maxit; ++j) {
        const zc *pj = Pb + (size_t)j * N;
        orc_apply_half(N, 1, -1, R, C, pj, wv);                            /* w = M(p_j) */
        ld a = 0.0L;
        for (int64_t i = 0; i < N; ++i) a += (ld)creal(pj[i]) * (ld)creal(wv[i]) + (ld)cimag(pj[i]) * (ld)cimag(wv[i]);
        alpha[j] = (double)a;
        for (int pass = 0; pass < 2; ++pass)
            for (int p = 0; p <= j; ++p) {
                const zc *pp = Pb + (size_t)p * N; const zc *xp = Xb + (size_t)p * N;
                ld s = 0.0L;
                for (int64_t i = 0; i < N; ++i) s += (ld)creal(pp[i]) * (ld)creal(wv[i]) + (ld)cimag(pp[i]) * (ld)cimag(wv[i]);
                double cf = (double)s;                                       /* real coefficient */
                for (int64_t i = 0; i < N; ++i) wv[i] -= cf * xp[i];
            }
        orc_apply_half(N, 1, +1, R, C, wv, pw);                             /* pw = P(w) */
        ld b2 = 0.0L;
        for (int64_t i = 0; i < N; ++i) b2 += (ld)creal(wv[i]) * (ld)creal(pw[i]) + (ld)cimag(wv[i]) * (ld)cimag(pw[i]);
        m = j + 1;
        double xn1 = 0.0;
        double b = 0.0;
        int breakdown = 0;
        if (b2 > 0.0L) {
            b = sqrt((double)b2);
            for (int64_t i = 0; i < N; ++i) { Xb[(size_t)(j + 1) * N + i] = wv[i] / b; Pb[(size_t)(j + 1) * N + i] = pw[i] / b; }
            xn1 = nrm2(N, Xb + (size_t)(j + 1) * N);
        } else if (nrm2(N, wv) > 1e-10) {
            result = -1000000; break;                                         /* not positive definite */
        } else breakdown = 1;
        beta[j + 1] = b;
        int last = (m == maxit) || breakdown;
        if (m >= nev && m >= minit && (m % check == 0 || last)) {
            S = (double *)realloc(S, sizeof(double) * m * m);
            th = (double *)realloc(th, sizeof(double) * m);
            if (orc_tridiag_ql(m, alpha, beta + 1, th, S)) break;            /* T = tridiag(beta, alpha, beta) */
            if (!(th[0] > 0.0)) { result = -1000000; break; }
            double hn = sqrt(fabs(th[m - 1]));
            /* eigenpairs of H from the leading converged Ritz pairs of G (all of them if this is the last chance) */
            int found = 0, all_converged = 1;
            for (int i = 0; i < m && found < nev; ++i) {
                double om = sqrt(th[i]);
                double ri = sqrt(2.0) * b * fabs(S[(m - 1) * m + i]) * xn1 / om * (sqrt(om) / 2.0);
                if (ri > tol * hn) {                                          /* an unconverged Ritz value below the target */
                    if (!last) break;
                    all_converged = 0;
                }
                double sc = sqrt(om) / 2.0;
                for (int64_t r = 0; r < N; ++r) {
                    zc x = 0.0, y = 0.0;
                    for (int p = 0; p < m; ++p) {
                        double s = S[p * m + i];
                        x += Xb[(size_t)p * N + r] * s;
                        y += Pb[(size_t)p * N + r] * s;
                    }
                    y /= om;
                    cand[r] = sc * (x + y);
                    cand[r + N] = sc * conj(x - y);
                }
                for (int pass = 0; pass < 2; ++pass)                          /* Sigma-orthogonalise against the accepted ones */
                    for (int q = 0; q < found; ++q) {
                        zc cf = sigma_dot(N, Vec + q, nev, cand, 1);
                        for (int64_t r = 0; r < 2 * N; ++r) cand[r] -= Vec[r * nev + q] * cf;
                    }
                double left = creal(sigma_dot(N, cand, 1, cand, 1));
                if (!(left > 1e-4)) continue;                                 /* the second copy of an accepted eigenpair */
                double nrm = 1.0 / sqrt(left);
                for (int64_t r = 0; r < 2 * N; ++r) Vec[r * nev + found] = cand[r] * nrm;
                omega[found] = om;
                res[found] = ri;
                ++found;
            }
            int ok = (found == nev) && all_converged;
            if (ok || last) { result = ok ? m : -m; break; }
        }
        if (last) break;
    }
done:
    free(Xb); free(Pb); free(alpha); free(beta); free(wv); free(pw); free(cand); free(S); free(th);
    return result;
}

/* ------------------------------------------------------------------------------------------
 * Second structure-preserving variant ("Gruning": "three variations of a structure-preserving Lanczos
 * iteration ... very similar in terms of operations"; the recurrence itself is in refs not in the container, DESIGN.md
 * reading R9, derived from Eq. 1): Lanczos on H ITSELF -- no squaring -- in the inner product of Omega = Sigma H, in which H is
 * self-adjoint (<u, H v>_Omega = u^H Omega Sigma Omega v; pseudo-Hermitian Lanczos).  Started at u_1 = [z_1; conj z_1], every
 * Lanczos vector keeps the block structure with alternating sign, u_j = [z_j; s_j conj z_j], s_j = (-1)^(j+1), because
 *     H [z; s conj z] = [w; -s conj w],   w = R z + s C conj(z)   (= P(z) for s = +1, M(z) for s = -1),
 * and Omega u_j = [w_j; s_j conj w_j], so that <u_i, u_j>_Omega = 2 Re(w_i^H z_j) for equal signs.  The diagonal recurrence
 * coefficient alpha_j = <u_j, H u_j>_Omega = |w_j|^2 - |w_j|^2 vanishes identically:
 *     beta_{j+1} u_{j+1} = H u_j - beta_j u_{j-1}   ->   half vectors:  beta_{j+1} z_{j+1} = w_j - beta_j z_{j-1},
 * T = tridiag(beta, 0, beta) has the eigenvalues +-theta in pairs and theta_i > 0 approximates omega_i DIRECTLY (one half apply
 * per Lanczos vector; two of these steps span what one step of orc_lanczos_full spans).  Normalisation <u, u>_Omega = 1:
 * 2 Re(z^H w) = 1.  Full reorthogonalisation (twice) of the new vector against the stored vectors of ITS OWN sign, with the real
 * coefficients 2 Re(w_i^H z): vectors of the other sign are Omega-orthogonal to it in exact arithmetic (the coefficient would be
 * purely imaginary) and are left alone, as the +-i copies are in orc_lanczos_full (reading R1).
 * Ritz vector for (theta, s): x = sum_{j odd} s_j z_j, y = sum_{j even} s_j z_j, v = [x + y; conj(x - y)], scaled to v^H Sigma v = 1.
 * Residual estimate |H v - theta v|_2 = beta_{n+1} |s_n| sqrt(2) |z_{n+1}|_2 (times that scale).  Multiplicity as in
 * orc_lanczos_full (candidates Sigma-orthogonalised against the accepted eigenvectors).  maxit counts Lanczos vectors.
 * Out: omega (nev ascending), Vec (2N x nev row-major), res (nev).  Returns the number of Lanczos vectors (<0: failed).
 * Pins (tests/test_oracle_eig.py): bse_direct on the same matrices; Ritz values of 2 m vectors = Ritz values of m steps of
 * orc_lanczos_full; residuals; Sigma-orthonormality; distinct omega on a run to the whole space.
 * ------------------------------------------------------------------------------------------ */
int orc_lanczos_full_gruning(int64_t N, const zc *R, const zc *C, int nev, double tol, int maxit, int check, int minit,
                             const zc *x0, double *omega, zc *Vec, double *res, double *ritz_out, int n_ritz)
{
    if (maxit > 4 * N) maxit = (int)(4 * N);
    zc *Zb = (zc *)malloc(sizeof(zc) * (size_t)N * (maxit + 1));      /* half vectors z_j            */
    zc *Wb = (zc *)malloc(sizeof(zc) * (size_t)N * (maxit + 1));      /* images w_j = P / M (z_j)    */
    double *beta = (double *)calloc(maxit + 2, sizeof(double)), *zero = (double *)calloc(maxit + 2, sizeof(double));
    zc *zv = (zc *)malloc(sizeof(zc) * N), *cand = (zc *)malloc(sizeof(zc) * 2 * (size_t)N);
    double *S = NULL, *th = NULL;
    int result = -1;
    /* u_1: 2 Re(z^H P z) = 1 */
    orc_apply_half(N, 1, +1, R, C, x0, Wb);
    {
        ld s = 0.0L;
        for (int64_t i = 0; i < N; ++i) s += (ld)creal(x0[i]) * (ld)creal(Wb[i]) + (ld)cimag(x0[i]) * (ld)cimag(Wb[i]);
        if (!(s > 0.0L)) { result = -1000000; goto done; }
        double sc = 1.0 / sqrt(2.0 * (double)s);
        for (int64_t i = 0; i < N; ++i) { Zb[i] = x0[i] * sc; Wb[i] *= sc; }
    }
    for (int j = 0; j < maxit; ++j) {                      /* vector index j (0-based), sign +1 for even j */
        /* candidate half vector of u_{j+1}: w_j (- beta_j z_{j-1}, covered by the reorthogonalisation) */
        memcpy(zv, Wb + (size_t)j * N, sizeof(zc) * N);
        for (int pass = 0; pass < 2; ++pass)
            for (int p = (j + 1) % 2; p <= j; p += 2) {    /* stored vectors with the sign of u_{j+1} */
                const zc *wp = Wb + (size_t)p * N, *zp = Zb + (size_t)p * N;
                ld s = 0.0L;
                for (int64_t i = 0; i < N; ++i) s += (ld)creal(wp[i]) * (ld)creal(zv[i]) + (ld)cimag(wp[i]) * (ld)cimag(zv[i]);
                double cf = 2.0 * (double)s;
                for (int64_t i = 0; i < N; ++i) zv[i] -= cf * zp[i];
            }
        zc *wn = Wb + (size_t)(j + 1) * N;
        orc_apply_half(N, 1, ((j + 1) % 2 == 0) ? +1 : -1, R, C, zv, wn);
        ld b2 = 0.0L;
        for (int64_t i = 0; i < N; ++i) b2 += (ld)creal(zv[i]) * (ld)creal(wn[i]) + (ld)cimag(zv[i]) * (ld)cimag(wn[i]);
        const int n = j + 1;                               /* Lanczos vectors so far */
        double b = 0.0, zn1 = 0.0;
        int breakdown = 0;
        if (b2 > 0.0L) {
            b = sqrt(2.0 * (double)b2);
            for (int64_t i = 0; i < N; ++i) { Zb[(size_t)(j + 1) * N + i] = zv[i] / b; wn[i] /= b; }
            zn1 = nrm2(N, Zb + (size_t)(j + 1) * N);
        } else if (nrm2(N, zv) > 1e-10) {
            result = -1000000; break;                      /* Omega not positive definite */
        } else breakdown = 1;
        beta[j + 1] = b;
        const int last = (n == maxit) || breakdown;
        if (n >= 2 * nev && n >= minit && n % 2 == 0 && (n % check == 0 || last)) {
            S = (double *)realloc(S, sizeof(double) * n * n);
            th = (double *)realloc(th, sizeof(double) * n);
            if (orc_tridiag_ql(n, zero, beta + 1, th, S)) break;          /* T = tridiag(beta, 0, beta) */
            const int h0 = n / 2;                                         /* th[h0 ...] are the positive eigenvalues, ascending */
            if (ritz_out) for (int i = 0; i < n_ritz && i < n - h0; ++i) ritz_out[i] = th[h0 + i];
            const double hn = th[n - 1];
            int found = 0, all_converged = 1;
            for (int i = h0; i < n && found < nev; ++i) {
                const double om = th[i];
                if (!(om > 0.0)) { all_converged = 0; if (!last) break; else continue; }
                for (int64_t r = 0; r < N; ++r) {
                    zc x = 0.0, y = 0.0;
                    for (int p = 0; p < n; ++p) {
                        if (p % 2 == 0) x += Zb[(size_t)p * N + r] * S[p * n + i];
                        else y += Zb[(size_t)p * N + r] * S[p * n + i];
                    }
                    cand[r] = x + y;
                    cand[r + N] = conj(x - y);
                }
                double sn = creal(sigma_dot(N, cand, 1, cand, 1));
                if (!(sn > 0.0)) { all_converged = 0; if (!last) break; else continue; }
                double sc = 1.0 / sqrt(sn);
                for (int64_t r = 0; r < 2 * N; ++r) cand[r] *= sc;
                const double ri = sc * b * fabs(S[(n - 1) * n + i]) * sqrt(2.0) * zn1;
                if (ri > tol * hn) {
                    if (!last) break;
                    all_converged = 0;
                }
                for (int pass = 0; pass < 2; ++pass)
                    for (int q = 0; q < found; ++q) {
                        zc cf = sigma_dot(N, Vec + q, nev, cand, 1);
                        for (int64_t r = 0; r < 2 * N; ++r) cand[r] -= Vec[r * nev + q] * cf;
                    }
                double left = creal(sigma_dot(N, cand, 1, cand, 1));
                if (!(left > 1e-4)) continue;                             /* the second copy of an accepted eigenpair */
                double nrm = 1.0 / sqrt(left);
                for (int64_t r = 0; r < 2 * N; ++r) Vec[r * nev + found] = cand[r] * nrm;
                omega[found] = om;
                res[found] = ri;
                ++found;
            }
            int ok = (found == nev) && all_converged;
            if (ok || last) { result = ok ? n : -n; break; }
        }
        if (last) break;
    }
done:
    free(Zb); free(Wb); free(beta); free(zero); free(zv); free(cand); free(S); free(th);
    return result;
}

/* ------------------------------------------------------------------------------------------
 * Lanczos with quadrature rules ("a Lanczos iteration with quadrature rules to obtain the
 * optical absorption spectrum directly, without explicitly computing the eigenpairs"), TDA case.
 * Textbook three-term recurrence on the Hermitian R started at d / |d| (no reorthogonalisation, no stored basis):
 *   beta_0 = |d|;  w = R v_j - beta_j v_{j-1};  alpha_j = Re(v_j^H w);  w -= alpha_j v_j;
 *   beta_{j+1} = |w|;  v_{j+1} = w / beta_{j+1}.
 * alpha[0..steps), beta[0..steps]: beta[0] = |d|, beta[j] (j >= 1) couples steps j-1 and j.
 * Returns the number of steps done (stops early when beta_{j+1} = 0).
 * The Gauss quadrature it defines reproduces the moments d^H R^p d, p <= 2 steps - 1, and the resolvent
 *   d^H (z - R)^{-1} d  ~=  beta_0^2 / (z - alpha_0 - beta_1^2 / (z - alpha_1 - beta_2^2 / ( ... ))).
 * ------------------------------------------------------------------------------------------ */
int orc_lanczos_quadrature(int64_t N, const zc *R, const zc *d, int steps, double *alpha, double *beta)
{
    zc *v = (zc *)malloc(sizeof(zc) * N), *vp = (zc *)calloc(N, sizeof(zc)), *w = (zc *)malloc(sizeof(zc) * N);
    double b0 = nrm2(N, d);
    beta[0] = b0;
    for (int64_t i = 0; i < N; ++i) v[i] = d[i] / b0;
    int done = 0;
    for (int j = 0; j < steps; ++j) {
        orc_apply_tda(N, 1, R, v, w);
        for (int64_t i = 0; i < N; ++i) w[i] -= beta[j] * vp[i] * (j > 0 ? 1.0 : 0.0);
        ld a = 0.0L;
        for (int64_t i = 0; i < N; ++i) a += (ld)creal(v[i]) * (ld)creal(w[i]) + (ld)cimag(v[i]) * (ld)cimag(w[i]);
        alpha[j] = (double)a;
        for (int64_t i = 0; i < N; ++i) w[i] -= alpha[j] * v[i];
        double b = nrm2(N, w);
        beta[j + 1] = b;
        done = j + 1;
        if (b == 0.0) break;
        for (int64_t i = 0; i < N; ++i) { vp[i] = v[i]; v[i] = w[i] / b; }
    }
    free(v); free(vp); free(w);
    return done;
}

/* Continued fraction of the Jacobi matrix: out[i] = beta_0^2 * [ (z_i - T)^{-1} ]_{00},  z_i = omega_i + i eta. */
void orc_quadrature_resolvent(int steps, const double *alpha, const double *beta, int n_omega, const double *omega,
                              double eta, zc *out)
{
    for (int i = 0; i < n_omega; ++i) {
        zc z = omega[i] + I * eta;
        zc f = z - alpha[steps - 1];
        for (int j = steps - 2; j >= 0; --j) f = z - alpha[j] - beta[j + 1] * beta[j + 1] / f;
        out[i] = beta[0] * beta[0] / f;
    }
}

/* ------------------------------------------------------------------------------------------
 * Lanczos with quadrature rules, full (pseudo-Hermitian) case (PAPER.md:65 with the operator of Eq. 1,
 * PAPER.md:18, A = R^*, C = C^T).  Reading (R7), derived from Eq. (1) with the maps of reading S4,
 *   P(x) = R x + C conj(x),  M(y) = R y - C conj(y),  H [x; conj x] = [P x; -conj P x],  H [y; -conj y] = [M y; conj M y]:
 * for u = [d; conj d] and Sigma = diag(I, -I),
 *   u^H Sigma (z - H)^{-1} u  =  2 <d, (z^2 - G)^{-1} d>_P,     G = M o P,   <a, b>_P = Re(a^H P(b)),
 * because (z - H)^{-1} = (z + H)(z^2 - H^2)^{-1}, H^2 [x; conj x] = [G x; conj G x], Sigma H = Omega with
 * [a; conj a]^H Omega [b; conj b] = 2 <a, b>_P, and the term with z alone is the quadratic form of an antisymmetric
 * matrix (P(i x) = i M(x)), hence zero.  G is self-adjoint in <.,.>_P, so the three-term recurrence of
 * orc_lanczos_full WITHOUT reorthogonalisation and without a stored basis gives a real Jacobi matrix:
 *   beta_0 = sqrt(<d, d>_P);  x_1 = d / beta_0, p_1 = P(x_1);
 *   w = M(p_j) - beta_j x_{j-1};  alpha_j = Re(p_j^H w);  w -= alpha_j x_j;  pw = P(w);
 *   beta_{j+1} = sqrt(Re(w^H pw));  x_{j+1} = w / beta_{j+1},  p_{j+1} = pw / beta_{j+1},
 * and  u^H Sigma (z - H)^{-1} u ~= 2 beta_0^2 [ (z^2 - T)^{-1} ]_00  (continued fraction in z^2).
 * The other start vector of the structure, [y; -conj y], equals -i [iy; conj(iy)]: call with d = i y.
 * Odd moments: u^H Sigma H^(2p+1) u = 2 beta_0^2 (T^p)_00 for p <= 2 steps - 1; even moments vanish.
 * Returns the number of steps done; -1000000 if Re(w^H P w) < 0 is met (Omega not positive definite).
 * ------------------------------------------------------------------------------------------ */
int orc_lanczos_quadrature_full(int64_t N, const zc *R, const zc *C, const zc *d, int steps, double *alpha, double *beta)
{
    zc *x = (zc *)malloc(sizeof(zc) * N), *xp = (zc *)calloc(N, sizeof(zc)), *p = (zc *)malloc(sizeof(zc) * N);
    zc *w = (zc *)malloc(sizeof(zc) * N), *pw = (zc *)malloc(sizeof(zc) * N);
    int done = 0;
    orc_apply_half(N, 1, +1, R, C, d, p);
    ld s0 = 0.0L;
    for (int64_t i = 0; i < N; ++i) s0 += (ld)creal(d[i]) * (ld)creal(p[i]) + (ld)cimag(d[i]) * (ld)cimag(p[i]);
    if (!(s0 > 0.0L)) { done = -1000000; goto out; }
    beta[0] = sqrt((double)s0);
    for (int64_t i = 0; i < N; ++i) { x[i] = d[i] / beta[0]; p[i] = p[i] / beta[0]; }
    for (int j = 0; j < steps; ++j) {
        orc_apply_half(N, 1, -1, R, C, p, w);                                  /* w = M(p_j) */
        if (j > 0) for (int64_t i = 0; i < N; ++i) w[i] -= beta[j] * xp[i];
        ld a = 0.0L;
        for (int64_t i = 0; i < N; ++i) a += (ld)creal(p[i]) * (ld)creal(w[i]) + (ld)cimag(p[i]) * (ld)cimag(w[i]);
        alpha[j] = (double)a;
        for (int64_t i = 0; i < N; ++i) w[i] -= alpha[j] * x[i];
        orc_apply_half(N, 1, +1, R, C, w, pw);                                 /* pw = P(w) */
        ld b2 = 0.0L;
        for (int64_t i = 0; i < N; ++i) b2 += (ld)creal(w[i]) * (ld)creal(pw[i]) + (ld)cimag(w[i]) * (ld)cimag(pw[i]);
        if (b2 < 0.0L) { done = -1000000; goto out; }
        double b = sqrt((double)b2);
        beta[j + 1] = b;
        done = j + 1;
        if (b == 0.0) break;
        for (int64_t i = 0; i < N; ++i) { xp[i] = x[i]; x[i] = w[i] / b; p[i] = pw[i] / b; }
    }
out:
    free(x); free(xp); free(p); free(w); free(pw);
    return done;
}

/* Continued fraction at arbitrary complex arguments: out[i] = beta_0^2 * [ (s_i - T)^{-1} ]_{00}. */
void orc_quadrature_resolvent_at(int steps, const double *alpha, const double *beta, int n, const zc *s, zc *out)
{
    for (int i = 0; i < n; ++i) {
        zc f = s[i] - alpha[steps - 1];
        for (int j = steps - 2; j >= 0; --j) f = s[i] - alpha[j] - beta[j + 1] * beta[j + 1] / f;
        out[i] = beta[0] * beta[0] / f;
    }
}

/* ------------------------------------------------------------------------------------------
 * Single-precision operand.  PAPER.md:111 and the caption of Table 2
 * (PAPER.md:115): the paper's BSE matrices are computed and stored in single precision.  The
 * complex64-stored operator is, by definition, the matrix whose entries are the IEEE 754 binary32
 * round-to-nearest-even images of the real and imaginary parts; everything downstream (apply,
 * Lanczos) is the same FP64 arithmetic on that matrix.  The rounding is written out from the
 * format's definition (24-bit significand, exponents 2^-126 .. 2^127, gradual underflow with
 * quantum 2^-149) instead of a cast, so that it can be checked by eye:
 *     x = m 2^e, 1/2 <= |m| < 1     ->  rint(m 2^24) 2^(e-24)      (normal range, e >= -125)
 *                                   ->  rint(x 2^149) 2^-149       (below 2^-126)
 *     |result| >= 2^128             ->  +-infinity
 * rint() rounds to nearest, ties to even, in the default rounding mode.
 * Pins (tests/test_oracle_c64.py): hand-computed ties and neighbours of 1, the error bound
 * |fl(x) - x| <= 2^-24 |x|, idempotence, exact agreement with the hardware conversion (numpy
 * astype) on random and special inputs, Weyl's bound for the eigenvalues of the rounded matrix.
 * ------------------------------------------------------------------------------------------ */
static double round_binary32(double x)
{
    if (x == 0.0 || isnan(x) || isinf(x)) return x;
    int e;
    double m = frexp(x, &e);                       /* x = m 2^e, 1/2 <= |m| < 1 */
    double r;
    if (e >= -125) r = ldexp(rint(ldexp(m, 24)), e - 24);
    else r = ldexp(rint(ldexp(x, 149)), -149);
    if (fabs(r) >= ldexp(1.0, 128)) r = copysign(INFINITY, x);
    return r;
}
void orc_round_c64(int64_t n, const zc *in, zc *out)
{
    double *o = (double *)out;                     /* parts written separately: re + I*im would turn -0 into +0 */
    for (int64_t i = 0; i < n; ++i) {
        o[2 * i] = round_binary32(creal(in[i]));
        o[2 * i + 1] = round_binary32(cimag(in[i]));
    }
}
