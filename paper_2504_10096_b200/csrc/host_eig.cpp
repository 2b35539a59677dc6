// Host eigensolver for the small projected problem (north_star: "the small projected
// eigenproblem may stay on the host").  Complex Hermitian m x m -> all eigenvalues (ascending) and the first nz
// eigenvectors.  Householder reduction to real symmetric tridiagonal form, implicit-shift QL on the tridiagonal
// with the plane rotations accumulated in a real matrix, then Z = Q * Zr.  No LAPACK dependency.
//
// Layout choices (m ~ 1000 at config 4, called once per restart):
//   * the Hermitian matrix-vector product of the reduction walks the stored lower triangle by COLUMNS only
//     (axpy for the part below the diagonal, dot for its conjugate-transposed image), per-thread accumulators;
//   * the rotation sweep of a QL iteration is a dependency chain along the column index but independent across
//     rows: Zr is stored in panels of 8 rows, [panel][column][8], so the chain runs on 8-row SIMD vectors with the
//     updated column carried in registers (one load and one store per rotation and panel);
//   * the back-transformation applies each reflector to 8 eigenvector columns at a time.
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace bse {

typedef std::complex<double> zc;

namespace {
constexpr int RP = 8;       // rows per panel of the rotation accumulator
constexpr int JB = 8;       // eigenvector columns per back-transformation task
inline int max_threads();
// threads worth starting for an m x m problem: the parallel regions of a step are short (a mat-vec, a rank-2 update, a
// panel sweep), and with more than one thread per ~64 rows the fork / barrier costs more than it saves (m = 200 on
// 8 cores: 11.1 ms with 8 threads, 7.1 ms with 4)
inline int threads_for(int m);
inline int max_threads()
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
inline int threads_for(int m) { return std::max(1, std::min(max_threads(), m / 64)); }

// The four hot loops, in explicit real arithmetic on interleaved (re, im) doubles (std::complex multiplication does
// not vectorise without -ffast-math) and compiled for SSE2 / AVX2+FMA / AVX-512 with run-time dispatch, so that the
// in-tree .so runs on whatever host CPU the GPU box has.
#if defined(__x86_64__) && defined(__GNUC__) && !defined(__clang__)
#define BSE_CLONES __attribute__((target_clones("default", "arch=x86-64-v3", "arch=x86-64-v4")))
#else
#define BSE_CLONES
#endif

// Columns c = c0, c0 + cs, ... of the Hermitian A22 (lower triangle, column-major, ld in complex elements):
//   xl[c..n) += A22[c..n, c] v[c],   xl[c] += sum_{r > c} conj(A22[r, c]) v[r]
BSE_CLONES void herm_matvec_columns(int n, const double *A22, int64_t ld, const double *v, double *xl, int c0, int cs)
{
    for (int c = c0; c < n; c += cs) {
        const double *col = A22 + 2 * ((int64_t)c * ld);
        const double vcr = v[2 * c], vci = v[2 * c + 1];
        double sr = 0.0, si = 0.0;
        xl[2 * c] += col[2 * c] * vcr;                 // real diagonal
        xl[2 * c + 1] += col[2 * c] * vci;
#pragma omp simd reduction(+ : sr, si)
        for (int r = c + 1; r < n; ++r) {
            const double ar = col[2 * r], ai = col[2 * r + 1];
            xl[2 * r] += ar * vcr - ai * vci;
            xl[2 * r + 1] += ar * vci + ai * vcr;
            sr += ar * v[2 * r] + ai * v[2 * r + 1];
            si += ar * v[2 * r + 1] - ai * v[2 * r];
        }
        xl[2 * c] += sr;
        xl[2 * c + 1] += si;
    }
}

// A22[c.., c] -= v w_c^* + w v_c^*  for columns c0 <= c < c1
BSE_CLONES void rank2_update_columns(int n, double *A22, int64_t ld, const double *v, const double *x, int c0, int c1)
{
    for (int c = c0; c < c1; ++c) {
        double *col = A22 + 2 * ((int64_t)c * ld);
        const double wr = x[2 * c], wi = -x[2 * c + 1], ur = v[2 * c], ui = -v[2 * c + 1];   // conj(w_c), conj(v_c)
#pragma omp simd
        for (int r = c; r < n; ++r) {
            const double vr = v[2 * r], vi = v[2 * r + 1], xr = x[2 * r], xi = x[2 * r + 1];
            col[2 * r] -= vr * wr - vi * wi + xr * ur - xi * ui;
            col[2 * r + 1] -= vr * wi + vi * wr + xr * ui + xi * ur;
        }
    }
}

// One panel of RP rows: rotations q = mm-1 down to ilo on columns (q, q+1); zb[(column) * RP + row]
BSE_CLONES void rotate_panel(double *zb, int mm, int ilo, const double *rc, const double *rs)
{
    double f[RP];
#pragma omp simd
    for (int rr = 0; rr < RP; ++rr) f[rr] = zb[(size_t)mm * RP + rr];
    for (int q = mm - 1; q >= ilo; --q) {
        const double cq = rc[q], sq = rs[q];
        double *zq = zb + (size_t)q * RP;
#pragma omp simd
        for (int rr = 0; rr < RP; ++rr) {
            const double g = zq[rr];
            zq[RP + rr] = sq * g + cq * f[rr];
            f[rr] = cq * g - sq * f[rr];
        }
    }
#pragma omp simd
    for (int rr = 0; rr < RP; ++rr) zb[(size_t)ilo * RP + rr] = f[rr];
}

// z_j <- (I - tau v v^H) z_j for nb <= JB columns; v = vi[lo .. m) (interleaved), zc[jj] interleaved columns
BSE_CLONES void reflect_columns(int lo, int m, const double *vi, double taur, double taui, double *const *zcol, int nb)
{
    double sr[JB], si[JB];
    for (int jj = 0; jj < nb; ++jj) {
        const double *z = zcol[jj];
        double ar = 0.0, ai = 0.0;
#pragma omp simd reduction(+ : ar, ai)
        for (int r = lo; r < m; ++r) {                       // conj(v_r) z_r
            ar += vi[2 * r] * z[2 * r] + vi[2 * r + 1] * z[2 * r + 1];
            ai += vi[2 * r] * z[2 * r + 1] - vi[2 * r + 1] * z[2 * r];
        }
        sr[jj] = taur * ar - taui * ai;
        si[jj] = taur * ai + taui * ar;
    }
    for (int jj = 0; jj < nb; ++jj) {
        double *z = zcol[jj];
        const double pr = sr[jj], pi = si[jj];
#pragma omp simd
        for (int r = lo; r < m; ++r) {
            z[2 * r] -= vi[2 * r] * pr - vi[2 * r + 1] * pi;
            z[2 * r + 1] -= vi[2 * r] * pi + vi[2 * r + 1] * pr;
        }
    }
}
}  // namespace

// Implicit QL on the real symmetric tridiagonal (d, e) with the rotations accumulated in Zr (real m x m) stored in
// panels of RP rows, Zb[(panel * m + column) * RP + row_in_panel]; eigenvalues sorted ascending into w, ord = the
// permutation.  Shared by the complex Hermitian and the real symmetric driver.  Returns 0, or >0 if QL failed.
static int tridiag_ql(int m, std::vector<double> &d, std::vector<double> &e, std::vector<double> &Zb, std::vector<int> &ord,
                      double *w, bool want_z = true)
{
    // ---- implicit QL on (d, e) with the rotations accumulated in Zr (real m x m), stored in panels of RP rows:
    //      Zb[(panel * m + column) * RP + row_in_panel]
    const int npan = want_z ? (m + RP - 1) / RP : 0;     // want_z = false: eigenvalues only, O(m^2)
    Zb.assign((size_t)npan * m * RP, 0.0);
    if (want_z)
        for (int i = 0; i < m; ++i) Zb[((size_t)(i / RP) * m + i) * RP + i % RP] = 1.0;
    std::vector<double> rc(m), rs(m);
    int fail = 0;
    for (int l = 0; l < m; ++l) {
        int iter = 0;
        while (true) {
            int mm = l;
            for (; mm < m - 1; ++mm) {
                double dd = std::fabs(d[mm]) + std::fabs(d[mm + 1]);
                if (std::fabs(e[mm]) <= 2.3e-16 * dd) break;
            }
            if (mm == l) break;
            if (++iter > 80) { fail = l + 1; break; }
            double gg = (d[l + 1] - d[l]) / (2.0 * e[l]);
            double r = std::hypot(gg, 1.0);
            gg = d[mm] - d[l] + e[l] / (gg + std::copysign(r, gg));
            double s = 1.0, c = 1.0, p = 0.0;
            int i;
            bool under = false;
            for (i = mm - 1; i >= l; --i) {
                double f = s * e[i], b = c * e[i];
                r = std::hypot(f, gg);
                e[i + 1] = r;
                if (r == 0.0) { d[i + 1] -= p; e[mm] = 0.0; under = true; break; }
                s = f / r; c = gg / r;
                gg = d[i + 1] - p;
                r = (d[i] - gg) * s + 2.0 * c * b;
                p = s * r;
                d[i + 1] = gg + p;
                gg = c * r - b;
                rc[i] = c; rs[i] = s;
            }
            const int ilo = under ? i + 1 : l;
            // apply the recorded rotations (q = mm-1 down to ilo) to columns (q, q+1): z[q+1] = s z[q] + c f,
            // z[q] = c z[q] - s f with f the old z[q+1]; the new z[q] is the next step's f and stays in registers
            if (want_z && mm - 1 >= ilo) {
                const int64_t work = (int64_t)(mm - ilo) * m;
#pragma omp parallel for schedule(static) num_threads(threads_for(m)) if (work > 32768)
                for (int pn = 0; pn < npan; ++pn) rotate_panel(&Zb[(size_t)pn * m * RP], mm, ilo, rc.data(), rs.data());
            }
            if (under) continue;
            d[l] -= p;
            e[l] = gg;
            e[mm] = 0.0;
        }
        if (fail) break;
    }
    // ---- sort ascending
    ord.resize(m);
    std::iota(ord.begin(), ord.end(), 0);
    std::sort(ord.begin(), ord.end(), [&](int p, int q) { return d[p] < d[q]; });
    for (int i = 0; i < m; ++i) w[i] = d[ord[i]];
    return fail;
}

// A (column-major, lda, lower triangle referenced and destroyed).  Returns 0, or >0 if QL failed to converge.
int host_heev(int m, void *A_, int lda, double *w, void *Z_, int ldz, int nz)
{
    zc *A = static_cast<zc *>(A_), *Z = static_cast<zc *>(Z_);
    if (m <= 0) return 0;
    if (nz > m) nz = m;
    std::vector<double> d(m), e(m, 0.0);
    std::vector<zc> tau(m, zc(0.0));
    auto a = [&](int i, int j) -> zc & { return A[i + (int64_t)j * lda]; };

    // ---- Householder tridiagonalisation, lower variant:  A = Q T Q^H,  Q = H_0 H_1 ... H_{m-2},  H_i = I - tau v v^H
    const int nth = threads_for(m);
    std::vector<zc> x(m), v(m), xt((size_t)nth * m);
    for (int i = 0; i < m - 1; ++i) {
        const int n = m - i - 1;                  // length of the column below the diagonal
        zc alpha = a(i + 1, i);
        double xnorm2 = 0.0;
        for (int r = i + 2; r < m; ++r) xnorm2 += std::norm(a(r, i));
        zc t(0.0);
        double beta = alpha.real();
        if (xnorm2 != 0.0 || alpha.imag() != 0.0) {
            beta = -std::copysign(std::sqrt(std::norm(alpha) + xnorm2), alpha.real());
            t = zc((beta - alpha.real()) / beta, -alpha.imag() / beta);
            zc sc = 1.0 / (alpha - beta);
            for (int r = i + 2; r < m; ++r) a(r, i) *= sc;
        }
        e[i] = beta;
        tau[i] = t;
        a(i + 1, i) = 1.0;                         // v = A(i+1:m, i) with v_0 = 1
        if (t != zc(0.0)) {
            for (int r = 0; r < n; ++r) v[r] = a(i + 1 + r, i);
            // x = tau * A22 * v   (A22 Hermitian, lower triangle stored), column by column:
            //   x[c..n) += A22[c..n, c] v[c]   and   x[c] += sum_{r > c} conj(A22[r, c]) v[r]
            const bool par = n > 128 && nth > 1;
            int nt_act = 1;                           // the team the runtime actually grants (may be < nth)
#pragma omp parallel num_threads(nth) if (par)
            {
#ifdef _OPENMP
                const int tid = omp_get_thread_num(), team = omp_get_num_threads();
#else
                const int tid = 0, team = 1;
#endif
                if (tid == 0) nt_act = team;
                zc *xl = &xt[(size_t)tid * m];
                for (int r = 0; r < n; ++r) xl[r] = zc(0.0);
                // cyclic columns: column lengths shrink linearly, a cyclic split balances them
                herm_matvec_columns(n, reinterpret_cast<const double *>(&a(i + 1, i + 1)), lda,
                                    reinterpret_cast<const double *>(v.data()), reinterpret_cast<double *>(xl), tid, team);
            }
            for (int r = 0; r < n; ++r) {
                zc s(0.0);
                for (int q = 0; q < nt_act; ++q) s += xt[(size_t)q * m + r];
                x[r] = t * s;
            }
            zc dot(0.0);
            for (int r = 0; r < n; ++r) dot += std::conj(x[r]) * v[r];
            zc al = -0.5 * t * dot;
            for (int r = 0; r < n; ++r) x[r] += al * v[r];                 // w
            // A22 -= v w^H + w v^H   (lower triangle)
#pragma omp parallel for schedule(static, 1) num_threads(nth) if (par)
            for (int c0 = 0; c0 < n; c0 += 4)
                rank2_update_columns(n, reinterpret_cast<double *>(&a(i + 1, i + 1)), lda,
                                     reinterpret_cast<const double *>(v.data()), reinterpret_cast<const double *>(x.data()),
                                     c0, std::min(c0 + 4, n));
        }
        d[i] = a(i, i).real();
    }
    d[m - 1] = a(m - 1, m - 1).real();

    std::vector<double> Zb;
    std::vector<int> ord;
    const int fail = tridiag_ql(m, d, e, Zb, ord, w);
    if (nz <= 0 || !Z) return fail;

    // ---- Z = Q * Zr[:, ord[0..nz)]:  start from the real eigenvectors and apply H_{m-2} ... H_0 from the left,
    //      each reflector to JB columns at a time (the reflector is read once per block, not once per column)
#pragma omp parallel for schedule(dynamic, 1) num_threads(nth) if (m > 64)
    for (int j0 = 0; j0 < nz; j0 += JB) {
        const int nb = std::min(JB, nz - j0);
        zc *zcol[JB];
        for (int jj = 0; jj < nb; ++jj) {
            zcol[jj] = Z + (int64_t)(j0 + jj) * ldz;
            const int src = ord[j0 + jj];
            for (int i = 0; i < m; ++i) zcol[jj][i] = Zb[((size_t)(i / RP) * m + src) * RP + i % RP];
        }
        double *zd[JB];
        for (int jj = 0; jj < nb; ++jj) zd[jj] = reinterpret_cast<double *>(zcol[jj]);
        for (int i = m - 2; i >= 0; --i) {
            if (tau[i] == zc(0.0)) continue;
            // v_r = A[r, i], r = i+1 .. m-1 (v_{i+1} = 1 stored)
            reflect_columns(i + 1, m, reinterpret_cast<const double *>(&a(0, i)), tau[i].real(), tau[i].imag(), zd, nb);
        }
    }
    return fail;
}


// ------------------------------------------------------------------------------------------------------------------
// Real symmetric variant (full mode: the projected matrix of the structure-preserving iteration is real symmetric,
// SURVEY.md 8(a) a8): the same three stages in real arithmetic -- a quarter of the flops of the complex driver in the
// reduction and the back-transformation, the same QL.
// ------------------------------------------------------------------------------------------------------------------
namespace {
BSE_CLONES void sym_matvec_columns(int n, const double *A22, int64_t ld, const double *v, double *xl, int c0, int cs)
{
    for (int c = c0; c < n; c += cs) {
        const double *col = A22 + (int64_t)c * ld;
        const double vc = v[c];
        double sr = 0.0;
        xl[c] += col[c] * vc;
#pragma omp simd reduction(+ : sr)
        for (int r = c + 1; r < n; ++r) {
            xl[r] += col[r] * vc;
            sr += col[r] * v[r];
        }
        xl[c] += sr;
    }
}
BSE_CLONES void rank2_update_columns_real(int n, double *A22, int64_t ld, const double *v, const double *x, int c0, int c1)
{
    for (int c = c0; c < c1; ++c) {
        double *col = A22 + (int64_t)c * ld;
        const double wc = x[c], vc = v[c];
#pragma omp simd
        for (int r = c; r < n; ++r) col[r] -= v[r] * wc + x[r] * vc;
    }
}
BSE_CLONES void reflect_columns_real(int lo, int m, const double *vi, double tau, double *const *zcol, int nb)
{
    for (int jj = 0; jj < nb; ++jj) {
        double *z = zcol[jj];
        double a = 0.0;
#pragma omp simd reduction(+ : a)
        for (int r = lo; r < m; ++r) a += vi[r] * z[r];
        const double p = tau * a;
#pragma omp simd
        for (int r = lo; r < m; ++r) z[r] -= vi[r] * p;
    }
}
}  // namespace

// A (real, column-major, lda, lower triangle referenced and destroyed); Z real m x nz.  Returns 0, or >0 if QL failed.
int host_syev(int m, double *A, int lda, double *w, double *Z, int ldz, int nz)
{
    if (m <= 0) return 0;
    if (nz > m) nz = m;
    std::vector<double> d(m), e(m, 0.0), tau(m, 0.0);
    auto a = [&](int i, int j) -> double & { return A[i + (int64_t)j * lda]; };
    const int nth = threads_for(m);
    std::vector<double> x(m), v(m), xt((size_t)nth * m);
    for (int i = 0; i < m - 1; ++i) {
        const int n = m - i - 1;
        const double alpha = a(i + 1, i);
        double xnorm2 = 0.0;
        for (int r = i + 2; r < m; ++r) xnorm2 += a(r, i) * a(r, i);
        double t = 0.0, beta = alpha;
        if (xnorm2 != 0.0) {
            beta = -std::copysign(std::sqrt(alpha * alpha + xnorm2), alpha);
            t = (beta - alpha) / beta;
            const double sc = 1.0 / (alpha - beta);
            for (int r = i + 2; r < m; ++r) a(r, i) *= sc;
        }
        e[i] = beta;
        tau[i] = t;
        a(i + 1, i) = 1.0;
        if (t != 0.0) {
            for (int r = 0; r < n; ++r) v[r] = a(i + 1 + r, i);
            const bool par = n > 256 && nth > 1;
            int nt_act = 1;
#pragma omp parallel num_threads(nth) if (par)
            {
#ifdef _OPENMP
                const int tid = omp_get_thread_num(), team = omp_get_num_threads();
#else
                const int tid = 0, team = 1;
#endif
                if (tid == 0) nt_act = team;
                double *xl = &xt[(size_t)tid * m];
                for (int r = 0; r < n; ++r) xl[r] = 0.0;
                sym_matvec_columns(n, &a(i + 1, i + 1), lda, v.data(), xl, tid, team);
            }
            double dot = 0.0;
            for (int r = 0; r < n; ++r) {
                double s = 0.0;
                for (int q = 0; q < nt_act; ++q) s += xt[(size_t)q * m + r];
                x[r] = t * s;
                dot += x[r] * v[r];
            }
            const double al = -0.5 * t * dot;
            for (int r = 0; r < n; ++r) x[r] += al * v[r];
#pragma omp parallel for schedule(static, 1) num_threads(nth) if (par)
            for (int c0 = 0; c0 < n; c0 += 8)
                rank2_update_columns_real(n, &a(i + 1, i + 1), lda, v.data(), x.data(), c0, std::min(c0 + 8, n));
        }
        d[i] = a(i, i);
    }
    d[m - 1] = a(m - 1, m - 1);

    std::vector<double> Zb;
    std::vector<int> ord;
    const int fail = tridiag_ql(m, d, e, Zb, ord, w);
    if (nz <= 0 || !Z) return fail;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nth) if (m > 64)
    for (int j0 = 0; j0 < nz; j0 += JB) {
        const int nb = std::min(JB, nz - j0);
        double *zcol[JB];
        for (int jj = 0; jj < nb; ++jj) {
            zcol[jj] = Z + (int64_t)(j0 + jj) * ldz;
            const int src = ord[j0 + jj];
            for (int i = 0; i < m; ++i) zcol[jj][i] = Zb[((size_t)(i / RP) * m + src) * RP + i % RP];
        }
        for (int i = m - 2; i >= 0; --i) {
            if (tau[i] == 0.0) continue;
            reflect_columns_real(i + 1, m, &a(0, i), tau[i], zcol, nb);
        }
    }
    return fail;
}

// Eigenvectors of the nz lowest eigenvalues w[0..nz) (ascending, already computed) of the real symmetric tridiagonal (d, e) by
// inverse iteration: LU with partial pivoting of T - w_j I, a seeded random start, a few solves, and modified Gram-Schmidt
// against the earlier vectors of the same cluster of close eigenvalues (gaps below 1e-5 ||T||_1) -- the textbook method
// behind LAPACK's dstein, restated.  O(m) per solve; clusters are independent and run in parallel.  Returns 0, or j + 1 if
// vector j did not reach a residual of 1e-12 ||T||_1.
static int tridiag_inverse_iteration(int m, const double *d, const double *e, const double *w, int nz, double *Z, int ldz)
{
    const double eps = 2.220446049250313e-16;
    double onenrm = 0.0;
    for (int i = 0; i < m; ++i) {
        const double v = std::fabs(d[i]) + (i > 0 ? std::fabs(e[i - 1]) : 0.0) + (i + 1 < m ? std::fabs(e[i]) : 0.0);
        onenrm = std::max(onenrm, v);
    }
    if (onenrm == 0.0) onenrm = 1.0;
    // (dstein re-orthogonalises below 1e-3 ||T||; 1e-5 leaves eps ||T|| / gap <= 2e-11 between clusters, far inside the 1e-7
    //  the eigenvectors of H are held to, and keeps the clusters of a dense spectrum short)
    const double ortol = 1e-5 * onenrm, tiny = eps * onenrm;
    // cluster boundaries
    std::vector<int> start;
    for (int j = 0; j < nz; ++j)
        if (j == 0 || w[j] - w[j - 1] > ortol) start.push_back(j);
    start.push_back(nz);
    int fail = 0;
    const int ncl = (int)start.size() - 1;
    int largest = 0;
    for (int cl = 0; cl < ncl; ++cl) largest = std::max(largest, start[cl + 1] - start[cl]);
    // many small clusters: one thread per cluster; a large one: clusters in turn, its Gram-Schmidt sums threaded
    const bool outer = largest <= 64;
#pragma omp parallel for schedule(dynamic, 1) if (outer && nz > 8)
    for (int cl = 0; cl < ncl; ++cl) {
        std::vector<double> a(m), b(m), b2(m), l(m), x(m), dots(start[cl + 1] - start[cl]);
        std::vector<char> piv(m);
        double prev = 0.0;
        for (int j = start[cl]; j < start[cl + 1]; ++j) {
            double lam = w[j];
            if (j > start[cl] && lam - prev < 10.0 * eps * std::fabs(lam) + 10.0 * tiny) lam = prev + 10.0 * eps * std::fabs(lam) + 10.0 * tiny;
            prev = lam;
            // ---- P L U = T - lam I
            for (int i = 0; i < m; ++i) { a[i] = d[i] - lam; b[i] = i + 1 < m ? e[i] : 0.0; b2[i] = 0.0; }
            for (int k = 0; k + 1 < m; ++k) {
                const double c = e[k];
                if (std::fabs(a[k]) >= std::fabs(c)) {
                    if (std::fabs(a[k]) < tiny) a[k] = std::copysign(tiny, a[k] == 0.0 ? 1.0 : a[k]);
                    const double mult = c / a[k];
                    a[k + 1] -= mult * b[k];
                    l[k] = mult; piv[k] = 0;
                } else {
                    const double mult = a[k] / c, t = a[k + 1];
                    a[k] = c;
                    a[k + 1] = b[k] - mult * t;
                    if (k + 2 < m) { b2[k] = b[k + 1]; b[k + 1] = -mult * b2[k]; }
                    b[k] = t;
                    l[k] = mult; piv[k] = 1;
                }
            }
            if (std::fabs(a[m - 1]) < tiny) a[m - 1] = std::copysign(tiny, a[m - 1] == 0.0 ? 1.0 : a[m - 1]);
            // ---- seeded start
            uint64_t rs = 0x9E3779B97F4A7C15ull * (uint64_t)(j + 1) + 12345u;
            for (int i = 0; i < m; ++i) {
                rs = rs * 6364136223846793005ull + 1442695040888963407ull;
                x[i] = ((double)(rs >> 11) / 9007199254740992.0) - 0.5;
            }
            double *zj = Z + (int64_t)j * ldz;
            bool ok = false;
            for (int it = 0; it < 8 && !ok; ++it) {
                for (int k = 0; k + 1 < m; ++k) {                                  // forward
                    if (piv[k]) std::swap(x[k], x[k + 1]);
                    x[k + 1] -= l[k] * x[k];
                }
                x[m - 1] /= a[m - 1];                                              // backward
                if (m > 1) x[m - 2] = (x[m - 2] - b[m - 2] * x[m - 1]) / a[m - 2];
                for (int k = m - 3; k >= 0; --k) x[k] = (x[k] - b[k] * x[k + 1] - b2[k] * x[k + 2]) / a[k];
                // re-orthogonalise inside the cluster: classical Gram-Schmidt, twice (sums over all earlier vectors at once)
                const int nq = j - start[cl];
                const double *Zc = Z + (int64_t)start[cl] * ldz;
                for (int rep = 0; rep < 2 && nq > 0; ++rep) {
                    const bool par = !outer && (int64_t)nq * m > 65536;
#pragma omp parallel for schedule(static) if (par)
                    for (int q = 0; q < nq; ++q) {
                        const double *zq = Zc + (int64_t)q * ldz;
                        double dot = 0.0;
#pragma omp simd reduction(+ : dot)
                        for (int i = 0; i < m; ++i) dot += zq[i] * x[i];
                        dots[q] = dot;
                    }
#pragma omp parallel for schedule(static) if (par)
                    for (int i0 = 0; i0 < m; i0 += 512) {
                        const int i1 = std::min(m, i0 + 512);
                        for (int q = 0; q < nq; ++q) {
                            const double *zq = Zc + (int64_t)q * ldz;
                            const double dq = dots[q];
#pragma omp simd
                            for (int i = i0; i < i1; ++i) x[i] -= dq * zq[i];
                        }
                    }
                }
                double nrm = 0.0;
                for (int i = 0; i < m; ++i) nrm += x[i] * x[i];
                nrm = std::sqrt(nrm);
                if (!(nrm > 0.0) || !std::isfinite(nrm)) break;
                for (int i = 0; i < m; ++i) x[i] /= nrm;
                if (it >= 1) {                                                      // residual of the normalised vector
                    double r2 = 0.0;
                    for (int i = 0; i < m; ++i) {
                        double v = (d[i] - w[j]) * x[i];
                        if (i > 0) v += e[i - 1] * x[i - 1];
                        if (i + 1 < m) v += e[i] * x[i + 1];
                        r2 += v * v;
                    }
                    ok = std::sqrt(r2) <= 1e-12 * onenrm;
                }
            }
            for (int i = 0; i < m; ++i) zj[i] = x[i];
            if (!ok) {
#pragma omp critical
                if (!fail) fail = j + 1;
            }
        }
    }
    return fail;
}

// Real symmetric tridiagonal (d: m diagonal entries, e: m - 1 sub-diagonal entries, both untouched): all eigenvalues
// ascending in w and the eigenvectors of the nz lowest in Z (m x nz, column-major, ldz).  The last stage of the direct
// route (bse_direct.cu).  Eigenvalues by QL without accumulation, O(m^2), vectors by inverse iteration, O(m) each plus the
// Gram-Schmidt sums inside clusters; tiny problems, and any problem on which inverse iteration misses its residual bound,
// take QL with the rotations accumulated, O(m^3).  Returns 0, or >0 if QL failed.
int host_stev(int m, double *d_in, double *e_in, double *w, double *Z, int ldz, int nz)
{
    if (m <= 0) return 0;
    if (nz > m) nz = m;
    const bool want = nz > 0 && Z;
    std::vector<double> Zb;
    std::vector<int> ord;
    auto ql = [&](bool accumulate) {
        std::vector<double> d(d_in, d_in + m), e(m, 0.0);
        for (int i = 0; i + 1 < m; ++i) e[i] = e_in[i];
        return tridiag_ql(m, d, e, Zb, ord, w, accumulate);
    };
    if (!want) return ql(false);
    if (m > 64) {
        if (int fail = ql(false)) return fail;
        if (tridiag_inverse_iteration(m, d_in, e_in, w, nz, Z, ldz) == 0) return 0;
    }
    if (int fail = ql(true)) return fail;
#pragma omp parallel for schedule(static) if ((int64_t)m * nz > 65536)
    for (int j = 0; j < nz; ++j) {
        const int src = ord[j];
        double *z = Z + (int64_t)j * ldz;
        for (int i = 0; i < m; ++i) z[i] = Zb[((size_t)(i / RP) * m + src) * RP + i % RP];
    }
    return 0;
}

// The nz lowest eigenvalues of the real symmetric tridiagonal (d, e) by bisection on the Sturm count (number of negative
// pivots of the LDL^T factorisation of T - x I), each to the last bit the count can resolve (absolute accuracy ~ eps ||T||, as
// QL); O(m) per count, ~60 counts per eigenvalue, eigenvalues in parallel.
static void tridiag_bisect_lowest(int m, const double *d, const double *e, int nz, double *w)
{
    const double eps = 2.220446049250313e-16;
    double lo0 = d[0], hi0 = d[0], tnorm = 0.0;
    for (int i = 0; i < m; ++i) {
        const double r = (i > 0 ? std::fabs(e[i - 1]) : 0.0) + (i + 1 < m ? std::fabs(e[i]) : 0.0);
        lo0 = std::min(lo0, d[i] - r);
        hi0 = std::max(hi0, d[i] + r);
        tnorm = std::max(tnorm, std::fabs(d[i]) + r);
    }
    const double pivmin = std::max(eps * tnorm * eps, 1e-300);
    auto count_below = [&](double x) {                      // number of eigenvalues < x
        int c = 0;
        double q = d[0] - x;
        if (std::fabs(q) < pivmin) q = -pivmin;
        if (q < 0.0) ++c;
        for (int i = 1; i < m; ++i) {
            q = d[i] - x - e[i - 1] * e[i - 1] / q;
            if (std::fabs(q) < pivmin) q = -pivmin;
            if (q < 0.0) ++c;
        }
        return c;
    };
    lo0 -= 2.0 * eps * tnorm + pivmin;
    hi0 += 2.0 * eps * tnorm + pivmin;
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = 0; i < nz; ++i) {
        double lo = lo0, hi = hi0;                          // invariant: count(lo) <= i < count(hi)
        for (int it = 0; it < 200; ++it) {
            const double mid = 0.5 * (lo + hi);
            if (!(mid > lo && mid < hi)) break;            // adjacent doubles
            if (count_below(mid) <= i) lo = mid; else hi = mid;
            if (hi - lo <= 2.0 * eps * std::max(std::fabs(lo), std::fabs(hi))) break;
        }
        w[i] = 0.5 * (lo + hi);
    }
}

// The nz lowest eigenpairs only (w: nz values).  A small part of the spectrum (8 nz <= m): bisection + inverse iteration, no
// O(m^2) sweep over the whole matrix; otherwise host_stev.
int host_stev_lowest(int m, double *d, double *e, int nz, double *w, double *Z, int ldz)
{
    if (m <= 0 || nz <= 0) return 0;
    if (nz > m) nz = m;
    if (m > 64 && 8 * nz <= m) {
        tridiag_bisect_lowest(m, d, e, nz, w);
        if (!Z || tridiag_inverse_iteration(m, d, e, w, nz, Z, ldz) == 0) return 0;
    }
    std::vector<double> wall(m);
    const int fail = host_stev(m, d, e, wall.data(), Z, ldz, Z ? nz : 0);
    for (int i = 0; i < nz; ++i) w[i] = wall[i];
    return fail;
}

}  // namespace bse
