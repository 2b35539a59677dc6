// Host eigensolver for the small projected problem (north_star: "the small projected
// eigenproblem may stay on the host").  Complex Hermitian m x m -> all eigenvalues (ascending) and the first nz
// eigenvectors.  Householder reduction to real symmetric tridiagonal form, implicit-shift QL on the tridiagonal
// with the plane rotations accumulated in a real matrix, then Z = Q * Zr.  No LAPACK dependency.
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <numeric>
#include <vector>

namespace bse {

typedef std::complex<double> zc;

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
    std::vector<zc> x(m), v(m);
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
            // x = tau * A22 * v   (A22 Hermitian, lower triangle stored)
#pragma omp parallel for schedule(static) if (n > 128)
            for (int r = 0; r < n; ++r) {
                zc s(0.0);
                for (int c = 0; c <= r; ++c) s += a(i + 1 + r, i + 1 + c) * v[c];
                for (int c = r + 1; c < n; ++c) s += std::conj(a(i + 1 + c, i + 1 + r)) * v[c];
                x[r] = t * s;
            }
            zc dot(0.0);
            for (int r = 0; r < n; ++r) dot += std::conj(x[r]) * v[r];
            zc al = -0.5 * t * dot;
            for (int r = 0; r < n; ++r) x[r] += al * v[r];                 // w
            // A22 -= v w^H + w v^H   (lower triangle)
#pragma omp parallel for schedule(static) if (n > 128)
            for (int c = 0; c < n; ++c) {
                zc wc = std::conj(x[c]), vc = std::conj(v[c]);
                for (int r = c; r < n; ++r) a(i + 1 + r, i + 1 + c) -= v[r] * wc + x[r] * vc;
            }
        }
        d[i] = a(i, i).real();
    }
    d[m - 1] = a(m - 1, m - 1).real();

    // ---- implicit QL on (d, e) with rotations accumulated in the real row-major matrix Zr (m x m)
    std::vector<double> Zr((size_t)m * m, 0.0);
    for (int i = 0; i < m; ++i) Zr[(size_t)i * m + i] = 1.0;
    std::vector<double> rc(m), rs(m);
    int fail = 0;
    // shift e so that e[i] couples i and i+1 (already the case), e[m-1] = 0
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
            // apply the recorded rotations (i = mm-1 down to ilo) to columns (i, i+1) of Zr, all rows in parallel
#pragma omp parallel for schedule(static) if (m > 128)
            for (int row = 0; row < m; ++row) {
                double *z = &Zr[(size_t)row * m];
                for (int q = mm - 1; q >= ilo; --q) {
                    double f = z[q + 1];
                    z[q + 1] = rs[q] * z[q] + rc[q] * f;
                    z[q] = rc[q] * z[q] - rs[q] * f;
                }
            }
            if (under) continue;
            d[l] -= p;
            e[l] = gg;
            e[mm] = 0.0;
        }
        if (fail) break;
    }
    // ---- sort ascending
    std::vector<int> ord(m);
    std::iota(ord.begin(), ord.end(), 0);
    std::sort(ord.begin(), ord.end(), [&](int p, int q) { return d[p] < d[q]; });
    for (int i = 0; i < m; ++i) w[i] = d[ord[i]];
    if (nz <= 0 || !Z) return fail;

    // ---- Z = Q * Zr[:, ord[0..nz)]:  start from the real eigenvectors and apply H_{m-2} ... H_0 from the left
    for (int j = 0; j < nz; ++j)
        for (int i = 0; i < m; ++i) Z[i + (int64_t)j * ldz] = Zr[(size_t)i * m + ord[j]];
#pragma omp parallel for schedule(static) if (m > 64)
    for (int j = 0; j < nz; ++j) {
        zc *z = Z + (int64_t)j * ldz;
        for (int i = m - 2; i >= 0; --i) {
            if (tau[i] == zc(0.0)) continue;
            zc s(0.0);
            for (int r = i + 1; r < m; ++r) s += std::conj(a(r, i)) * z[r];   // v^H z  (v_0 = 1 stored)
            s *= tau[i];
            for (int r = i + 1; r < m; ++r) z[r] -= a(r, i) * s;
        }
    }
    return fail;
}

}  // namespace bse
