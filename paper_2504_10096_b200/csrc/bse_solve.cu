// bse_solve: thick-restart block Lanczos (SURVEY.md 8(a) chain a1-a10).
//   TDA : Hermitian block Lanczos on R, complex Euclidean inner product.
//   FULL: structure-preserving variant (reading S4): half vectors x in C^N, operator G = M o P with
//         P(x) = R x + C conj(x), M(y) = R y - C conj(y), real inner product <x, z>_P = Re(x^H P(z)), real
//         coefficients, two stored bases X and PX = P(X).  G has the eigenvalues omega^2 (each twice in R^2N).
// The host loop only sequences kernels, keeps the small projected matrix T and calls the host eigensolver.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <complex>
#include <vector>
#include <cstdio>
#include <cstdlib>

#include "bse_internal.h"

namespace bse {

typedef std::complex<double> zc;

#define ST(call)                          \
    do {                                  \
        bse_status_t st__ = (call);       \
        if (st__ != BSE_OK) { return st__; } \
    } while (0)

struct DevBuf {
    void *p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    bse_status_t alloc(size_t bytes)
    {
        if (cudaMalloc(&p, bytes ? bytes : 16) != cudaSuccess) { cudaGetLastError(); p = nullptr; return BSE_ERR_ALLOC; }
        return BSE_OK;
    }
};

static double now_s()
{
    return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

struct Solver {
    bse_handle_s *h;
    int64_t n;
    bool full;
    int nev, k, ncv;
    double tol;
    int64_t ld;            // leading dimension of the basis buffers (= n)
    DevBuf V, PV, rot, coef, omega_d;
    // variant BSE_VARIANT_GRUNING (reading R9): the sign -1 Lanczos vectors Y and their images MY = M(Y); Bm (ncv x ncv, real,
    // column-major) holds the Y-coefficients of P(X): P(X) = Y Bm, so that the projected matrix of H is [[0, Bm^T], [Bm, 0]]
    int variant = 0;
    DevBuf Yb, MYb;
    std::vector<double> Bm;
    std::vector<zc> B1;     // k x k factor of the last Y block
    std::vector<zc> T;     // ncv x ncv, column-major
    int mp = 0;            // processed columns (T is mp x mp); the basis holds mp + k columns
    // TDA: converged leading Ritz pairs are LOCKED at a restart: they stay in V[:, 0:nlock) (every new block is still
    // orthogonalised against them), their coupling to the rest of the projected matrix -- residual-sized, below tol ||H|| -- is
    // dropped, and the Rayleigh-Ritz problem and the Ritz rotation work on the active columns [nlock, mp) only
    int nlock = 0;
    std::vector<double> th_lock, res_lock;
    uint64_t seed, rng = 0;
    bse_info_t info{};
    double normest = 0.0;
    // device-side timing of the applies (no host synchronisation for the clock): ev[0..1] around the block apply, ev[2..3]
    // around the P(W) apply issued between projection and normalisation in full mode
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    bool timed_second_apply = false;
    ~Solver() { for (auto &e : ev) if (e) cudaEventDestroy(e); }

    // || <V, V> - I ||_F over the first mtot basis columns in the active inner product (reading S10)
    bse_status_t basis_orth_error(int mtot, double *err)
    {
        const bool cplx = !full;
        ST(gram_basis(h, cplx ? V.p : PV.p, ld, mtot, V.p, ld, mtot, cplx, n, (double *)coef.p));
        const int ldo = cplx ? 2 * mtot : mtot;
        std::vector<double> g((size_t)ldo * mtot);
        BSE_CUDA(cudaMemcpyAsync(g.data(), coef.p, g.size() * 8, cudaMemcpyDeviceToHost, h->stream));
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        double s2 = 0.0;
        for (int b = 0; b < mtot; ++b)
            for (int a = 0; a < mtot; ++a) {
                const double re = g[a + (size_t)b * ldo] - (a == b ? 1.0 : 0.0);
                const double im = cplx ? g[a + mtot + (size_t)b * ldo] : 0.0;
                s2 += re * re + im * im;
            }
        *err = std::sqrt(s2);
        return BSE_OK;
    }

    char *col(DevBuf &b, int64_t c) { return (char *)b.p + (size_t)c * ld * 16; }

    // upload S (rows x l complex, host column-major ld = ldS) to `coef` in the coefficient layout gemm_basis consumes
    bse_status_t upload_coef(const zc *S, int rows, int ldS, int l, bool cplx)
    {
        const int ldo = cplx ? 2 * rows : rows;
        std::vector<double> c((size_t)ldo * l);
        for (int j = 0; j < l; ++j)
            for (int a = 0; a < rows; ++a) {
                c[a + (size_t)j * ldo] = S[a + (size_t)j * ldS].real();
                if (cplx) c[a + rows + (size_t)j * ldo] = S[a + (size_t)j * ldS].imag();
            }
        BSE_CUDA(cudaMemcpyAsync(coef.p, c.data(), c.size() * 8, cudaMemcpyHostToDevice, h->stream));
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        return BSE_OK;
    }
    // out = basis * S  (complex S in the TDA case, real S in full mode)
    bse_status_t rotate(const void *basis, int rows, const zc *S, int ldS, int l, void *out, int64_t ldo_c)
    {
        const bool cplx = !full;
        ST(upload_coef(S, rows, ldS, l, cplx));
        return gemm_basis(h, basis, ld, rows, cplx, (const double *)coef.p, cplx ? 2 * rows : rows, l, n, out, ldo_c,
                          1.0, 0.0);
    }

    // Full mode, reading R1: on C^N = R^2N every omega^2 is a double eigenvalue of G = M o P (x and K x = i P(x) / omega
    // give the same eigenvector of H up to the phase i), a block iteration finds both copies, and a genuinely degenerate
    // omega has four.  Which of the first `nc` Ritz pairs are DISTINCT eigenpairs of H is therefore decided from the
    // vectors, never from the values: with x_a = X s_a, p_a = PX s_a, y_a = p_a / w_a, v_a = [x_a + y_a; conj(x_a - y_a)] sqrt(w_a)/2,
    //     v_a^H Sigma v_b = sqrt(w_a w_b)/2 * ( Re(x_a^H p_b)/w_b + Re(x_b^H p_a)/w_a + i [Im(x_a^H x_b) + Im(p_a^H p_b)/(w_a w_b)] ),
    // i.e. one complex Gram matrix of [x | p] on the device.  Runs of Ritz values closer than 1e-6 relative are taken
    // together and a pivoted Cholesky of their Sigma-Gram block keeps a maximal independent set (pivot > 1e-4: a copy
    // leaves the square of the eigenvector error, an independent eigenvector of a degenerate omega at least 2/3 in the
    // best pivot); different runs are Sigma-orthogonal to eigenvector accuracy.  Outputs: sel (candidate index of every
    // returned pair, ascending, at most nev), Cm (nc x nev complex, column-major): returned vector j = sum_a v_a Cm[a, j]
    // is Sigma-normalised and Sigma-orthogonal to the others of its run.  Leaves x in rot[:, 0:nc), p in rot[:, nc:2nc).
    // pad: fill up to nev pairs with rejected candidates (best estimates when the iteration did not converge).
    bse_status_t select_distinct(int mp, const std::vector<zc> &S, const std::vector<double> &theta, int nc, bool pad,
                                 std::vector<int> &sel, std::vector<zc> &Cm)
    {
        ST(rotate(V.p, mp, S.data(), mp, nc, rot.p, n));
        ST(rotate(PV.p, mp, S.data(), mp, nc, col(rot, nc), n));
        const int m2 = 2 * nc, ldo = 2 * m2;
        ST(gram_basis(h, rot.p, ld, m2, rot.p, ld, m2, true, n, (double *)coef.p));
        std::vector<double> g((size_t)ldo * m2);
        BSE_CUDA(cudaMemcpyAsync(g.data(), coef.p, g.size() * 8, cudaMemcpyDeviceToHost, h->stream));
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        auto G = [&](int a, int b) { return zc(g[a + (size_t)b * ldo], g[a + m2 + (size_t)b * ldo]); };   // Z^H Z, Z = [x | p]
        std::vector<double> w(nc);
        for (int a = 0; a < nc; ++a) w[a] = std::sqrt(std::max(theta[a], 0.0));
        std::vector<zc> Gs((size_t)nc * nc);
        for (int b = 0; b < nc; ++b)
            for (int a = 0; a < nc; ++a) {
                const double re = G(a, nc + b).real() / w[b] + G(b, nc + a).real() / w[a];
                const double im = G(a, b).imag() + G(nc + a, nc + b).imag() / (w[a] * w[b]);
                Gs[a + (size_t)b * nc] = 0.5 * std::sqrt(w[a] * w[b]) * zc(re, im);
            }
        sel.clear();
        Cm.assign((size_t)nc * nev, zc(0.0));
        std::vector<int> rejected;
        for (int r0 = 0; r0 < nc && (int)sel.size() < nev;) {
            int r1 = r0 + 1;
            while (r1 < nc && theta[r1] - theta[r1 - 1] <= 1e-6 * std::fabs(theta[r1])) ++r1;
            const int q = r1 - r0;
            // pivoted Cholesky of the run's Sigma-Gram block: A = L L^H on the accepted (pivot) candidates
            std::vector<zc> L((size_t)q * q, zc(0.0));
            std::vector<double> left(q);
            std::vector<int> piv;
            std::vector<char> used(q, 0);
            for (int a = 0; a < q; ++a) left[a] = Gs[(r0 + a) + (size_t)(r0 + a) * nc].real();
            while ((int)piv.size() < q) {
                int best = -1;
                for (int a = 0; a < q; ++a)
                    if (!used[a] && (best < 0 || left[a] > left[best])) best = a;
                if (best < 0 || !(left[best] > 1e-4)) break;
                const int j = (int)piv.size();
                used[best] = 1;
                piv.push_back(best);
                const double d = std::sqrt(left[best]);
                // column j of L for every candidate a of the run (row index a): L[a, j] = (A[a, best] - sum_i L[a, i] conj(L[best, i])) / d
                for (int a = 0; a < q; ++a) {
                    zc v = Gs[(r0 + a) + (size_t)(r0 + best) * nc];
                    for (int i = 0; i < j; ++i) v -= L[a + (size_t)i * q] * std::conj(L[best + (size_t)i * q]);
                    L[a + (size_t)j * q] = v / d;
                    if (!used[a]) left[a] -= std::norm(L[a + (size_t)j * q]);
                }
                left[best] = 0.0;
            }
            for (int a = 0; a < q; ++a)
                if (!used[a]) rejected.push_back(r0 + a);
            // orthonormal combinations: with Lp = L restricted to the pivot rows (lower triangular in pivot order),
            // [v_piv] Lp^-H is Sigma-orthonormal.  Returned in ascending candidate order.
            const int na = (int)piv.size();
            std::vector<zc> Linv((size_t)na * na, zc(0.0));            // Lp^-1, lower triangular
            for (int c = 0; c < na; ++c) {
                Linv[c + (size_t)c * na] = 1.0 / L[piv[c] + (size_t)c * q];
                for (int r = c + 1; r < na; ++r) {
                    zc v(0.0);
                    for (int i = c; i < r; ++i) v += L[piv[r] + (size_t)i * q] * Linv[i + (size_t)c * na];
                    Linv[r + (size_t)c * na] = -v / L[piv[r] + (size_t)r * q];
                }
            }
            std::vector<int> order(na);
            for (int c = 0; c < na; ++c) order[c] = c;
            std::sort(order.begin(), order.end(), [&](int a, int b) { return piv[a] < piv[b]; });
            for (int oi = 0; oi < na && (int)sel.size() < nev; ++oi) {
                const int c = order[oi], j = (int)sel.size();          // output j = sum_{r <= c} v_{piv[r]} conj(Linv[c, r])
                for (int r = 0; r <= c; ++r) Cm[(r0 + piv[r]) + (size_t)j * nc] = std::conj(Linv[c + (size_t)r * na]);
                sel.push_back(r0 + piv[c]);
            }
            r0 = r1;
        }
        if (pad)
            for (size_t i = 0; i < rejected.size() && (int)sel.size() < nev; ++i) {
                const int a = rejected[i], j = (int)sel.size();
                const double d = Gs[a + (size_t)a * nc].real();
                Cm[a + (size_t)j * nc] = d > 0.0 ? 1.0 / std::sqrt(d) : 1.0;
                sel.push_back(a);
            }
        return BSE_OK;
    }

    // W = V[:, c0+k .. c0+2k) <- operator applied to the block at c0 (TDA: R x;  full: M(P x), reading S4)
    bse_status_t apply_block(int c0)
    {
        if (!full) {
            ST(apply_vec(h, 0, col(V, c0), ld, col(V, c0 + k), ld, k));
        } else if (variant == BSE_VARIANT_GRUNING) {
            // u_{2j} = [y; -conj y]: H u_{2j-1} has the half vector P(x_j); orthonormalise it against the stored vectors of its
            // sign in the Omega inner product, <y_i, z>_M = Re(M(y_i)^H z) -- image recomputed after the projection (reading R3)
            const int my = c0;                                                                   // Y columns so far
            std::vector<zc> Hc1((size_t)std::max(my, 1) * k, zc(0.0));
            int rank = 0;
            ST(copy_block(h, col(PV, c0), ld, col(Yb, my), ld, n, k));
            ST(block_norm_scale(h, col(Yb, my), ld, nullptr, ld, k, false, ORTH_E_IN));
            ST(project_block(h, Yb.p, ld, my, MYb.p, ld, col(Yb, my), ld, k, nullptr, ld, false));
            bse_status_t st = bse_apply_half(h, -1, col(Yb, my), ld, col(MYb, my), ld, k);     // M(z)
            if (st) return st;
            ST(block_norm_scale(h, col(Yb, my), ld, nullptr, ld, k, false, ORTH_E_AFTER));
            ST(block_norm_scale(h, col(Yb, my), ld, col(MYb, my), ld, k, false, ORTH_G));
            B1.assign((size_t)k * k, zc(0.0));
            ST(normalize_block(h, Yb.p, ld, my, MYb.p, ld, col(Yb, my), ld, k, col(MYb, my), ld, false, 1, Hc1.data(),
                               B1.data(), &rank, seed, &rng, -1));
            for (int c = 0; c < k; ++c) {                                                        // P(X_j) = Y[:, :my] Hc1 + Y_j B1
                for (int a = 0; a < my; ++a) Bm[a + (size_t)(c0 + c) * ncv] = Hc1[a + (size_t)c * my].real();
                for (int a = 0; a < k; ++a) Bm[(my + a) + (size_t)(c0 + c) * ncv] = B1[a + (size_t)c * k].real();
            }
            // H u_{2j} has the half vector M(y_j): the next sign +1 candidate
            ST(copy_block(h, col(MYb, my), ld, col(V, c0 + k), ld, n, k));
        } else {
            ST(apply_vec(h, -1, col(PV, c0), ld, col(V, c0 + k), ld, k));                          // W = M(p)
        }
        info.n_apply += 1;
        return BSE_OK;
    }

    // Orthogonalise the new block at column m against the first m columns and orthonormalise it (a5-a7).
    // Full mode follows the oracle's order: project W, THEN pw = P(w) (a fresh apply), then the P-norm.
    bse_status_t orth_new_block(int m, void *Hc, void *B, int *rank)
    {
        if (!full)
            return orth_block(h, V.p, ld, m, nullptr, ld, col(V, m), ld, k, nullptr, ld, Hc, B, rank, seed, &rng);
        // the P-norm scale of the incoming block is estimated through Euclidean norms (device scalars, no host round trip)
        ST(block_norm_scale(h, col(V, m), ld, nullptr, ld, k, false, ORTH_E_IN));
        ST(project_block(h, V.p, ld, m, PV.p, ld, col(V, m), ld, k, nullptr, ld, false));
        BSE_CUDA(cudaEventRecord(ev[2], h->stream));
        ST(apply_vec(h, +1, col(V, m), ld, col(PV, m), ld, k));                                   // PW = P(W)
        BSE_CUDA(cudaEventRecord(ev[3], h->stream));
        timed_second_apply = true;
        info.n_apply += 1;
        ST(block_norm_scale(h, col(V, m), ld, nullptr, ld, k, false, ORTH_E_AFTER));
        ST(block_norm_scale(h, col(V, m), ld, col(PV, m), ld, k, false, ORTH_G));
        return normalize_block(h, V.p, ld, m, PV.p, ld, col(V, m), ld, k, col(PV, m), ld, false, 1, Hc, B, rank,
                               seed, &rng);
    }
};

}  // namespace bse

using namespace bse;

extern "C" bse_status_t bse_solve(bse_handle_t h, int32_t nev, int32_t k, int32_t ncv, double tol, int32_t max_restarts,
                                  uint64_t seed, double *hOmega, void *dVec, int64_t ldvec, double *hResid,
                                  bse_info_t *info_out)
{
    return bse_solve_variant(h, BSE_VARIANT_SHAO, nev, k, ncv, tol, max_restarts, seed, hOmega, dVec, ldvec, hResid, info_out);
}

extern "C" bse_status_t bse_solve_variant(bse_handle_t h, int32_t variant, int32_t nev, int32_t k, int32_t ncv, double tol,
                                          int32_t max_restarts, uint64_t seed, double *hOmega, void *dVec, int64_t ldvec,
                                          double *hResid, bse_info_t *info_out)
{
    if (!h || nev < 1 || k < 1 || !hOmega || !dVec || !(tol > 0.0) || max_restarts < 0) return BSE_ERR_INVALID_ARG;
    if (variant != BSE_VARIANT_SHAO && variant != BSE_VARIANT_GRUNING) return BSE_ERR_INVALID_ARG;
    if (h->mode != BSE_MODE_FULL) variant = BSE_VARIANT_SHAO;          // TDA: the Hermitian iteration has no variants
    if (is_incomplete(h)) return BSE_ERR_INVALID_ARG;
    // n: rows of every vector held here -- all N, or this rank's rows [vr_begin, vr_end) under bse_set_row_partition (the
    // dense kernels then work on the local rows, their Gram matrices are summed over the ranks, and apply_vec gathers the
    // operand block of every product); the returned eigenvectors are gathered to full length on every rank
    const bool rowpart = is_row_partitioned(h);
    if (rowpart && (!h->comm || variant == BSE_VARIANT_GRUNING)) return BSE_ERR_INVALID_ARG;
    const int64_t Nfull = h->N, n = vec_rows(h);
    const bool full = (h->mode == BSE_MODE_FULL);
    if ((int64_t)nev + k > Nfull || ldvec < (full ? 2 * Nfull : Nfull)) return BSE_ERR_INVALID_ARG;
    const int64_t dim = full ? 2 * Nfull : Nfull;       // real-linear (full) / complex (TDA) dimension of the space
    const int nwant = full ? 2 * nev : nev;             // Ritz values of G come in pairs in full mode
    if (ncv <= 0) {
        ncv = std::max(2 * nev, nev + 15);
        if (full) ncv *= 2;
        // a wide block needs room to iterate between restarts: with fewer than ~8 block steps per cycle the thick restart
        // stagnates (full mode, nev = 16, k = 8, ncv = 64: 889 restarts; ncv = 160: 46)
        ncv = std::max(ncv, nwant + 8 * k);
    }
    ncv = ((ncv + k - 1) / k) * k;
    if ((int64_t)ncv + k > dim) ncv = (int)(((dim - k) / k) * k);
    if (ncv < nwant + k && (int64_t)ncv + k < dim) ncv = ((nwant + k + k - 1) / k) * k;
    if (ncv < 2 * k || (int64_t)ncv + k > dim) return BSE_ERR_INVALID_ARG;

    const double t_start = now_s();
    Solver s;
    struct InfoGuard {      // report progress on every exit path
        bse_info_t *out; Solver *sv; double t0;
        ~InfoGuard() { if (out) { sv->info.norm_est = sv->normest; sv->info.seconds_total = now_s() - t0; *out = sv->info; } }
    } guard{info_out, &s, t_start};
    const bool verbose = getenv("BSE_VERBOSE") != nullptr;
    bool lock_on = true;                                          // BSE_SOLVE_LOCK=0: no locking (A/B tests)
    if (const char *e = getenv("BSE_SOLVE_LOCK")) lock_on = atoi(e) != 0;
    s.h = h; s.n = n; s.full = full; s.nev = nev; s.k = k; s.ncv = ncv; s.tol = tol; s.ld = n; s.seed = seed;
    s.variant = variant;
    for (auto &e : s.ev) BSE_CUDA(cudaEventCreate(&e));
    const bool gruning = variant == BSE_VARIANT_GRUNING;
    s.info.ncv = ncv;
    const size_t basis_bytes = (size_t)n * (ncv + k) * 16;
    ST(s.V.alloc(basis_bytes));
    if (full) ST(s.PV.alloc(basis_bytes));
    if (gruning) {
        ST(s.Yb.alloc(basis_bytes));
        ST(s.MYb.alloc(basis_bytes));
        s.Bm.assign((size_t)ncv * ncv, 0.0);
    }
    ST(s.rot.alloc((size_t)n * (ncv + k) * 16));
    const int ncmax = (ncv + k) / 2;                    // full mode: candidates of the multiplicity test (x and P x side by side in rot)
    ST(s.coef.alloc((size_t)2 * (ncv + k) * (ncv + k) * 8));
    ST(s.omega_d.alloc((size_t)std::max(nev, ncmax) * 8));
    s.T.assign((size_t)ncv * ncv, zc(0.0));
    const int ldT = ncv;
    ST(orth_reserve(h, ncv + k, k));

    // ---- start block: random, orthonormalised in the active inner product
    ST(fill_random_block(h, s.V.p, s.ld, n, k, seed, s.rng));
    s.rng += k;
    if (full) ST(apply_vec(h, +1, s.V.p, s.ld, s.PV.p, s.ld, k));
    {
        int rank = 0;
        ST(orth_block(h, nullptr, s.ld, 0, full ? s.PV.p : nullptr, s.ld, s.V.p, s.ld, k, full ? s.PV.p : nullptr, s.ld,
                      nullptr, nullptr, &rank, seed, &s.rng));
    }

    std::vector<zc> Hc((size_t)(ncv + k) * k), B((size_t)k * k), A, S;
    std::vector<double> theta(ncv), resid;
    bse_status_t result = BSE_ERR_NOT_CONVERGED;
    int restarts = 0;
    std::vector<int> sel;          // Ritz indices returned
    std::vector<zc> Cm;            // full mode: returned vectors as combinations of the candidate vectors (select_distinct)
    int nz = 0, ncand = 0;

    while (true) {
        // ---- one block step: apply (a2 / a3), orthogonalise (a5-a7), extend T
        double t0 = now_s();
        BSE_CUDA(cudaEventRecord(s.ev[0], h->stream));
        ST(s.apply_block(s.mp));
        BSE_CUDA(cudaEventRecord(s.ev[1], h->stream));
        const int m = s.mp + k;
        int rank = 0;
        s.timed_second_apply = false;
        {
            bse_status_t st_o = s.orth_new_block(m, Hc.data(), B.data(), &rank);      // ends with the step's one synchronisation
            if (verbose && st_o) fprintf(stderr, "[bse_solve] orthogonalisation failed (%d) at m = %d\n", (int)st_o, m);
            if (st_o) return st_o;
        }
        {
            float ms_a = 0.f, ms_b = 0.f;
            BSE_CUDA(cudaEventElapsedTime(&ms_a, s.ev[0], s.ev[1]));
            if (s.timed_second_apply) BSE_CUDA(cudaEventElapsedTime(&ms_b, s.ev[2], s.ev[3]));
            const double t_apply = 1e-3 * ((double)ms_a + (double)ms_b);
            s.info.seconds_apply += t_apply;
            s.info.seconds_orth += (now_s() - t0) - t_apply;
        }
        for (int c = 0; c < k; ++c)
            for (int a = 0; a < m; ++a) {
                zc v = Hc[a + (size_t)c * m];
                if (a >= s.mp) {   // diagonal block: enforce Hermitian symmetry
                    zc u = Hc[(s.mp + c) + (size_t)(a - s.mp) * m];
                    v = 0.5 * (v + std::conj(u));
                }
                s.T[a + (size_t)(s.mp + c) * ldT] = v;
                s.T[(s.mp + c) + (size_t)a * ldT] = std::conj(v);
            }
        s.mp = m;
        if (s.mp + k <= ncv) continue;

        // ---- Rayleigh-Ritz on the projected matrix (a8): the active block [nl, mp) (nl = locked pairs, TDA only)
        double t2 = now_s();
        const int mp = s.mp;
        const int nl = s.nlock, ma = mp - nl, nwant_a = std::max(nwant - nl, 1);
        nz = std::min(ma, (ma + nwant_a) / 2 + 1);
        S.assign((size_t)ma * nz, zc(0.0));
        if (full) {
            // real coefficients (reading S4): T is real symmetric -> the real driver, a quarter of the reduction flops
            std::vector<double> Ar((size_t)mp * mp), Sr((size_t)mp * nz);
            if (gruning) {
                // T = Bm^T Bm: the positive eigenvalues sigma of [[0, Bm^T], [Bm, 0]] are the singular values of Bm, with the
                // same right singular vectors S (sign +1 coefficients); the sign -1 coefficients are U = Bm S / sigma
                const double *Bmp = s.Bm.data();
                double *Arp = Ar.data();
#pragma omp parallel for schedule(dynamic, 8)
                for (int j = 0; j < mp; ++j)
                    for (int i = 0; i <= j; ++i) {
                        double acc = 0.0;
                        for (int a = 0; a < mp; ++a) acc += Bmp[a + (size_t)i * ncv] * Bmp[a + (size_t)j * ncv];
                        Arp[i + (size_t)j * mp] = Arp[j + (size_t)i * mp] = acc;
                    }
            } else
            for (int j = 0; j < mp; ++j)
                for (int i = 0; i < mp; ++i) Ar[i + (size_t)j * mp] = s.T[i + (size_t)j * ldT].real();
            if (host_syev(mp, Ar.data(), mp, theta.data(), Sr.data(), mp, nz)) return BSE_ERR_INTERNAL;
            for (size_t q = 0; q < Sr.size(); ++q) S[q] = zc(Sr[q], 0.0);
        } else {
            A.assign((size_t)ma * ma, zc(0.0));
            for (int j = 0; j < ma; ++j)
                for (int i = 0; i < ma; ++i) A[i + (size_t)j * ma] = s.T[(nl + i) + (size_t)(nl + j) * ldT];
            if (host_heev(ma, A.data(), ma, theta.data(), S.data(), ma, nz)) return BSE_ERR_INTERNAL;
        }
        // sharded operator: rank 0's decomposition is everyone's (the host eigensolver's threaded sums may differ in the last bit)
        ST(comm_bcast_host(h, theta.data(), sizeof(double) * ma));
        ST(comm_bcast_host(h, S.data(), sizeof(zc) * (size_t)ma * nz));
        // residual estimates (a10):  r_i = || X_next B s_last,i ||  (Euclidean)
        std::vector<double> E((size_t)k * k, 0.0);   // Re(X_next^H X_next); identity in the TDA case
        if (full) {
            ST(gram_basis(h, s.col(s.V, mp), s.ld, k, s.col(s.V, mp), s.ld, k, true, n, (double *)s.coef.p));
            std::vector<double> g((size_t)2 * k * k);
            BSE_CUDA(cudaMemcpyAsync(g.data(), s.coef.p, g.size() * 8, cudaMemcpyDeviceToHost, h->stream));
            BSE_CUDA(cudaStreamSynchronize(h->stream));
            for (int j = 0; j < k; ++j)
                for (int i = 0; i < k; ++i) E[i + (size_t)j * k] = g[i + (size_t)j * 2 * k];
        } else {
            for (int i = 0; i < k; ++i) E[i + (size_t)i * k] = 1.0;
        }
        resid.assign(nz, 0.0);
        double tmax = std::max(std::fabs(theta[0]), std::fabs(theta[ma - 1]));
        for (double v : s.th_lock) tmax = std::max(tmax, std::fabs(v));
        if (verbose) fprintf(stderr, "[bse_solve] restart %d mp %d theta0 %.6e theta_max %.6e\n", restarts, mp, theta[0], theta[mp - 1]);
        if (full && !(theta[0] > 0.0)) return BSE_ERR_NOT_POSITIVE_DEFINITE;
        s.normest = std::max(s.normest, full ? std::sqrt(tmax) : tmax);
        std::vector<zc> Beff = B;                      // G x - theta x = X_next Beff s_last;  variant R9: Beff = B2 B1
        if (gruning)
            for (int a = 0; a < k; ++a)
                for (int b = 0; b < k; ++b) {
                    zc acc(0.0);
                    for (int q = 0; q < k; ++q) acc += B[a + (size_t)q * k] * s.B1[q + (size_t)b * k];
                    Beff[a + (size_t)b * k] = acc;
                }
        for (int i = 0; i < nz; ++i) {
            std::vector<zc> c(k, zc(0.0));
            for (int a = 0; a < k; ++a)
                for (int b = 0; b < k; ++b) c[a] += Beff[a + (size_t)b * k] * S[(ma - k + b) + (size_t)i * ma];
            double r2 = 0.0;
            for (int a = 0; a < k; ++a)
                for (int b = 0; b < k; ++b) r2 += (std::conj(c[a]) * E[a + (size_t)b * k] * c[b]).real();
            double r = std::sqrt(std::max(r2, 0.0));
            if (full) r /= std::sqrt(2.0 * std::sqrt(theta[i]));     // |Hv - wv| for v^H Sigma v = 1 (reading S4)
            resid[i] = r;
        }
        // ---- convergence of the wanted pairs (leading Ritz values must all be converged)
        int nconv = 0;
        for (int i = 0; i < nz; ++i) {
            // safety factor (reading S7: "builder may tighten the internal tol for margin"): normest is a LOWER bound of ||H||
            // and the estimate is exact only in exact arithmetic, so pairs accepted at exactly tol ||H||_est sat on the edge of
            // the bound they are certified against (sampled-row residuals of the oracle, tests/test_gpu_solve_configs.py)
            if (!(resid[i] <= 0.9 * tol * s.normest)) break;
            ++nconv;
        }
        bool done;
        if (!full) {
            // wanted = the nev smallest of (locked) + (active Ritz values); converged = the locked ones and the leading
            // converged run of the active ones, counted below the first unconverged active value
            int ntot = nconv;
            const bool open = nconv < ma;                      // an unconverged (or uncomputed) active pair exists
            for (double v : s.th_lock)
                if (!open || v <= theta[nconv]) ++ntot;
            done = ntot >= nev;
            s.info.nconv = std::min(ntot, nev);
        } else {
            // Every eigenpair of H owns exactly two Ritz values of G (reading R1), whatever the multiplicity of omega:
            // 2 nev - 1 leading converged Ritz pairs contain nev distinct eigenpairs, and so do nev value-separated
            // ones (a single-vector iteration sees one copy of each).  WHICH pairs are returned is decided from the
            // vectors (select_distinct), once, when this count says the iteration can stop.
            int nsep = 0;
            for (int i = 0; i < nconv; ++i)
                if (i == 0 || theta[i] - theta[i - 1] > 1e-6 * std::fabs(theta[i])) ++nsep;
            const int lower = std::max(nsep, (nconv + 1) / 2);
            s.info.nconv = std::min(lower, nev);
            done = lower >= nev;
            if (done) {
                ncand = std::min(nconv, ncmax);
                ST(s.select_distinct(mp, S, theta, ncand, false, sel, Cm));
                if ((int)sel.size() < nev) done = false;       // only if ncmax cut the candidate list: keep iterating
            }
        }
        s.info.seconds_project += now_s() - t2;
        if (done || restarts >= max_restarts) {
            result = done ? BSE_OK : BSE_ERR_NOT_CONVERGED;
            if (!full) {
                // the nev smallest of locked + active (best estimates if not converged): indices < nl are locked columns,
                // nl + i is active Ritz pair i
                std::vector<std::pair<double, int>> all;
                for (int j = 0; j < nl; ++j) all.push_back({s.th_lock[j], j});
                for (int i = 0; i < nz; ++i) all.push_back({theta[i], nl + i});
                std::stable_sort(all.begin(), all.end(), [](const std::pair<double, int> &a, const std::pair<double, int> &b) { return a.first < b.first; });
                sel.clear();
                for (int i = 0; i < nev && i < (int)all.size(); ++i) sel.push_back(all[i].second);
            } else if (!done) {                                 // best estimates: the first nev distinct pairs, converged or not
                ncand = std::min(nz, ncmax);
                ST(s.select_distinct(mp, S, theta, ncand, true, sel, Cm));
            }
            break;
        }
        // ---- thick restart (a9): keep l Ritz vectors and the residual block
        double t3 = now_s();
        double keep = 0.5;                                   // fraction of the unconverged part of the basis kept (reading S6)
        if (const char *e = getenv("BSE_KEEP_FRACTION")) { double v = atof(e); if (v > 0.05 && v < 0.95) keep = v; }
        // l counts kept columns INCLUDING the locked ones (the same basis sizes as without locking); la of them are active
        const int nct = std::min(nl + nconv, nwant);
        int l = nct + (int)((mp - nct) * keep);
        l = std::max(l, std::min(nwant, nl + nz));
        l = std::min(l, std::min(nl + nz, ncv - k));
        const int la = l - nl;
        ST(s.rotate(s.col(s.V, nl), ma, S.data(), ma, la, s.rot.p, n));               // the active columns only
        ST(copy_block(h, s.col(s.V, mp), s.ld, s.col(s.rot, la), s.ld, n, k));       // residual block after the Ritz block
        ST(copy_block(h, s.rot.p, s.ld, s.col(s.V, nl), s.ld, n, la + k));
        if (full) {
            ST(s.rotate(s.PV.p, mp, S.data(), mp, l, s.rot.p, n));
            ST(copy_block(h, s.col(s.PV, mp), s.ld, s.col(s.rot, l), s.ld, n, k));
            ST(copy_block(h, s.rot.p, s.ld, s.PV.p, s.ld, n, l + k));
        }
        if (gruning) {
            std::vector<zc> U((size_t)mp * l, zc(0.0));
            const double *Bmp = s.Bm.data();
#pragma omp parallel for schedule(static)
            for (int j = 0; j < l; ++j) {
                std::vector<double> u(mp, 0.0);
                for (int q = 0; q < mp; ++q) {
                    const double sq = S[q + (size_t)j * mp].real();
                    for (int a = 0; a < mp; ++a) u[a] += Bmp[a + (size_t)q * ncv] * sq;
                }
                const double sg = std::sqrt(std::max(theta[j], 1e-300));
                for (int a = 0; a < mp; ++a) U[a + (size_t)j * mp] = u[a] / sg;
            }
            ST(s.rotate(s.Yb.p, mp, U.data(), mp, l, s.rot.p, n));
            ST(copy_block(h, s.rot.p, s.ld, s.Yb.p, s.ld, n, l));
            ST(s.rotate(s.MYb.p, mp, U.data(), mp, l, s.rot.p, n));
            ST(copy_block(h, s.rot.p, s.ld, s.MYb.p, s.ld, n, l));
            std::fill(s.Bm.begin(), s.Bm.end(), 0.0);
            for (int i = 0; i < l; ++i) s.Bm[i + (size_t)i * ncv] = std::sqrt(std::max(theta[i], 0.0));
        }
        std::fill(s.T.begin(), s.T.end(), zc(0.0));
        if (!full) {
            // lock the leading converged active pairs that were kept (never all wanted ones: the last restart decides)
            const int nnew = lock_on ? std::max(0, std::min(std::min(nconv, la), nev - 1 - nl)) : 0;
            for (int i = 0; i < nnew; ++i) { s.th_lock.push_back(theta[i]); s.res_lock.push_back(resid[i]); }
            for (int j = 0; j < nl + nnew; ++j) s.T[j + (size_t)j * ldT] = s.th_lock[j];
            for (int i = nnew; i < la; ++i) s.T[(nl + i) + (size_t)(nl + i) * ldT] = theta[i];
            s.nlock = nl + nnew;
        } else
            for (int i = 0; i < l; ++i) s.T[i + (size_t)i * ldT] = theta[i];
        s.mp = l;
        ++restarts;
        s.info.n_restart = restarts;
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        s.info.seconds_restart += now_s() - t3;
    }

    // ---- eigenvalues, eigenvectors (a10)
    const int mp = s.mp;
    ST(s.basis_orth_error(mp + k, &s.info.basis_orth_err));
    const int nsel = (int)sel.size();
    std::vector<zc> Ssel((size_t)mp * nev, zc(0.0));
    std::vector<double> om(nev, 0.0);
    const int nlf = s.nlock, maf = mp - nlf;                      // S is maf x nz over the active columns (nlf = 0 in full mode)
    for (int j = 0; j < nev && j < nsel; ++j) {
        const int i = sel[j];
        if (!full && i < nlf) {                                    // a locked pair: the column itself
            Ssel[i + (size_t)j * mp] = 1.0;
            om[j] = s.th_lock[i];
            if (hResid) hResid[j] = s.res_lock[i];
        } else {
            const int ia = i - nlf;
            for (int a = 0; a < maf; ++a) Ssel[(nlf + a) + (size_t)j * mp] = S[a + (size_t)ia * maf];
            om[j] = full ? std::sqrt(std::max(theta[ia], 0.0)) : theta[ia];
            if (hResid) hResid[j] = resid[ia];
        }
        hOmega[j] = om[j];
    }
    if (!full) {
        if (!rowpart) ST(s.rotate(s.V.p, mp, Ssel.data(), mp, nev, dVec, ldvec));
        else {
            ST(s.rotate(s.V.p, mp, Ssel.data(), mp, nev, s.rot.p, n));
            ST(zero_block(h, dVec, ldvec, Nfull, nev));
            ST(copy_block(h, s.rot.p, n, (char *)dVec + (size_t)h->vr_begin * 16, ldvec, n, nev));
            ST(comm_sum_block(h, dVec, ldvec, Nfull, nev));
        }
    } else {
        // candidates (left in rot by select_distinct): x = X s, p = PX s;  v = [x + p/w; conj(x - p/w)] sqrt(w)/2, assembled
        // into the storage of X (no longer needed), then the returned vectors are their combinations Cm
        std::vector<double> wc(ncand);
        for (int a = 0; a < ncand; ++a) wc[a] = std::sqrt(std::max(theta[a], 0.0));
        BSE_CUDA(cudaMemcpyAsync(s.omega_d.p, wc.data(), sizeof(double) * ncand, cudaMemcpyHostToDevice, h->stream));
        ST(assemble_full_vectors(h, s.rot.p, s.col(s.rot, ncand), n, ncand, (const double *)s.omega_d.p, s.V.p, 2 * n));
        ST(s.upload_coef(Cm.data(), ncand, ncand, nev, true));
        if (!rowpart)
            ST(gemm_basis(h, s.V.p, 2 * n, ncand, true, (const double *)s.coef.p, 2 * ncand, nev, 2 * n, dVec, ldvec, 1.0, 0.0));
        else {
            // local rows of [X; Y] (2 n x nev) -> their places in the full-length vectors, summed over the ranks
            ST(gemm_basis(h, s.V.p, 2 * n, ncand, true, (const double *)s.coef.p, 2 * ncand, nev, 2 * n, s.rot.p, 2 * n, 1.0, 0.0));
            ST(zero_block(h, dVec, ldvec, 2 * Nfull, nev));
            ST(copy_block(h, s.rot.p, 2 * n, (char *)dVec + (size_t)h->vr_begin * 16, ldvec, n, nev));
            ST(copy_block(h, (char *)s.rot.p + (size_t)n * 16, 2 * n, (char *)dVec + (size_t)(Nfull + h->vr_begin) * 16, ldvec, n, nev));
            ST(comm_sum_block(h, dVec, ldvec, 2 * Nfull, nev));
        }
    }
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    return result;
}
