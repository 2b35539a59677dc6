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
    std::vector<zc> T;     // ncv x ncv, column-major
    int mp = 0;            // processed columns (T is mp x mp); the basis holds mp + k columns
    uint64_t seed, rng = 0;
    bse_info_t info{};
    double normest = 0.0;

    char *col(DevBuf &b, int64_t c) { return (char *)b.p + (size_t)c * ld * 16; }

    // upload S (rows x l complex, host column-major ld = ldS) in coefficient layout and form out = basis * S
    bse_status_t rotate(DevBuf &basis, int rows, const zc *S, int ldS, int l, void *out, int64_t ldo_c)
    {
        const bool cplx = !full;
        const int ldo = cplx ? 2 * rows : rows;
        std::vector<double> c((size_t)ldo * l);
        for (int j = 0; j < l; ++j)
            for (int a = 0; a < rows; ++a) {
                c[a + (size_t)j * ldo] = S[a + (size_t)j * ldS].real();
                if (cplx) c[a + rows + (size_t)j * ldo] = S[a + (size_t)j * ldS].imag();
            }
        BSE_CUDA(cudaMemcpyAsync(coef.p, c.data(), c.size() * 8, cudaMemcpyHostToDevice, h->stream));
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        return gemm_basis(h, basis.p, ld, rows, cplx, (const double *)coef.p, ldo, l, n, out, ldo_c, 1.0, 0.0);
    }

    // W = V[:, c0+k .. c0+2k) <- operator applied to the block at c0 (TDA: R x;  full: M(P x), reading S4)
    bse_status_t apply_block(int c0)
    {
        if (!full) {
            ST(zero_block(h, col(V, c0 + k), ld, n, k));
            ST(launch_apply_pass(h, h->R, 0, 1.0, col(V, c0), ld, col(V, c0 + k), ld, k));
            ST(comm_sum_block(h, col(V, c0 + k), ld, n, k));
        } else {
            bse_status_t st = bse_apply_half(h, -1, col(PV, c0), ld, col(V, c0 + k), ld, k);      // W = M(p)
            if (st) return st;
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
        double e_in = 0.0, e_after = 0.0, g_after = 0.0;
        ST(block_norm_scale(h, col(V, m), ld, nullptr, ld, k, false, &e_in));
        ST(project_block(h, V.p, ld, m, PV.p, ld, col(V, m), ld, k, nullptr, ld, false, Hc));
        bse_status_t st = bse_apply_half(h, +1, col(V, m), ld, col(PV, m), ld, k);                // PW = P(W)
        if (st) return st;
        ST(block_norm_scale(h, col(V, m), ld, nullptr, ld, k, false, &e_after));
        ST(block_norm_scale(h, col(V, m), ld, col(PV, m), ld, k, false, &g_after));
        // scale of the incoming block in the P-norm, estimated through the Euclidean norms
        double scale2 = (e_after > 0.0) ? g_after * (e_in / e_after) : g_after;
        return normalize_block(h, V.p, ld, m, PV.p, ld, col(V, m), ld, k, col(PV, m), ld, false, scale2, Hc, B, rank,
                               seed, &rng);
    }
};

}  // namespace bse

using namespace bse;

extern "C" bse_status_t bse_solve(bse_handle_t h, int32_t nev, int32_t k, int32_t ncv, double tol, int32_t max_restarts,
                                  uint64_t seed, double *hOmega, void *dVec, int64_t ldvec, double *hResid,
                                  bse_info_t *info_out)
{
    if (!h || nev < 1 || k < 1 || !hOmega || !dVec || !(tol > 0.0) || max_restarts < 0) return BSE_ERR_INVALID_ARG;
    if (is_incomplete(h)) return BSE_ERR_INVALID_ARG;
    const int64_t n = h->N;
    const bool full = (h->mode == BSE_MODE_FULL);
    if ((int64_t)nev + k > n || ldvec < (full ? 2 * n : n)) return BSE_ERR_INVALID_ARG;
    const int64_t dim = full ? 2 * n : n;               // real-linear (full) / complex (TDA) dimension of the space
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
    s.h = h; s.n = n; s.full = full; s.nev = nev; s.k = k; s.ncv = ncv; s.tol = tol; s.ld = n; s.seed = seed;
    s.info.ncv = ncv;
    const size_t basis_bytes = (size_t)n * (ncv + k) * 16;
    ST(s.V.alloc(basis_bytes));
    if (full) ST(s.PV.alloc(basis_bytes));
    ST(s.rot.alloc((size_t)n * (ncv + k) * 16));
    ST(s.coef.alloc((size_t)2 * ncv * ncv * 8));
    ST(s.omega_d.alloc((size_t)nev * 8));
    s.T.assign((size_t)ncv * ncv, zc(0.0));
    const int ldT = ncv;
    ST(orth_reserve(h, ncv + k, k));

    // ---- start block: random, orthonormalised in the active inner product
    ST(fill_random_block(h, s.V.p, s.ld, n, k, seed, s.rng));
    s.rng += k;
    if (full) {
        bse_status_t st = bse_apply_half(h, +1, s.V.p, s.ld, s.PV.p, s.ld, k);
        if (st) return st;
    }
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
    int nz = 0;

    while (true) {
        // ---- one block step: apply (a2 / a3), orthogonalise (a5-a7), extend T
        double t0 = now_s();
        ST(s.apply_block(s.mp));
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        double t1 = now_s();
        s.info.seconds_apply += t1 - t0;
        const int m = s.mp + k;
        int rank = 0;
        {
            bse_status_t st_o = s.orth_new_block(m, Hc.data(), B.data(), &rank);
            if (verbose && st_o) fprintf(stderr, "[bse_solve] orthogonalisation failed (%d) at m = %d\n", (int)st_o, m);
            if (st_o) return st_o;
        }
        s.info.seconds_orth += now_s() - t1;
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

        // ---- Rayleigh-Ritz on the projected matrix (a8)
        double t2 = now_s();
        const int mp = s.mp;
        nz = std::min(mp, (mp + nwant) / 2 + 1);
        S.assign((size_t)mp * nz, zc(0.0));
        if (full) {
            // real coefficients (reading S4): T is real symmetric -> the real driver, a quarter of the reduction flops
            std::vector<double> Ar((size_t)mp * mp), Sr((size_t)mp * nz);
            for (int j = 0; j < mp; ++j)
                for (int i = 0; i < mp; ++i) Ar[i + (size_t)j * mp] = s.T[i + (size_t)j * ldT].real();
            if (host_syev(mp, Ar.data(), mp, theta.data(), Sr.data(), mp, nz)) return BSE_ERR_INTERNAL;
            for (size_t q = 0; q < Sr.size(); ++q) S[q] = zc(Sr[q], 0.0);
        } else {
            A.assign((size_t)mp * mp, zc(0.0));
            for (int j = 0; j < mp; ++j)
                for (int i = 0; i < mp; ++i) A[i + (size_t)j * mp] = s.T[i + (size_t)j * ldT];
            if (host_heev(mp, A.data(), mp, theta.data(), S.data(), mp, nz)) return BSE_ERR_INTERNAL;
        }
        // sharded operator: rank 0's decomposition is everyone's (the host eigensolver's threaded sums may differ in the last bit)
        ST(comm_bcast_host(h, theta.data(), sizeof(double) * mp));
        ST(comm_bcast_host(h, S.data(), sizeof(zc) * (size_t)mp * nz));
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
        double tmax = std::max(std::fabs(theta[0]), std::fabs(theta[mp - 1]));
        if (verbose) fprintf(stderr, "[bse_solve] restart %d mp %d theta0 %.6e theta_max %.6e\n", restarts, mp, theta[0], theta[mp - 1]);
        if (full && !(theta[0] > 0.0)) return BSE_ERR_NOT_POSITIVE_DEFINITE;
        s.normest = std::max(s.normest, full ? std::sqrt(tmax) : tmax);
        for (int i = 0; i < nz; ++i) {
            std::vector<zc> c(k, zc(0.0));
            for (int a = 0; a < k; ++a)
                for (int b = 0; b < k; ++b) c[a] += B[a + (size_t)b * k] * S[(mp - k + b) + (size_t)i * mp];
            double r2 = 0.0;
            for (int a = 0; a < k; ++a)
                for (int b = 0; b < k; ++b) r2 += (std::conj(c[a]) * E[a + (size_t)b * k] * c[b]).real();
            double r = std::sqrt(std::max(r2, 0.0));
            if (full) r /= std::sqrt(2.0 * std::sqrt(theta[i]));     // |Hv - wv| for v^H Sigma v = 1 (reading S4)
            resid[i] = r;
        }
        // ---- convergence of the wanted pairs (leading Ritz values must all be converged)
        int nconv = 0, nfound = 0;
        sel.clear();
        for (int i = 0; i < nz; ++i) {
            if (!(resid[i] <= tol * s.normest)) break;
            ++nconv;
            bool newc = true;
            if (full && !sel.empty()) newc = (theta[i] - theta[sel.back()]) > 1e-7 * std::fabs(theta[i]);
            if (newc) { sel.push_back(i); ++nfound; }
            if (nfound == nev) break;
        }
        s.info.nconv = nfound;
        s.info.seconds_project += now_s() - t2;
        const bool done = (nfound >= nev);
        if (done || restarts >= max_restarts) {
            result = done ? BSE_OK : BSE_ERR_NOT_CONVERGED;
            if (!done) {   // best estimates: the first nev distinct Ritz values
                sel.clear();
                for (int i = 0; i < nz && (int)sel.size() < nev; ++i)
                    if (!full || sel.empty() || (theta[i] - theta[sel.back()]) > 1e-7 * std::fabs(theta[i])) sel.push_back(i);
                for (int i = 0; (int)sel.size() < nev && i < nz; ++i)
                    if (std::find(sel.begin(), sel.end(), i) == sel.end()) sel.push_back(i);
                std::sort(sel.begin(), sel.end());
            }
            break;
        }
        // ---- thick restart (a9): keep l Ritz vectors and the residual block
        double t3 = now_s();
        double keep = 0.5;                                   // fraction of the unconverged part of the basis kept (reading S6)
        if (const char *e = getenv("BSE_KEEP_FRACTION")) { double v = atof(e); if (v > 0.05 && v < 0.95) keep = v; }
        int l = std::min(nconv, nwant) + (int)((mp - std::min(nconv, nwant)) * keep);
        l = std::max(l, std::min(nwant, nz));
        l = std::min(l, std::min(nz, ncv - k));
        ST(s.rotate(s.V, mp, S.data(), mp, l, s.rot.p, n));
        ST(copy_block(h, s.col(s.V, mp), s.ld, s.col(s.rot, l), s.ld, n, k));       // residual block after the Ritz block
        ST(copy_block(h, s.rot.p, s.ld, s.V.p, s.ld, n, l + k));
        if (full) {
            ST(s.rotate(s.PV, mp, S.data(), mp, l, s.rot.p, n));
            ST(copy_block(h, s.col(s.PV, mp), s.ld, s.col(s.rot, l), s.ld, n, k));
            ST(copy_block(h, s.rot.p, s.ld, s.PV.p, s.ld, n, l + k));
        }
        std::fill(s.T.begin(), s.T.end(), zc(0.0));
        for (int i = 0; i < l; ++i) s.T[i + (size_t)i * ldT] = theta[i];
        s.mp = l;
        ++restarts;
        s.info.n_restart = restarts;
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        s.info.seconds_restart += now_s() - t3;
    }

    // ---- eigenvalues, eigenvectors (a10)
    const int mp = s.mp;
    const int nsel = (int)sel.size();
    std::vector<zc> Ssel((size_t)mp * nev, zc(0.0));
    std::vector<double> om(nev, 0.0);
    for (int j = 0; j < nev && j < nsel; ++j) {
        const int i = sel[j];
        for (int a = 0; a < mp; ++a) Ssel[a + (size_t)j * mp] = S[a + (size_t)i * mp];
        om[j] = full ? std::sqrt(std::max(theta[i], 0.0)) : theta[i];
        hOmega[j] = om[j];
        if (hResid) hResid[j] = resid[i];
    }
    if (!full) {
        ST(s.rotate(s.V, mp, Ssel.data(), mp, nev, dVec, ldvec));
    } else {
        // x = X s, px = PX s;  v = [x + px/w; conj(x - px/w)] sqrt(w)/2
        ST(s.rotate(s.V, mp, Ssel.data(), mp, nev, s.rot.p, n));
        ST(s.rotate(s.PV, mp, Ssel.data(), mp, nev, s.V.p, n));     // X is no longer needed: reuse its storage
        BSE_CUDA(cudaMemcpyAsync(s.omega_d.p, om.data(), sizeof(double) * nev, cudaMemcpyHostToDevice, h->stream));
        ST(assemble_full_vectors(h, s.rot.p, s.V.p, n, nev, (const double *)s.omega_d.p, dVec, ldvec));
    }
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    return result;
}
