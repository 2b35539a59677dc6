// Block classical Gram-Schmidt with reorthogonalisation + intra-block orthonormalisation
// (PAPER.md:67, 71).  The host only sequences kernels and factors k x k matrices.
#include <cmath>
#include <complex>
#include <cstring>
#include <vector>

#include "bse_internal.h"

namespace bse {

typedef std::complex<double> zc;

__global__ void scale_block_kernel(double2 *W, int64_t ldw, int64_t n, int k, double alpha)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (i < n && c < k) {
        double2 v = W[i + c * ldw];
        W[i + c * ldw] = make_double2(alpha * v.x, alpha * v.y);
    }
}
static bse_status_t scale_block(bse_handle_s *h, void *W, int64_t ldw, int64_t n, int k, double alpha)
{
    scale_block_kernel<<<dim3((unsigned)((n + 255) / 256), k), 256, 0, h->stream>>>((double2 *)W, ldw, n, k, alpha);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

// device coefficient layout <-> host complex (ld = rows)
static void coef_to_host(const double *c, int m, int k, bool cplx, zc *out, bool accumulate)
{
    const int ldo = cplx ? 2 * m : m;
    for (int col = 0; col < k; ++col)
        for (int a = 0; a < m; ++a) {
            zc v(c[a + (size_t)col * ldo], cplx ? c[a + m + (size_t)col * ldo] : 0.0);
            if (accumulate) out[a + (size_t)col * m] += v; else out[a + (size_t)col * m] = v;
        }
}
static void host_to_coef(const zc *in, int m, int k, bool cplx, double *c)
{
    const int ldo = cplx ? 2 * m : m;
    for (int col = 0; col < k; ++col)
        for (int a = 0; a < m; ++a) {
            c[a + (size_t)col * ldo] = in[a + (size_t)col * m].real();
            if (cplx) c[a + m + (size_t)col * ldo] = in[a + (size_t)col * m].imag();
        }
}

#define ST(call)                         \
    do {                                 \
        bse_status_t st__ = (call);      \
        if (st__ != BSE_OK) return st__; \
    } while (0)

struct OrthWs {
    double *c1, *c2, *g, *binv;   // device coefficient buffers
    double *tmpW, *tmpPW;         // device n x k complex temporaries
    double *hc1, *hc2, *hg, *hbinv;   // pinned host mirrors
};

static bse_status_t orth_ws(bse_handle_s *h, int m, int k, OrthWs &w)
{
    const int64_t n = h->N;
    size_t cm = (size_t)2 * (m > 0 ? m : 1) * k, ck = (size_t)2 * k * k;
    size_t doubles = 2 * cm + 2 * ck + (size_t)4 * n * k;
    ST(ensure_ws2(h, doubles * 8));
    ST(ensure_pin(h, (2 * cm + 2 * ck) * 8));
    double *p = (double *)h->ws2;
    w.tmpW = p; p += (size_t)2 * n * k;         // keep the large blocks first (16-byte aligned)
    w.tmpPW = p; p += (size_t)2 * n * k;
    w.c1 = p; p += cm;
    w.c2 = p; p += cm;
    w.g = p; p += ck;
    w.binv = p;
    double *q = (double *)h->hpin;
    w.hc1 = q; q += cm;
    w.hc2 = q; q += cm;
    w.hg = q; q += ck;
    w.hbinv = q;
    return BSE_OK;
}

// G (k x k, coefficient layout on device) -> host complex, after synchronising the stream
static bse_status_t fetch_coef(bse_handle_s *h, const double *dev, double *pin, int m, int k, bool cplx)
{
    size_t bytes = (size_t)(cplx ? 2 * m : m) * k * 8;
    BSE_CUDA(cudaMemcpyAsync(pin, dev, bytes, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    return BSE_OK;
}

// <W, W> in the active inner product: Euclidean W^H W (complex) or Re(W^H PW) (real)
static bse_status_t block_gram(bse_handle_s *h, const void *W, int64_t ldw, const void *PW, int64_t ldpw, int k,
                               bool cplx, OrthWs &w, std::vector<zc> &G)
{
    ST(gram_basis(h, W, ldw, k, cplx ? W : PW, cplx ? ldw : ldpw, k, cplx, h->N, w.g));
    ST(fetch_coef(h, w.g, w.hg, k, k, cplx));
    G.assign((size_t)k * k, zc(0.0));
    coef_to_host(w.hg, k, k, cplx, G.data(), false);
    return BSE_OK;
}

// W <- W * S (k x k, host complex S), PW likewise (S real in that mode)
static bse_status_t block_times_small(bse_handle_s *h, void *W, int64_t ldw, void *PW, int64_t ldpw, int k, bool cplx,
                                      const zc *S, OrthWs &w)
{
    const int64_t n = h->N;
    host_to_coef(S, k, k, cplx, w.hbinv);
    size_t bytes = (size_t)(cplx ? 2 * k : k) * k * 8;
    BSE_CUDA(cudaMemcpyAsync(w.binv, w.hbinv, bytes, cudaMemcpyHostToDevice, h->stream));
    const int ldo = cplx ? 2 * k : k;
    ST(gemm_basis(h, W, ldw, k, cplx, w.binv, ldo, k, n, w.tmpW, n, 1.0, 0.0));
    ST(copy_block(h, w.tmpW, n, W, ldw, n, k));
    if (!cplx) {
        ST(gemm_basis(h, PW, ldpw, k, false, w.binv, ldo, k, n, w.tmpPW, n, 1.0, 0.0));
        ST(copy_block(h, w.tmpPW, n, PW, ldpw, n, k));
    }
    // the pinned buffer is reused by later calls: make sure the upload has been consumed
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    return BSE_OK;
}

// one projection pass of columns [c0, c0+kc) of W against the basis A (coefficients in the active inner product)
static bse_status_t project_pass(bse_handle_s *h, const void *V, int64_t ldv, const void *PV, int64_t ldpv, int m,
                                 void *W, int64_t ldw, void *PW, int64_t ldpw, int kc, bool cplx, double *coef)
{
    if (m <= 0) return BSE_OK;
    const int64_t n = h->N;
    const int ldo = cplx ? 2 * m : m;
    ST(gram_basis(h, cplx ? V : PV, cplx ? ldv : ldpv, m, W, ldw, kc, cplx, n, coef));
    ST(gemm_basis(h, V, ldv, m, cplx, coef, ldo, kc, n, W, ldw, -1.0, 1.0));
    if (!cplx && PW) ST(gemm_basis(h, PV, ldpv, m, false, coef, ldo, kc, n, PW, ldpw, -1.0, 1.0));
    return BSE_OK;
}

// Euclidean squared column norms of a block (max over columns), used as the scale of rank decisions when the
// P-image of the block is not available yet.
static bse_status_t euclid_max_norm2(bse_handle_s *h, const void *W, int64_t ldw, int k, OrthWs &w, double *out)
{
    std::vector<zc> G;
    ST(block_gram(h, W, ldw, nullptr, 0, k, true, w, G));
    double m2 = 0.0;
    for (int j = 0; j < k; ++j) m2 = std::max(m2, G[j + (size_t)j * k].real());
    *out = m2;
    return BSE_OK;
}

// Block CGS, two passes against V (a5 + a6, twice).  PW may be NULL in the real inner product: then only W is
// updated and the caller recomputes P(W) afterwards (what bse_solve does: updating PW by linear combination lets
// PW drift away from P(W) exponentially over the iteration).
// Reserve the orthogonalisation workspace for a basis of up to m_max columns (avoids reallocation while it grows).
bse_status_t orth_reserve(bse_handle_s *h, int m_max, int k)
{
    OrthWs w;
    return orth_ws(h, m_max, k, w);
}

bse_status_t project_block(bse_handle_s *h, const void *V, int64_t ldv, int m, const void *PV, int64_t ldpv, void *W,
                           int64_t ldw, int k, void *PW, int64_t ldpw, bool cplx, void *hcoef_host)
{
    if (m <= 0) return BSE_OK;
    OrthWs w;
    ST(orth_ws(h, m, k, w));
    std::vector<zc> Hc((size_t)m * k, zc(0.0));
    ST(project_pass(h, V, ldv, PV, ldpv, m, W, ldw, PW, ldpw, k, cplx, w.c1));
    ST(project_pass(h, V, ldv, PV, ldpv, m, W, ldw, PW, ldpw, k, cplx, w.c2));
    size_t bytes = (size_t)(cplx ? 2 * m : m) * k * 8;
    BSE_CUDA(cudaMemcpyAsync(w.hc1, w.c1, bytes, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaMemcpyAsync(w.hc2, w.c2, bytes, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    coef_to_host(w.hc1, m, k, cplx, Hc.data(), false);      // h = h1 + h2
    coef_to_host(w.hc2, m, k, cplx, Hc.data(), true);
    if (hcoef_host) std::memcpy(hcoef_host, Hc.data(), sizeof(zc) * (size_t)m * k);
    return BSE_OK;
}

bse_status_t block_norm_scale(bse_handle_s *h, const void *W, int64_t ldw, const void *PW, int64_t ldpw, int k,
                              bool cplx, double *scale2)
{
    OrthWs w;
    ST(orth_ws(h, 0, k, w));
    if (!cplx && !PW) return euclid_max_norm2(h, W, ldw, k, w, scale2);
    std::vector<zc> G;
    ST(block_gram(h, W, ldw, PW, ldpw, k, cplx, w, G));
    double s2 = 0.0, gmax = 0.0;
    for (int j = 0; j < k; ++j) s2 = std::max(s2, G[j + (size_t)j * k].real());
    for (auto &v : G) gmax = std::max(gmax, std::abs(v));
    if (!cplx)
        for (int j = 0; j < k; ++j)
            if (G[j + (size_t)j * k].real() < -1e-10 * gmax) return BSE_ERR_NOT_POSITIVE_DEFINITE;
    *scale2 = s2;
    return BSE_OK;
}

// Intra-block orthonormalisation (a7) of a block already projected against V.  scale2: squared norm scale of the
// block BEFORE projection in the active inner product (rank decisions are relative to it); hcoef_host (m x k, may
// be NULL) receives the corrections of the column-wise path.
bse_status_t normalize_block(bse_handle_s *h, const void *V, int64_t ldv, int m, const void *PV, int64_t ldpv, void *W,
                             int64_t ldw, int k, void *PW, int64_t ldpw, bool cplx, double scale2, void *hcoef_host,
                             void *bfac_host, int *rank_out, uint64_t seed, uint64_t *rng_counter, int image_sign)
{
    const int64_t n = h->N;
    OrthWs w;
    ST(orth_ws(h, m, k, w));
    std::vector<zc> G, Hc((size_t)(m > 0 ? m : 1) * k, zc(0.0)), B((size_t)k * k, zc(0.0));
    if (hcoef_host && m > 0) std::memcpy(Hc.data(), hcoef_host, sizeof(zc) * (size_t)m * k);
    char *Wc = (char *)W, *PWc = (char *)PW;
    double gmax = scale2;

    // ---- intra-block orthonormalisation (a7): CholQR2 on the column-scaled Gram matrix; column-wise fallback
    bool slow = false;
    std::vector<zc> Btot((size_t)k * k, zc(0.0));
    for (int j = 0; j < k; ++j) Btot[j + (size_t)j * k] = 1.0;
    for (int rep = 0; rep < 2 && !slow; ++rep) {
        ST(block_gram(h, W, ldw, PW, ldpw, k, cplx, w, G));       // synchronises: hc1/hc2 are valid after this
        std::vector<double> dsc(k);
        for (int j = 0; j < k; ++j) {
            double gj = G[j + (size_t)j * k].real();
            if (!(gj > 1e-26 * scale2) || !(gj > 0.0)) { slow = true; break; }
            dsc[j] = std::sqrt(gj);
        }
        if (slow) break;
        // Cholesky of the unit-diagonal scaled matrix  G' = D^-1 G D^-1 = U^H U
        std::vector<zc> U((size_t)k * k, zc(0.0));
        for (int j = 0; j < k && !slow; ++j) {
            for (int i = 0; i <= j; ++i) {
                zc s = G[i + (size_t)j * k] / (dsc[i] * dsc[j]);
                for (int p = 0; p < i; ++p) s -= std::conj(U[p + (size_t)i * k]) * U[p + (size_t)j * k];
                if (i < j) U[i + (size_t)j * k] = s / U[i + (size_t)i * k].real();
                else {
                    if (!(s.real() > 1e-6)) { slow = true; break; }   // sine of the angle to the previous columns < 1e-3
                    U[j + (size_t)j * k] = std::sqrt(s.real());
                }
            }
        }
        if (slow) break;
        // B_rep = U D (upper);  W <- W B_rep^-1
        std::vector<zc> Br((size_t)k * k, zc(0.0)), Binv((size_t)k * k, zc(0.0));
        for (int j = 0; j < k; ++j)
            for (int i = 0; i <= j; ++i) Br[i + (size_t)j * k] = U[i + (size_t)j * k] * dsc[j];
        for (int j = 0; j < k; ++j) {          // upper triangular inverse by back substitution, column j
            Binv[j + (size_t)j * k] = 1.0 / Br[j + (size_t)j * k];
            for (int i = j - 1; i >= 0; --i) {
                zc s(0.0);
                for (int p = i + 1; p <= j; ++p) s += Br[i + (size_t)p * k] * Binv[p + (size_t)j * k];
                Binv[i + (size_t)j * k] = -s / Br[i + (size_t)i * k];
            }
        }
        ST(block_times_small(h, W, ldw, PW, ldpw, k, cplx, Binv.data(), w));
        std::vector<zc> T((size_t)k * k, zc(0.0));           // Btot = Br * Btot
        for (int j = 0; j < k; ++j)
            for (int i = 0; i < k; ++i) {
                zc s(0.0);
                for (int p = 0; p < k; ++p) s += Br[i + (size_t)p * k] * Btot[p + (size_t)j * k];
                T[i + (size_t)j * k] = s;
            }
        Btot.swap(T);
    }
    int rank = k;
    if (!slow) {
        B = Btot;
    } else {
        // column-by-column classical Gram-Schmidt (twice) inside the block; deficient columns are replaced by
        // orthonormalised pseudo-random vectors (reading S12).  W so far = (partially processed) * Btot^-1, so the
        // factor found here is multiplied by Btot at the end.
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        std::vector<zc> Bs((size_t)k * k, zc(0.0));
        rank = 0;
        const double thr2 = 1e-26 * scale2;
        for (int j = 0; j < k; ++j) {
            char *wj = Wc + (size_t)j * ldw * 16, *pwj = cplx ? nullptr : PWc + (size_t)j * ldpw * 16;
            for (int pass = 0; pass < 2 && j > 0; ++pass) {
                if (pass == 1 && m > 0) {
                    // what is left of the column may be tiny compared with what was projected against V: restore
                    // its orthogonality to V at its own scale (the correction belongs to column j of h)
                    ST(project_pass(h, V, ldv, PV, ldpv, m, wj, ldw, pwj, ldpw, 1, cplx, w.c2));
                    ST(fetch_coef(h, w.c2, w.hc2, m, 1, cplx));
                    coef_to_host(w.hc2, m, 1, cplx, &Hc[(size_t)j * m], true);
                }
                ST(project_pass(h, W, ldw, PW, ldpw, j, wj, ldw, pwj, ldpw, 1, cplx, w.c1));
                ST(fetch_coef(h, w.c1, w.hc1, j, 1, cplx));
                coef_to_host(w.hc1, j, 1, cplx, &Bs[(size_t)j * k], true);   // column j, rows 0..j-1 (ld = j == rows)
            }
            std::vector<zc> g1;
            ST(block_gram(h, wj, ldw, pwj, ldpw, 1, cplx, w, g1));
            double nn = g1[0].real();
            if (!cplx && nn < -1e-10 * gmax) return BSE_ERR_NOT_POSITIVE_DEFINITE;
            if (!(nn > thr2) || !(nn > 0.0)) {
                // dependent column: replace by a random vector orthonormal to V and to the previous columns
                Bs[j + (size_t)j * k] = 0.0;
                for (int tries = 0; tries < 3; ++tries) {
                    ST(fill_random_block(h, wj, ldw, n, 1, seed, (*rng_counter)++));
                    if (!cplx) {
                        bse_status_t st = bse_apply_half(h, image_sign, wj, ldw, pwj, ldpw, 1);
                        if (st) return st;
                    }
                    for (int pass = 0; pass < 2; ++pass) {
                        ST(project_pass(h, V, ldv, PV, ldpv, m, wj, ldw, pwj, ldpw, 1, cplx, w.c2));
                        if (j > 0) ST(project_pass(h, W, ldw, PW, ldpw, j, wj, ldw, pwj, ldpw, 1, cplx, w.c2));
                    }
                    ST(block_gram(h, wj, ldw, pwj, ldpw, 1, cplx, w, g1));
                    nn = g1[0].real();
                    if (nn > 0.0) break;
                }
                if (!(nn > 0.0)) return cplx ? BSE_ERR_INTERNAL : BSE_ERR_NOT_POSITIVE_DEFINITE;
                ST(scale_block(h, wj, ldw, n, 1, 1.0 / std::sqrt(nn)));
                if (!cplx) ST(scale_block(h, pwj, ldpw, n, 1, 1.0 / std::sqrt(nn)));
            } else {
                ++rank;
                double nrm = std::sqrt(nn);
                Bs[j + (size_t)j * k] = nrm;
                ST(scale_block(h, wj, ldw, n, 1, 1.0 / nrm));
                if (!cplx) ST(scale_block(h, pwj, ldpw, n, 1, 1.0 / nrm));
            }
        }
        // Bs columns were stored with ld = j for rows < j: re-lay them out with ld = k
        std::vector<zc> Bfull((size_t)k * k, zc(0.0));
        for (int j = 0; j < k; ++j) {
            for (int i = 0; i < j; ++i) Bfull[i + (size_t)j * k] = Bs[(size_t)j * k + i];
            Bfull[j + (size_t)j * k] = Bs[j + (size_t)j * k];
        }
        for (int j = 0; j < k; ++j)
            for (int i = 0; i < k; ++i) {
                zc s(0.0);
                for (int p = 0; p < k; ++p) s += Bfull[i + (size_t)p * k] * Btot[p + (size_t)j * k];
                B[i + (size_t)j * k] = s;
            }
    }
    if (hcoef_host && m > 0) std::memcpy(hcoef_host, Hc.data(), sizeof(zc) * (size_t)m * k);
    if (bfac_host) std::memcpy(bfac_host, B.data(), sizeof(zc) * (size_t)k * k);
    if (rank_out) *rank_out = rank;
    return BSE_OK;
}

bse_status_t orth_block(bse_handle_s *h, const void *V, int64_t ldv, int m, const void *PV, int64_t ldpv, void *W,
                        int64_t ldw, int k, void *PW, int64_t ldpw, void *hcoef_host, void *bfac_host, int *rank_out,
                        uint64_t seed, uint64_t *rng_counter)
{
    const bool cplx = (PV == nullptr);
    double scale2 = 0.0;
    ST(block_norm_scale(h, W, ldw, PW, ldpw, k, cplx, &scale2));
    std::vector<zc> Hc((size_t)(m > 0 ? m : 1) * k, zc(0.0));
    ST(project_block(h, V, ldv, m, PV, ldpv, W, ldw, k, PW, ldpw, cplx, Hc.data()));
    ST(normalize_block(h, V, ldv, m, PV, ldpv, W, ldw, k, PW, ldpw, cplx, scale2, Hc.data(), bfac_host, rank_out, seed,
                       rng_counter));
    if (hcoef_host && m > 0) std::memcpy(hcoef_host, Hc.data(), sizeof(zc) * (size_t)m * k);
    return BSE_OK;
}

}  // namespace bse

using namespace bse;

extern "C" bse_status_t bse_orth(bse_handle_t h, const void *dV, int64_t ldv, int32_t m, const void *dBV, int64_t ldbv,
                                 void *dW, int64_t ldw, int32_t k, void *dBW, int64_t ldbw, void *dHcoef, void *dBfac,
                                 int32_t *hRank)
{
    if (!h || !dW || k < 1 || m < 0 || ldw < h->N || is_incomplete(h)) return BSE_ERR_INVALID_ARG;
    if (m > 0 && (!dV || ldv < h->N)) return BSE_ERR_INVALID_ARG;
    if (dBV || dBW) {
        if (h->mode != BSE_MODE_FULL || !dBW || ldbw < h->N || (m > 0 && (!dBV || ldbv < h->N))) return BSE_ERR_INVALID_ARG;
    }
    const bool real_ip = (dBW != nullptr);
    // in the real inner product with m == 0 there is no dBV: pass dBW's own pointer as a non-null marker
    const void *pv = real_ip ? (m > 0 ? dBV : dBW) : nullptr;
    std::vector<std::complex<double>> Hc((size_t)(m > 0 ? m : 1) * k), B((size_t)k * k);
    int rank = 0;
    uint64_t ctr = 1000;
    bse_status_t st = orth_block(h, dV, ldv, m, pv, ldbv, dW, ldw, k, dBW, ldbw, Hc.data(), B.data(), &rank, 12345, &ctr);
    if (st) return st;
    if (dHcoef && m > 0) BSE_CUDA(cudaMemcpyAsync(dHcoef, Hc.data(), sizeof(double) * 2 * (size_t)m * k, cudaMemcpyHostToDevice, h->stream));
    if (dBfac) BSE_CUDA(cudaMemcpyAsync(dBfac, B.data(), sizeof(double) * 2 * (size_t)k * k, cudaMemcpyHostToDevice, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    if (hRank) *hRank = rank;
    return BSE_OK;
}
