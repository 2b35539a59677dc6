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
[[maybe_unused]] static void host_to_coef(const zc *in, int m, int k, bool cplx, double *c)
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

enum { SC_E_IN = 0, SC_E_AFTER = 1, SC_G = 2, SC_SCALE2 = 3, SC_COUNT = 8 };      // device scalar slots
enum { F_SLOW = 0, F_NOT_PD = 1, F_COUNT = 8 };                                   // device flags (doubles: 0 / 1)

struct OrthWs {
    double *c1, *c2, *g, *binv;   // device coefficient buffers
    double *tmpW, *tmpPW;         // device n x k complex temporaries
    double *scal, *flags, *btot, *scratch;      // device: scalars, flags, accumulated k x k factor (complex), Cholesky scratch
    double *hc1, *hc2, *hg, *hbinv;   // pinned host mirrors
    double *hsmall;                   // pinned mirror of [scal | flags | btot]
};

// Layout: everything whose offset depends only on (n, k) first, the m-dependent coefficient buffers last, so that the
// scalar slots keep their place while the basis grows (orth_reserve sizes the buffer for the largest m up front).
static bse_status_t orth_ws(bse_handle_s *h, int m, int k, OrthWs &w)
{
    const int64_t n = vec_rows(h);
    size_t cm = (size_t)2 * (m > 0 ? m : 1) * k, ck = (size_t)2 * k * k;
    const size_t small = SC_COUNT + F_COUNT + ck;
    size_t doubles = (size_t)4 * n * k + small + 2 * ck + 4 * ck + 2 * cm;
    ST(ensure_ws2(h, doubles * 8));
    ST(ensure_pin(h, (2 * cm + 2 * ck + small) * 8));
    double *p = (double *)h->ws2;
    w.tmpW = p; p += (size_t)2 * n * k;         // keep the large blocks first (16-byte aligned)
    w.tmpPW = p; p += (size_t)2 * n * k;
    w.scal = p; p += SC_COUNT;
    w.flags = p; p += F_COUNT;
    w.btot = p; p += ck;
    w.g = p; p += ck;
    w.binv = p; p += ck;
    w.scratch = p; p += 4 * ck;
    w.c1 = p; p += cm;
    w.c2 = p;
    double *q = (double *)h->hpin;
    w.hsmall = q; q += small;
    w.hg = q; q += ck;
    w.hbinv = q; q += ck;
    w.hc1 = q; q += cm;
    w.hc2 = q;
    return BSE_OK;
}

// ---- k x k work on the device (one thread: k^3 complex operations), so that the block step needs ONE host synchronisation
// instead of one per factorisation.  g: Gram matrix in coefficient layout (real parts, then imaginary parts, per column).
__device__ __forceinline__ double2 g_at(const double *g, int k, int cplx, int i, int j)
{
    const int ldo = cplx ? 2 * k : k;
    return make_double2(g[i + (size_t)j * ldo], cplx ? g[i + k + (size_t)j * ldo] : 0.0);
}
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) { return make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }   // conj(a) b
__device__ __forceinline__ double2 cdiv(double2 a, double2 b)
{
    const double d = b.x * b.x + b.y * b.y;
    return make_double2((a.x * b.x + a.y * b.y) / d, (a.y * b.x - a.x * b.y) / d);
}

// scal[slot] = max_j G_jj;  real inner product with check_pd: a diagonal entry below -1e-10 max|G| flags "not positive definite"
__global__ void diag_stats_kernel(const double *g, int k, int cplx, double *scal, int slot, double *flags, int check_pd)
{
    if (threadIdx.x || blockIdx.x) return;
    double s2 = 0.0, gmax = 0.0;
    for (int j = 0; j < k; ++j) {
        s2 = fmax(s2, g_at(g, k, cplx, j, j).x);
        for (int i = 0; i < k; ++i) { const double2 v = g_at(g, k, cplx, i, j); gmax = fmax(gmax, sqrt(v.x * v.x + v.y * v.y)); }
    }
    if (check_pd)
        for (int j = 0; j < k; ++j)
            if (g_at(g, k, cplx, j, j).x < -1e-10 * gmax) flags[F_NOT_PD] = 1.0;
    scal[slot] = s2;
}

// One CholQR round on the device: G = (U D)^H (U D) with the unit-diagonal scaled Cholesky factor U; writes Binv = (U D)^-1 in
// coefficient layout and Btot <- (U D) Btot.  Same decisions as the host code it replaces: a diagonal entry not above
// 1e-26 scale2, or a pivot (squared sine of the angle to the previous columns) not above 1e-6, sets F_SLOW and leaves
// Binv = I -- the host then takes the column-by-column path.  scale2: the squared norm scale of the incoming block
// (scale_mode 0: scal[SC_E_IN];  1: scal[SC_G] * scal[SC_E_IN] / scal[SC_E_AFTER], the P-norm estimated through Euclidean norms).
__global__ void cholqr_kernel(const double *g, int k, int cplx, double *scal, int scale_mode, int first, double *binv,
                              double2 *btot, double *flags, double2 *scratch, int use_smem)
{
    // small k: Gram matrix and scratch in shared memory (a single thread walking global memory pays its latency on every
    // dependent access: 100+ us per call at k = 4); large k: the global scratch
    extern __shared__ double2 chol_sm[];
    const int ldo = cplx ? 2 * k : k;
    if (use_smem) {
        double *gs = reinterpret_cast<double *>(chol_sm + 4 * (size_t)k * k);
        for (int i = threadIdx.x; i < ldo * k; i += blockDim.x) gs[i] = g[i];
        __syncthreads();
        g = gs;
        scratch = chol_sm;
    }
    if (threadIdx.x || blockIdx.x) return;
    double2 *U = scratch, *Br = scratch + (size_t)k * k, *Bi = scratch + 2 * (size_t)k * k, *T = scratch + 3 * (size_t)k * k;
    double scale2;
    if (scale_mode == 0) scale2 = scal[SC_E_IN];
    else scale2 = (scal[SC_E_AFTER] > 0.0) ? scal[SC_G] * (scal[SC_E_IN] / scal[SC_E_AFTER]) : scal[SC_G];
    if (first) {
        scal[SC_SCALE2] = scale2;
        for (int i = 0; i < k * k; ++i) btot[i] = make_double2(0.0, 0.0);
        for (int j = 0; j < k; ++j) btot[j + (size_t)j * k] = make_double2(1.0, 0.0);
    }
    bool slow = flags[F_SLOW] != 0.0;
    for (int j = 0; j < k && !slow; ++j) {
        const double gj = g_at(g, k, cplx, j, j).x;
        if (!(gj > 1e-26 * scale2) || !(gj > 0.0)) slow = true;
    }
    for (int i = 0; i < k * k; ++i) U[i] = Br[i] = Bi[i] = make_double2(0.0, 0.0);
    for (int j = 0; j < k && !slow; ++j)
        for (int i = 0; i <= j; ++i) {
            const double di = sqrt(g_at(g, k, cplx, i, i).x), dj = sqrt(g_at(g, k, cplx, j, j).x);
            double2 sv = g_at(g, k, cplx, i, j);
            sv.x /= di * dj; sv.y /= di * dj;
            for (int p = 0; p < i; ++p) { const double2 t = cmulc(U[p + (size_t)i * k], U[p + (size_t)j * k]); sv.x -= t.x; sv.y -= t.y; }
            if (i < j) { const double d = U[i + (size_t)i * k].x; U[i + (size_t)j * k] = make_double2(sv.x / d, sv.y / d); }
            else {
                if (!(sv.x > 1e-6)) { slow = true; break; }
                U[j + (size_t)j * k] = make_double2(sqrt(sv.x), 0.0);
            }
        }
    if (slow) {                                            // identity: W is left as it is, the host continues column by column
        flags[F_SLOW] = 1.0;
        for (int j = 0; j < k; ++j)
            for (int i = 0; i < k; ++i) {
                binv[i + (size_t)j * ldo] = (i == j) ? 1.0 : 0.0;
                if (cplx) binv[i + k + (size_t)j * ldo] = 0.0;
            }
        return;
    }
    for (int j = 0; j < k; ++j) {
        const double dj = sqrt(g_at(g, k, cplx, j, j).x);
        for (int i = 0; i <= j; ++i) Br[i + (size_t)j * k] = make_double2(U[i + (size_t)j * k].x * dj, U[i + (size_t)j * k].y * dj);
    }
    for (int j = 0; j < k; ++j) {                          // upper triangular inverse by back substitution, column j
        Bi[j + (size_t)j * k] = cdiv(make_double2(1.0, 0.0), Br[j + (size_t)j * k]);
        for (int i = j - 1; i >= 0; --i) {
            double2 sv = make_double2(0.0, 0.0);
            for (int p = i + 1; p <= j; ++p) { const double2 t = cmul(Br[i + (size_t)p * k], Bi[p + (size_t)j * k]); sv.x += t.x; sv.y += t.y; }
            Bi[i + (size_t)j * k] = cdiv(make_double2(-sv.x, -sv.y), Br[i + (size_t)i * k]);
        }
    }
    for (int j = 0; j < k; ++j)
        for (int i = 0; i < k; ++i) {
            binv[i + (size_t)j * ldo] = Bi[i + (size_t)j * k].x;
            if (cplx) binv[i + k + (size_t)j * ldo] = Bi[i + (size_t)j * k].y;
            double2 sv = make_double2(0.0, 0.0);           // T = Br * Btot
            for (int p = 0; p < k; ++p) { const double2 t = cmul(Br[i + (size_t)p * k], btot[p + (size_t)j * k]); sv.x += t.x; sv.y += t.y; }
            T[i + (size_t)j * k] = sv;
        }
    for (int i = 0; i < k * k; ++i) btot[i] = T[i];
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
    ST(gram_basis(h, W, ldw, k, cplx ? W : PW, cplx ? ldw : ldpw, k, cplx, vec_rows(h), w.g));
    ST(fetch_coef(h, w.g, w.hg, k, k, cplx));
    G.assign((size_t)k * k, zc(0.0));
    coef_to_host(w.hg, k, k, cplx, G.data(), false);
    return BSE_OK;
}

// one projection pass of columns [c0, c0+kc) of W against the basis A (coefficients in the active inner product)
static bse_status_t project_pass(bse_handle_s *h, const void *V, int64_t ldv, const void *PV, int64_t ldpv, int m,
                                 void *W, int64_t ldw, void *PW, int64_t ldpw, int kc, bool cplx, double *coef)
{
    if (m <= 0) return BSE_OK;
    const int64_t n = vec_rows(h);
    const int ldo = cplx ? 2 * m : m;
    ST(gram_basis(h, cplx ? V : PV, cplx ? ldv : ldpv, m, W, ldw, kc, cplx, n, coef));
    ST(gemm_basis(h, V, ldv, m, cplx, coef, ldo, kc, n, W, ldw, -1.0, 1.0));
    if (!cplx && PW) ST(gemm_basis(h, PV, ldpv, m, false, coef, ldo, kc, n, PW, ldpw, -1.0, 1.0));
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

// Asynchronous: the coefficients h1, h2 of the two passes stay on the device until normalize_block fetches them.
bse_status_t project_block(bse_handle_s *h, const void *V, int64_t ldv, int m, const void *PV, int64_t ldpv, void *W,
                           int64_t ldw, int k, void *PW, int64_t ldpw, bool cplx)
{
    if (m <= 0) return BSE_OK;
    OrthWs w;
    ST(orth_ws(h, m, k, w));
    ST(project_pass(h, V, ldv, PV, ldpv, m, W, ldw, PW, ldpw, k, cplx, w.c1));
    ST(project_pass(h, V, ldv, PV, ldpv, m, W, ldw, PW, ldpw, k, cplx, w.c2));
    return BSE_OK;
}

// Asynchronous: scal[slot] = max_j <w_j, w_j> in the active inner product (Euclidean when PW is NULL).  slot == SC_E_IN
// opens a block step: the flags are cleared.
bse_status_t block_norm_scale(bse_handle_s *h, const void *W, int64_t ldw, const void *PW, int64_t ldpw, int k,
                              bool cplx, int slot)
{
    OrthWs w;
    ST(orth_ws(h, 0, k, w));
    if (slot == SC_E_IN) BSE_CUDA(cudaMemsetAsync(w.flags, 0, sizeof(double) * F_COUNT, h->stream));
    const bool euclid = cplx || !PW;
    ST(gram_basis(h, W, ldw, k, euclid ? W : PW, euclid ? ldw : ldpw, k, euclid, vec_rows(h), w.g));
    diag_stats_kernel<<<1, 32, 0, h->stream>>>(w.g, k, euclid ? 1 : 0, w.scal, slot, w.flags, euclid ? 0 : 1);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

// Intra-block orthonormalisation (a7) of a block already projected against V, and the ONE host synchronisation of the block
// step.  scale_mode: how the squared norm scale of the block BEFORE projection is formed from the device scalars (see
// cholqr_kernel; rank decisions are relative to it).  hcoef_host (m x k, may be NULL) receives h1 + h2 of project_block plus
// the corrections of the column-wise path; bfac_host the k x k factor.
bse_status_t normalize_block(bse_handle_s *h, const void *V, int64_t ldv, int m, const void *PV, int64_t ldpv, void *W,
                             int64_t ldw, int k, void *PW, int64_t ldpw, bool cplx, int scale_mode, void *hcoef_host,
                             void *bfac_host, int *rank_out, uint64_t seed, uint64_t *rng_counter, int image_sign)
{
    const int64_t n = vec_rows(h);
    OrthWs w;
    ST(orth_ws(h, m, k, w));
    std::vector<zc> G, Hc((size_t)(m > 0 ? m : 1) * k, zc(0.0)), B((size_t)k * k, zc(0.0));
    char *Wc = (char *)W, *PWc = (char *)PW;
    const int ldo = cplx ? 2 * k : k;

    // ---- intra-block orthonormalisation (a7): CholQR2 on the column-scaled Gram matrix, factorised on the device
    for (int rep = 0; rep < 2; ++rep) {
        ST(gram_basis(h, W, ldw, k, cplx ? W : PW, cplx ? ldw : ldpw, k, cplx, n, w.g));
        const size_t chol_smem = (size_t)4 * k * k * 16 + (size_t)ldo * k * 8;
        const int use_smem = chol_smem <= 48 * 1024 ? 1 : 0;
        cholqr_kernel<<<1, 32, use_smem ? chol_smem : 0, h->stream>>>(w.g, k, cplx ? 1 : 0, w.scal, scale_mode, rep == 0 ? 1 : 0,
                                                                      w.binv, (double2 *)w.btot, w.flags, (double2 *)w.scratch,
                                                                      use_smem);
        count_launch();
        ST(gemm_basis(h, W, ldw, k, cplx, w.binv, ldo, k, n, w.tmpW, n, 1.0, 0.0));       // W <- W Binv
        ST(copy_block(h, w.tmpW, n, W, ldw, n, k));
        if (!cplx) {
            ST(gemm_basis(h, PW, ldpw, k, false, w.binv, ldo, k, n, w.tmpPW, n, 1.0, 0.0));
            ST(copy_block(h, w.tmpPW, n, PW, ldpw, n, k));
        }
    }
    BSE_CUDA(cudaGetLastError());
    // ---- the block step's one synchronisation: scalars, flags, accumulated factor, projection coefficients
    const size_t small = SC_COUNT + F_COUNT + (size_t)2 * k * k;
    BSE_CUDA(cudaMemcpyAsync(w.hsmall, w.scal, small * 8, cudaMemcpyDeviceToHost, h->stream));
    if (m > 0) {
        const size_t bytes = (size_t)(cplx ? 2 * m : m) * k * 8;
        BSE_CUDA(cudaMemcpyAsync(w.hc1, w.c1, bytes, cudaMemcpyDeviceToHost, h->stream));
        BSE_CUDA(cudaMemcpyAsync(w.hc2, w.c2, bytes, cudaMemcpyDeviceToHost, h->stream));
    }
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    if (m > 0) {
        coef_to_host(w.hc1, m, k, cplx, Hc.data(), false);      // h = h1 + h2
        coef_to_host(w.hc2, m, k, cplx, Hc.data(), true);
    }
    const double *hscal = w.hsmall, *hflags = w.hsmall + SC_COUNT, *hbtot = w.hsmall + SC_COUNT + F_COUNT;
    if (hflags[F_NOT_PD] != 0.0) return BSE_ERR_NOT_POSITIVE_DEFINITE;
    const double scale2 = hscal[SC_SCALE2];
    const double gmax = scale2;
    bool slow = hflags[F_SLOW] != 0.0;
    std::vector<zc> Btot((size_t)k * k, zc(0.0));
    for (int i = 0; i < k * k; ++i) Btot[i] = zc(hbtot[2 * i], hbtot[2 * i + 1]);
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
                        bse_status_t st = apply_vec(h, image_sign, wj, ldw, pwj, ldpw, 1);
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
    OrthWs w;
    ST(orth_ws(h, m, k, w));                                  // sized for this m before the first kernel writes into it
    ST(block_norm_scale(h, W, ldw, PW, ldpw, k, cplx, SC_E_IN));
    ST(project_block(h, V, ldv, m, PV, ldpv, W, ldw, k, PW, ldpw, cplx));
    std::vector<zc> Hc((size_t)(m > 0 ? m : 1) * k, zc(0.0));
    ST(normalize_block(h, V, ldv, m, PV, ldpv, W, ldw, k, PW, ldpw, cplx, 0, Hc.data(), bfac_host, rank_out, seed,
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
    if (!h || !dW || k < 1 || m < 0 || ldw < vec_rows(h) || is_incomplete(h)) return BSE_ERR_INVALID_ARG;
    if (m > 0 && (!dV || ldv < vec_rows(h))) return BSE_ERR_INVALID_ARG;
    if (dBV || dBW) {
        if (h->mode != BSE_MODE_FULL || !dBW || ldbw < vec_rows(h) || (m > 0 && (!dBV || ldbv < vec_rows(h)))) return BSE_ERR_INVALID_ARG;
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
