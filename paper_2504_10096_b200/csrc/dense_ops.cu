// Launch wrappers for the dense basis kernels and a few elementwise kernels.
#include <algorithm>

#include "bse_internal.h"
#include "dense_kernels.cuh"
#include "gemm_kernel.cuh"
#include "rng.cuh"

namespace bse {

bse_status_t gram_basis(bse_handle_s *h, const void *A, int64_t lda, int m, const void *B, int64_t ldb, int k,
                        bool cplx, int64_t n, double *out)
{
    if (m <= 0 || k <= 0) return BSE_OK;
    const int64_t nr = 2 * n;
    const int ldo = cplx ? 2 * m : m;
    BSE_CUDA(cudaMemsetAsync(out, 0, sizeof(double) * (size_t)ldo * k, h->stream));
    static std::atomic<uint64_t> attr_devices{0};         // per device (cudaFuncSetAttribute is)
    int dev = 0;
    BSE_CUDA(cudaGetDevice(&dev));
    if (dev >= 64 || !(attr_devices.load(std::memory_order_acquire) & (1ull << dev))) {
        BSE_CUDA(cudaFuncSetAttribute(gram_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, GRAM_SMEM));
        BSE_CUDA(cudaFuncSetAttribute(gram_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, GRAM_SMEM));
        if (dev < 64) attr_devices.fetch_or(1ull << dev, std::memory_order_release);
    }
    // one CTA per SM (the rings take the shared memory): 64-column groups x row chunks ~ BSE_GRAM_CTAS x the SM count
    const int gx = (m + 8 * GRAM_WARPS - 1) / (8 * GRAM_WARPS);
    static const int ctas_per_sm = [] {                  // BSE_GRAM_CTAS: read once per process
        int v = 1;
        if (const char *e = getenv("BSE_GRAM_CTAS")) { int u = atoi(e); if (u >= 1 && u <= 16) v = u; }
        return v;
    }();
    const int64_t want = std::max<int64_t>(1, (int64_t)ctas_per_sm * h->num_sms / gx);
    int64_t rows = (nr + want - 1) / want;
    rows = ((rows + 31) / 32) * 32;
    const int gy = (int)((nr + rows - 1) / rows);
    // up to 8 complex / 16 real columns per launch (two N-tiles); one N-tile when it is enough
    const int step = cplx ? 8 : 16;
    for (int c0 = 0; c0 < k; c0 += step) {
        int kc = (k - c0) < step ? (k - c0) : step;
        const int ncols = cplx ? 2 * kc : kc;
        const double *Bp = (const double *)B + 2 * (int64_t)c0 * ldb;
        double *op = out + (int64_t)c0 * ldo;
        if (ncols <= 8)
            gram_kernel<1><<<dim3(gx, gy), 32 * GRAM_WARPS, GRAM_SMEM, h->stream>>>((const double *)A, 2 * lda, m, Bp, 2 * ldb, kc, ncols,
                                                               nr, rows, op, ldo, cplx ? m : 0);
        else
            gram_kernel<2><<<dim3(gx, gy), 32 * GRAM_WARPS, GRAM_SMEM, h->stream>>>((const double *)A, 2 * lda, m, Bp, 2 * ldb, kc, ncols,
                                                               nr, rows, op, ldo, cplx ? m : 0);
        count_launch();
    }
    BSE_CUDA(cudaGetLastError());
    // row-partitioned vectors: every rank holds part of the rows, the Gram matrix is the sum over the ranks.  Replicated
    // vectors: the partial sums were combined with floating-point atomics, so on a sharded operator rank 0's result is everyone's
    if (is_row_partitioned(h)) return comm_sum_dev(h, out, (int64_t)ldo * k);
    return comm_bcast_dev(h, out, (int64_t)ldo * k);
}

template <int MT, int NT, int WM, int WN>
static bse_status_t launch_gemm(bse_handle_s *h, const double *A, int64_t lda2, int64_t nr, int m, int cplx,
                                const double *Bm, int64_t ldb, int l, double *C, int64_t ldc2, double alpha,
                                double beta)
{
    using Cfg = GemmCfg<MT, NT, WM, WN>;
    static std::atomic<uint64_t> attr_devices{0};         // per device (cudaFuncSetAttribute is)
    int dev = 0;
    BSE_CUDA(cudaGetDevice(&dev));
    if (dev >= 64 || !(attr_devices.load(std::memory_order_acquire) & (1ull << dev))) {
        BSE_CUDA(cudaFuncSetAttribute(gemm_nn_kernel<MT, NT, WM, WN>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      Cfg::SMEM));
        if (dev < 64) attr_devices.fetch_or(1ull << dev, std::memory_order_release);
    }
    dim3 grid((unsigned)((nr + Cfg::BM - 1) / Cfg::BM), (unsigned)((l + Cfg::BN - 1) / Cfg::BN));
    gemm_nn_kernel<MT, NT, WM, WN><<<grid, Cfg::THREADS, Cfg::SMEM, h->stream>>>(A, lda2, nr, m, cplx, Bm, ldb, l, C,
                                                                                  ldc2, alpha, beta);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

bse_status_t gemm_basis(bse_handle_s *h, const void *A, int64_t lda, int m, bool cplx_, const double *coef, int64_t ldo,
                        int l, int64_t n, void *C, int64_t ldc, double alpha, double beta, bool a_upper, bool c_lower)
{
    if (l <= 0) return BSE_OK;
    const int cplx = (cplx_ ? 1 : 0) | (a_upper ? 2 : 0) | (c_lower ? 4 : 0);          // kernel flags
    if (l <= 8)
        return launch_gemm<4, 1, 8, 1>(h, (const double *)A, 2 * lda, 2 * n, m, cplx, coef, ldo, l, (double *)C,
                                       2 * ldc, alpha, beta);
    if (l <= 32)
        return launch_gemm<2, 2, 4, 2>(h, (const double *)A, 2 * lda, 2 * n, m, cplx, coef, ldo, l, (double *)C,
                                       2 * ldc, alpha, beta);
    return launch_gemm<4, 4, 4, 2>(h, (const double *)A, 2 * lda, 2 * n, m, cplx, coef, ldo, l, (double *)C, 2 * ldc,
                                   alpha, beta);
}

__global__ void fill_random_kernel(double2 *W, int64_t ldw, int64_t n, int64_t row0, int k, uint64_t h0, uint64_t counter)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (i < n && c < k) W[i + c * ldw] = normal_pair(h0, (uint64_t)(row0 + i), counter + (uint64_t)c);
}
// n rows starting at this handle's first vector row (the entries are a function of the GLOBAL row index, so a row-partitioned
// block is the slice of the replicated one)
bse_status_t fill_random_block(bse_handle_s *h, void *W, int64_t ldw, int64_t n, int k, uint64_t seed, uint64_t counter)
{
    fill_random_kernel<<<dim3((unsigned)((n + 255) / 256), k), 256, 0, h->stream>>>((double2 *)W, ldw, n, h->vr_begin, k,
                                                                                    stream_key(seed, 6), counter);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

bse_status_t copy_block(bse_handle_s *h, const void *src, int64_t lds, void *dst, int64_t ldd, int64_t n, int k)
{
    BSE_CUDA(cudaMemcpy2DAsync(dst, (size_t)ldd * 16, src, (size_t)lds * 16, (size_t)n * 16, (size_t)k,
                               cudaMemcpyDeviceToDevice, h->stream));
    return BSE_OK;
}

__global__ void coef_to_complex_kernel(const double *c1, const double *c2, int m, int k, int cplx, double2 *dst)
{
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= m * k) return;
    int a = idx % m, col = idx / m;
    int ldo = cplx ? 2 * m : m;
    double re = c1[a + (int64_t)col * ldo] + (c2 ? c2[a + (int64_t)col * ldo] : 0.0);
    double im = 0.0;
    if (cplx) im = c1[a + m + (int64_t)col * ldo] + (c2 ? c2[a + m + (int64_t)col * ldo] : 0.0);
    dst[idx] = make_double2(re, im);
}
bse_status_t coef_to_complex(bse_handle_s *h, const double *c1, const double *c2, int m, int k, bool cplx, void *dst)
{
    if (m * k == 0) return BSE_OK;
    coef_to_complex_kernel<<<(m * k + 255) / 256, 256, 0, h->stream>>>(c1, c2, m, k, cplx ? 1 : 0, (double2 *)dst);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

__global__ void assemble_full_kernel(const double2 *x, const double2 *px, int64_t N, int nev, const double *omega,
                                     double2 *vec, int64_t ldvec)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (i >= N || c >= nev) return;
    double w = omega[c], sc = 0.5 * sqrt(w);
    double2 a = x[i + c * N], b = px[i + c * N];
    b.x /= w; b.y /= w;
    vec[i + c * ldvec] = make_double2(sc * (a.x + b.x), sc * (a.y + b.y));
    vec[i + N + c * ldvec] = make_double2(sc * (a.x - b.x), -sc * (a.y - b.y));
}
bse_status_t assemble_full_vectors(bse_handle_s *h, const void *x, const void *px, int64_t N, int nev,
                                   const double *d_omega, void *vec, int64_t ldvec)
{
    assemble_full_kernel<<<dim3((unsigned)((N + 255) / 256), nev), 256, 0, h->stream>>>(
        (const double2 *)x, (const double2 *)px, N, nev, d_omega, (double2 *)vec, ldvec);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

}  // namespace bse

namespace bse {
// out = [conj(v2); conj(v1)] (which = 0), [v1; -v2] (which = 1), [conj(v2); -conj(v1)] (which = 2) for v = [v1; v2]
__global__ void partner_kernel(const double2 *v, int64_t ldv, int64_t N, int nev, int which, double2 *out, int64_t ldo)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (i >= N || c >= nev) return;
    const double2 a = v[i + c * ldv], b = v[i + N + c * ldv];
    double2 o1, o2;
    if (which == 0) { o1 = make_double2(b.x, -b.y); o2 = make_double2(a.x, -a.y); }
    else if (which == 1) { o1 = a; o2 = make_double2(-b.x, -b.y); }
    else { o1 = make_double2(b.x, -b.y); o2 = make_double2(-a.x, a.y); }
    out[i + c * ldo] = o1;
    out[i + N + c * ldo] = o2;
}
}  // namespace bse

extern "C" bse_status_t bse_partner_vectors(bse_handle_t h, const void *dVec, int64_t ldvec, int32_t nev, int32_t which,
                                            void *dOut, int64_t ldout)
{
    if (!h || h->mode != BSE_MODE_FULL || !dVec || !dOut || dVec == dOut || nev < 1 || which < 0 || which > 2 ||
        ldvec < 2 * h->N || ldout < 2 * h->N)
        return BSE_ERR_INVALID_ARG;
    bse::partner_kernel<<<dim3((unsigned)((h->N + 255) / 256), nev), 256, 0, h->stream>>>(
        (const double2 *)dVec, ldvec, h->N, nev, which, (double2 *)dOut, ldout);
    bse::count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

namespace bse {
// S (m x l complex, ld m) -> coefficient layout of gemm_basis (real parts, then imaginary parts, per column)
__global__ void complex_to_coef_kernel(const double2 *S, int m, int l, int cplx, double *coef)
{
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= m * l) return;
    int a = idx % m, col = idx / m;
    int ldo = cplx ? 2 * m : m;
    double2 v = S[idx];
    coef[a + (int64_t)col * ldo] = v.x;
    if (cplx) coef[a + m + (int64_t)col * ldo] = v.y;
}

}  // namespace bse

using namespace bse;

extern "C" bse_status_t bse_gram(bse_handle_t h, const void *dA, int64_t lda, int32_t m, const void *dB, int64_t ldb, int32_t k,
                                 int32_t real_ip, void *dG)
{
    if (!h || !dA || !dB || !dG || m < 1 || k < 1 || lda < h->N || ldb < h->N) return BSE_ERR_INVALID_ARG;
    const bool cplx = !real_ip;
    bse_status_t st = ensure_ws(h, (size_t)2 * m * k * 8);
    if (st) return st;
    if ((st = gram_basis(h, dA, lda, m, dB, ldb, k, cplx, h->N, (double *)h->ws))) return st;
    return coef_to_complex(h, (const double *)h->ws, nullptr, m, k, cplx, dG);
}

extern "C" bse_status_t bse_update(bse_handle_t h, const void *dA, int64_t lda, int32_t m, const void *dS, int32_t l,
                                   int32_t real_ip, void *dC, int64_t ldc, double alpha, double beta)
{
    if (!h || !dA || !dS || !dC || m < 1 || l < 1 || lda < h->N || ldc < h->N || dA == dC) return BSE_ERR_INVALID_ARG;
    const bool cplx = !real_ip;
    bse_status_t st = ensure_ws(h, (size_t)2 * m * l * 8);
    if (st) return st;
    complex_to_coef_kernel<<<(m * l + 255) / 256, 256, 0, h->stream>>>((const double2 *)dS, m, l, cplx ? 1 : 0, (double *)h->ws);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return gemm_basis(h, dA, lda, m, cplx, (const double *)h->ws, cplx ? 2 * m : m, l, h->N, dC, ldc, alpha, beta);
}
