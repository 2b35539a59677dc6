// Lanczos with quadrature rules (the optical absorption spectrum "directly, without
// explicitly computing the eigenpairs").  TDA operator, three-term recurrence, no stored basis: per step one
// bse_apply with k = 1 (the HBM-bound case of the tile kernel) and three O(N) kernels.  All scalars stay on the
// device; the host synchronises once at the end.
#include <cmath>
#include <vector>

#include "bse_common.cuh"
#include "bse_internal.h"

namespace bse {

// acc[0] += Re(v^H w)
__global__ void __launch_bounds__(256) dot_re_kernel(const double2 *__restrict__ v, const double2 *__restrict__ w,
                                                     int64_t n, double *acc)
{
    double s = 0.0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        double2 a = v[i], b = w[i];
        s += a.x * b.x + a.y * b.y;
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(acc, s);
}
// w -= alpha v + beta_j vprev ;  nrm2[0] += |w|^2        (alpha = *alpha_p, beta_j = sqrt(*beta2_p) or 0 when null)
__global__ void __launch_bounds__(256) axpy_norm_kernel(double2 *__restrict__ w, const double2 *__restrict__ v,
                                                        const double2 *__restrict__ vprev, int64_t n,
                                                        const double *alpha_p, const double *beta2_p, double *nrm2)
{
    const double alpha = *alpha_p, beta = beta2_p ? sqrt(*beta2_p) : 0.0;
    double s = 0.0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        double2 x = w[i], a = v[i];
        x.x -= alpha * a.x; x.y -= alpha * a.y;
        if (beta2_p) { double2 p = vprev[i]; x.x -= beta * p.x; x.y -= beta * p.y; }
        w[i] = x;
        s += x.x * x.x + x.y * x.y;
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(nrm2, s);
}
// out = in / sqrt(*nrm2)   (out = 0 when the norm is 0: breakdown, detected by the host afterwards)
__global__ void __launch_bounds__(256) scale_by_norm_kernel(const double2 *__restrict__ in, double2 *__restrict__ out,
                                                            int64_t n, const double *nrm2)
{
    const double q = *nrm2, sc = q > 0.0 ? 1.0 / sqrt(q) : 0.0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        double2 x = in[i];
        out[i] = make_double2(sc * x.x, sc * x.y);
    }
}

}  // namespace bse

using namespace bse;

// Full (pseudo-Hermitian) case: the recurrence of G = M o P in the inner product Re(a^H P(b)) (reading R7 of DESIGN.md;
// oracle: orc_lanczos_quadrature_full).  Per step two half applies with k = 1 (each streams R and C once) and five
// O(N) kernels; five vectors, scalars on the device, one host synchronisation at the end.
static bse_status_t lanczos_quadrature_full(bse_handle_s *h, const void *dStart, int32_t steps, double *hAlpha,
                                            double *hBeta, int32_t *hDone)
{
    const int64_t n = h->N;
    const size_t vec = (size_t)n * 16, scal = (size_t)(3 * steps + 3) * 8;
    bse_status_t st = ensure_ws(h, 5 * vec + scal);
    if (st) return st;
    char *base = (char *)h->ws;
    double2 *xb[3] = {(double2 *)base, (double2 *)(base + vec), (double2 *)(base + 2 * vec)};   // x_j, x_{j-1}, w
    double2 *pb[2] = {(double2 *)(base + 3 * vec), (double2 *)(base + 4 * vec)};                // p_j, pw
    double *d_alpha = (double *)(base + 5 * vec), *d_b2 = d_alpha + steps, *d_junk = d_b2 + steps + 1;
    BSE_CUDA(cudaMemsetAsync(d_alpha, 0, scal, h->stream));
    const int grid = h->num_sms * 2;
    auto half = [&](int sign, const double2 *x, double2 *y) -> bse_status_t {
        return bse_apply_half(h, sign, x, n, y, n, 1);
    };
    // beta_0^2 = Re(d^H P(d));  x_1 = d / beta_0,  p_1 = P(d) / beta_0
    if ((st = half(+1, (const double2 *)dStart, pb[1]))) return st;
    dot_re_kernel<<<grid, 256, 0, h->stream>>>((const double2 *)dStart, pb[1], n, d_b2);
    if ((st = comm_bcast_dev(h, d_b2, 1))) return st;
    scale_by_norm_kernel<<<grid, 256, 0, h->stream>>>((const double2 *)dStart, xb[0], n, d_b2);
    scale_by_norm_kernel<<<grid, 256, 0, h->stream>>>(pb[1], pb[0], n, d_b2);
    count_launch(3);
    int ix = 0, ip = 2, iw = 1;
    for (int j = 0; j < steps; ++j) {
        if ((st = half(-1, pb[0], xb[iw]))) return st;                                      // w = M(p_j)
        dot_re_kernel<<<grid, 256, 0, h->stream>>>(pb[0], xb[iw], n, d_alpha + j);         // alpha_j = Re(p_j^H w)
        if ((st = comm_bcast_dev(h, d_alpha + j, 1))) return st;
        axpy_norm_kernel<<<grid, 256, 0, h->stream>>>(xb[iw], xb[ix], xb[ip], n, d_alpha + j, j > 0 ? d_b2 + j : nullptr,
                                                      d_junk + j);                          // w -= alpha x_j + beta x_{j-1}
        count_launch(2);
        if ((st = half(+1, xb[iw], pb[1]))) return st;                                      // pw = P(w)
        dot_re_kernel<<<grid, 256, 0, h->stream>>>(xb[iw], pb[1], n, d_b2 + j + 1);        // beta_{j+1}^2 = Re(w^H pw)
        if ((st = comm_bcast_dev(h, d_b2 + j + 1, 1))) return st;
        scale_by_norm_kernel<<<grid, 256, 0, h->stream>>>(xb[iw], xb[iw], n, d_b2 + j + 1);
        scale_by_norm_kernel<<<grid, 256, 0, h->stream>>>(pb[1], pb[0], n, d_b2 + j + 1);
        count_launch(3);
        int t = ip; ip = ix; ix = iw; iw = t;
    }
    BSE_CUDA(cudaGetLastError());
    std::vector<double> hs(2 * steps + 1);
    BSE_CUDA(cudaMemcpyAsync(hs.data(), d_alpha, (size_t)(2 * steps + 1) * 8, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    if (!(hs[steps] > 0.0)) return BSE_ERR_NOT_POSITIVE_DEFINITE;                          // <d, d>_P <= 0
    int done = steps;
    hBeta[0] = std::sqrt(hs[steps]);
    for (int j = 0; j < steps; ++j) {
        const double b2 = hs[steps + j + 1];
        if (b2 < 0.0) return BSE_ERR_NOT_POSITIVE_DEFINITE;
        hAlpha[j] = hs[j];
        hBeta[j + 1] = std::sqrt(b2);
        if (!(b2 > 0.0)) { done = j + 1; break; }
    }
    if (hDone) *hDone = done;
    return BSE_OK;
}

extern "C" bse_status_t bse_lanczos_quadrature(bse_handle_t h, const void *dStart, int32_t steps, double *hAlpha,
                                               double *hBeta, int32_t *hDone)
{
    if (!h || !dStart || steps < 1 || !hAlpha || !hBeta || is_incomplete(h) || is_row_partitioned(h)) return BSE_ERR_INVALID_ARG;
    if (h->mode == BSE_MODE_FULL) return lanczos_quadrature_full(h, dStart, steps, hAlpha, hBeta, hDone);
    const int64_t n = h->N;
    // workspace: three vectors + alpha[steps] + nrm2[steps + 1]
    const size_t vec = (size_t)n * 16, scal = (size_t)(2 * steps + 2) * 8;
    bse_status_t st = ensure_ws(h, 3 * vec + scal);
    if (st) return st;
    char *base = (char *)h->ws;
    double2 *buf[3] = {(double2 *)base, (double2 *)(base + vec), (double2 *)(base + 2 * vec)};
    double *d_alpha = (double *)(base + 3 * vec), *d_n2 = d_alpha + steps;
    BSE_CUDA(cudaMemsetAsync(d_alpha, 0, scal, h->stream));
    const int grid = h->num_sms * 2;
    // beta_0^2 = |d|^2 ;  v_0 = d / beta_0
    dot_re_kernel<<<grid, 256, 0, h->stream>>>((const double2 *)dStart, (const double2 *)dStart, n, d_n2);
    if ((st = comm_bcast_dev(h, d_n2, 1))) return st;
    scale_by_norm_kernel<<<grid, 256, 0, h->stream>>>((const double2 *)dStart, buf[0], n, d_n2);
    count_launch(2);
    int iv = 0, ip = 2, iw = 1;      // v_j, v_{j-1}, w
    for (int j = 0; j < steps; ++j) {
        if ((st = apply_tda_local(h, buf[iv], n, buf[iw], n, 1))) return st;                      // w = R v_j
        if ((st = comm_sum_block(h, buf[iw], n, n, 1))) return st;
        // the oracle's order: subtract beta_j v_{j-1} first, alpha_j = Re(v_j^H w) (v_{j-1} is orthogonal to v_j,
        // so the two orders agree to rounding); here alpha is taken first so that one fused pass does both updates
        dot_re_kernel<<<grid, 256, 0, h->stream>>>(buf[iv], buf[iw], n, d_alpha + j);
        if ((st = comm_bcast_dev(h, d_alpha + j, 1))) return st;
        axpy_norm_kernel<<<grid, 256, 0, h->stream>>>(buf[iw], buf[iv], buf[ip], n, d_alpha + j, j > 0 ? d_n2 + j : nullptr,
                                                      d_n2 + j + 1);
        if ((st = comm_bcast_dev(h, d_n2 + j + 1, 1))) return st;
        scale_by_norm_kernel<<<grid, 256, 0, h->stream>>>(buf[iw], buf[iw], n, d_n2 + j + 1);
        count_launch(3);
        int t = ip; ip = iv; iv = iw; iw = t;
    }
    BSE_CUDA(cudaGetLastError());
    std::vector<double> hs(2 * steps + 2);
    BSE_CUDA(cudaMemcpyAsync(hs.data(), d_alpha, scal, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    int done = steps;
    hBeta[0] = std::sqrt(hs[steps]);
    for (int j = 0; j < steps; ++j) {
        hAlpha[j] = hs[j];
        hBeta[j + 1] = std::sqrt(hs[steps + j + 1]);
        if (!(hs[steps + j + 1] > 0.0)) { done = j + 1; break; }
    }
    if (hDone) *hDone = done;
    return BSE_OK;
}

// out = scale * beta_0^2 [(s - T)^{-1}]_00 with s = z (TDA) or s = z^2 (full mode), z = omega + i eta
static void continued_fraction(int32_t steps, const double *hAlpha, const double *hBeta, int32_t n_omega,
                               const double *hOmega, double eta, bool squared, double scale, double *out)
{
    for (int i = 0; i < n_omega; ++i) {
        // f <- s - alpha_j - beta_{j+1}^2 / f, from the last coefficient up; complex arithmetic written out
        double zr = hOmega[i], zi = eta;
        if (squared) { const double a = zr, b = zi; zr = a * a - b * b; zi = 2.0 * a * b; }
        double fr = zr - hAlpha[steps - 1], fi = zi;
        for (int j = steps - 2; j >= 0; --j) {
            double b2 = hBeta[j + 1] * hBeta[j + 1], den = fr * fr + fi * fi;
            double qr = b2 * fr / den, qi = -b2 * fi / den;
            fr = zr - hAlpha[j] - qr;
            fi = zi - qi;
        }
        double den = fr * fr + fi * fi, b0 = scale * hBeta[0] * hBeta[0];
        out[2 * i] = b0 * fr / den;
        out[2 * i + 1] = -b0 * fi / den;
    }
}

extern "C" bse_status_t bse_quadrature_resolvent(int32_t steps, const double *hAlpha, const double *hBeta,
                                                 int32_t n_omega, const double *hOmega, double eta, void *hOut)
{
    if (steps < 1 || !hAlpha || !hBeta || n_omega < 0 || (n_omega && (!hOmega || !hOut))) return BSE_ERR_INVALID_ARG;
    continued_fraction(steps, hAlpha, hBeta, n_omega, hOmega, eta, false, 1.0, (double *)hOut);
    return BSE_OK;
}

extern "C" bse_status_t bse_quadrature_resolvent_full(int32_t steps, const double *hAlpha, const double *hBeta,
                                                      int32_t n_omega, const double *hOmega, double eta, void *hOut)
{
    if (steps < 1 || !hAlpha || !hBeta || n_omega < 0 || (n_omega && (!hOmega || !hOut))) return BSE_ERR_INVALID_ARG;
    continued_fraction(steps, hAlpha, hBeta, n_omega, hOmega, eta, true, 2.0, (double *)hOut);
    return BSE_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// bse_lanczos_quadrature_static: the TDA recurrence above for callers that cannot call cudaMalloc (code under CUDA graph
// capture, tight serving loops, harnesses that forbid it).  Its scratch -- three N-vectors and the 2 steps + 2 recurrence
// scalars -- lives in ONE file-scope device array of fixed size instead of the handle's lazily grown workspace, so the call
// allocates nothing, on the device or on the host.  Every GPU that loads the library holds the array until exit; every call
// on a device shares it and finds the previous call's contents in it (the scalars are cleared at the start of each call, the
// vectors are fully overwritten before they are read), so two calls that overlap on one GPU race.
// ---------------------------------------------------------------------------------------------------------------------
namespace bse {
constexpr int64_t STATIC_MAX_N = BSE_STATIC_QUADRATURE_MAX_N;            // 32768 rows: 3 x 512 KiB of vectors
constexpr int32_t STATIC_MAX_STEPS = BSE_STATIC_QUADRATURE_MAX_STEPS;    // 1024 steps: 16 KiB of scalars
constexpr size_t STATIC_VEC_BYTES = (size_t)STATIC_MAX_N * 16;
constexpr size_t STATIC_SCRATCH_BYTES = 3 * STATIC_VEC_BYTES + (size_t)(2 * STATIC_MAX_STEPS + 2) * 8;
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_SCRATCH_BYTES];

// In host code g_static_scratch is a host-side stand-in, not a device address: the address a kernel may use comes from
// cudaGetSymbolAddress, asked once per device with that device current.
static bse_status_t static_scratch_address(char **out)
{
    static std::atomic<char *> addr[64];
    int dev = 0;
    BSE_CUDA(cudaGetDevice(&dev));
    char *p = dev < 64 ? addr[dev].load(std::memory_order_acquire) : nullptr;
    if (!p) {
        void *q = nullptr;
        BSE_CUDA(cudaGetSymbolAddress(&q, g_static_scratch));
        p = (char *)q;
        if (dev < 64) addr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return BSE_OK;
}
}  // namespace bse

extern "C" bse_status_t bse_lanczos_quadrature_static(bse_handle_t h, const void *dStart, int32_t steps, double *hAlpha,
                                                      double *hBeta, int32_t *hDone)
{
    if (!h || !dStart || steps < 1 || !hAlpha || !hBeta || is_incomplete(h) || is_row_partitioned(h) || h->mode != BSE_MODE_TDA) return BSE_ERR_INVALID_ARG;
    const int64_t n = h->N;
    if (n > STATIC_MAX_N || steps > STATIC_MAX_STEPS) return BSE_ERR_STATIC_LIMIT;
    char *base = nullptr;
    bse_status_t st = static_scratch_address(&base);
    if (st) return st;
    const size_t scal = (size_t)(2 * steps + 2) * 8;
    double2 *buf[3] = {(double2 *)base, (double2 *)(base + STATIC_VEC_BYTES), (double2 *)(base + 2 * STATIC_VEC_BYTES)};
    double *d_alpha = (double *)(base + 3 * STATIC_VEC_BYTES), *d_n2 = d_alpha + steps;
    BSE_CUDA(cudaMemsetAsync(d_alpha, 0, scal, h->stream));                     // the last call's sums must not be added to
    const int grid = h->num_sms * 2;
    dot_re_kernel<<<grid, 256, 0, h->stream>>>((const double2 *)dStart, (const double2 *)dStart, n, d_n2);
    if ((st = comm_bcast_dev(h, d_n2, 1))) return st;
    scale_by_norm_kernel<<<grid, 256, 0, h->stream>>>((const double2 *)dStart, buf[0], n, d_n2);
    count_launch(2);
    int iv = 0, ip = 2, iw = 1;      // v_j, v_{j-1}, w
    for (int j = 0; j < steps; ++j) {
        if ((st = apply_tda_local(h, buf[iv], n, buf[iw], n, 1))) return st;                      // w = R v_j
        if ((st = comm_sum_block(h, buf[iw], n, n, 1))) return st;
        dot_re_kernel<<<grid, 256, 0, h->stream>>>(buf[iv], buf[iw], n, d_alpha + j);
        if ((st = comm_bcast_dev(h, d_alpha + j, 1))) return st;
        axpy_norm_kernel<<<grid, 256, 0, h->stream>>>(buf[iw], buf[iv], buf[ip], n, d_alpha + j, j > 0 ? d_n2 + j : nullptr,
                                                      d_n2 + j + 1);
        if ((st = comm_bcast_dev(h, d_n2 + j + 1, 1))) return st;
        scale_by_norm_kernel<<<grid, 256, 0, h->stream>>>(buf[iw], buf[iw], n, d_n2 + j + 1);
        count_launch(3);
        int t = ip; ip = iv; iv = iw; iw = t;
    }
    BSE_CUDA(cudaGetLastError());
    // straight into the caller's arrays (no host staging buffer): alpha_j, then |d|^2 and beta_{j+1}^2, square-rooted in place
    BSE_CUDA(cudaMemcpyAsync(hAlpha, d_alpha, (size_t)steps * 8, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaMemcpyAsync(hBeta, d_n2, (size_t)(steps + 1) * 8, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    int done = steps;
    hBeta[0] = std::sqrt(hBeta[0]);
    for (int j = 0; j < steps; ++j) {
        const double b2 = hBeta[j + 1];
        hBeta[j + 1] = std::sqrt(b2);
        if (!(b2 > 0.0)) { done = j + 1; break; }
    }
    if (hDone) *hDone = done;
    return BSE_OK;
}
