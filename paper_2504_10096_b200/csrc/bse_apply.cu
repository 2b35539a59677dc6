// bse_apply / bse_apply_host: the general operator apply built from tile passes.
#include "bse_common.cuh"
#include "bse_internal.h"

namespace bse {

// dst(:, c) = conj(src(:, c))        (n rows, k columns)
__global__ void conj_copy_kernel(const double2 *__restrict__ src, int64_t lds, double2 *__restrict__ dst, int64_t ldd,
                                 int64_t n, int k)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (i < n && c < k) {
        double2 v = src[i + c * lds];
        dst[i + c * ldd] = make_double2(v.x, -v.y);
    }
}
// y(:, c) = -conj(y(:, c))
__global__ void neg_conj_inplace_kernel(double2 *__restrict__ y, int64_t ldy, int64_t n, int k)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (i < n && c < k) {
        double2 v = y[i + c * ldy];
        y[i + c * ldy] = make_double2(-v.x, v.y);
    }
}

// u = (x1 + conj x2) / 2,  v = (x1 - conj x2) / 2
__global__ void split_uv_kernel(const double2 *__restrict__ x1, const double2 *__restrict__ x2, int64_t ldx,
                                double2 *__restrict__ u, double2 *__restrict__ v, int64_t n, int k)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (i < n && c < k) {
        double2 a = x1[i + c * ldx], b = x2[i + c * ldx];
        u[i + c * n] = make_double2(0.5 * (a.x + b.x), 0.5 * (a.y - b.y));
        v[i + c * n] = make_double2(0.5 * (a.x - b.x), 0.5 * (a.y + b.y));
    }
}
// y1 = pu + mv,  y2 = -conj(pu - mv)
__global__ void combine_uv_kernel(const double2 *__restrict__ pu, const double2 *__restrict__ mv, double2 *__restrict__ y1,
                                  double2 *__restrict__ y2, int64_t ldy, int64_t n, int k)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (i < n && c < k) {
        double2 a = pu[i + c * n], b = mv[i + c * n];
        y1[i + c * ldy] = make_double2(a.x + b.x, a.y + b.y);
        y2[i + c * ldy] = make_double2(-(a.x - b.x), a.y - b.y);
    }
}

}  // namespace bse

using namespace bse;

extern "C" {

bse_status_t bse_apply(bse_handle_t h, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k)
{
    if (!h || !dX || !dY || k < 1 || dX == dY) return BSE_ERR_INVALID_ARG;
    const int64_t N = h->N;
    if (h->mode == BSE_MODE_TDA) {
        if (ldx < N || ldy < N) return BSE_ERR_INVALID_ARG;
        bse_status_t st = zero_block(h, dY, ldy, N, k);
        if (st) return st;
        if ((st = launch_apply_pass(h, h->R, 0 /*HERM*/, 1.0, dX, ldx, dY, ldy, k))) return st;
        return comm_sum_block(h, dY, ldy, N, k);
    }
    // FULL:  Y1 = R X1 + C X2 ;  Y2 = -conj( R conj(X2) + C conj(X1) )     (Eq. 1 with A = R^*, C = C^T)
    if (ldx < 2 * N || ldy < 2 * N) return BSE_ERR_INVALID_ARG;
    const double2 *X1 = (const double2 *)dX, *X2 = X1 + N;
    double2 *Y1 = (double2 *)dY, *Y2 = Y1 + N;
    if (h->real_form) {
        // real-form store (S = R + C, D = R - C): with U = (X1 + conj X2)/2, V = (X1 - conj X2)/2,
        //   Y1 = R X1 + C X2 = P(U) + M(V),   Y2 = -conj(R conj X2 + C conj X1) = -conj(P(U) - M(V))
        bse_status_t st = ensure_ws(h, (size_t)4 * N * k * 16);
        if (st) return st;
        double2 *U = (double2 *)h->ws, *V = U + (size_t)N * k, *PU = V + (size_t)N * k, *MV = PU + (size_t)N * k;
        dim3 grid((unsigned)((N + 255) / 256), (unsigned)k);
        split_uv_kernel<<<grid, 256, 0, h->stream>>>(X1, X2, ldx, U, V, N, k);
        count_launch();
        if ((st = bse_apply_half(h, +1, U, N, PU, N, k))) return st;
        if ((st = bse_apply_half(h, -1, V, N, MV, N, k))) return st;
        combine_uv_kernel<<<grid, 256, 0, h->stream>>>(PU, MV, Y1, Y2, ldy, N, k);
        count_launch();
        BSE_CUDA(cudaGetLastError());
        return BSE_OK;
    }
    bse_status_t st = ensure_ws(h, (size_t)N * k * 16);
    if (st) return st;
    double2 *T1 = (double2 *)h->ws;   // conj(X2), N x k, ld N
    dim3 grid((unsigned)((N + 255) / 256), (unsigned)k);
    conj_copy_kernel<<<grid, 256, 0, h->stream>>>(X2, ldx, T1, N, N, k);
    count_launch();
    st = zero_block(h, dY, ldy, 2 * N, k);
    if (st) return st;
    if ((st = launch_apply_pass(h, h->R, 0, 1.0, X1, ldx, Y1, ldy, k))) return st;   // Y1 += R X1
    if ((st = launch_apply_pass(h, h->C, 1, 1.0, T1, N, Y1, ldy, k))) return st;     // Y1 += C conj(conj X2)
    if ((st = launch_apply_pass(h, h->R, 0, 1.0, T1, N, Y2, ldy, k))) return st;     // Z  += R conj(X2)
    if ((st = launch_apply_pass(h, h->C, 1, 1.0, X1, ldx, Y2, ldy, k))) return st;   // Z  += C conj(X1)
    neg_conj_inplace_kernel<<<grid, 256, 0, h->stream>>>(Y2, ldy, N, k);             // Y2 = -conj(Z)
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return comm_sum_block(h, dY, ldy, 2 * N, k);
}

bse_status_t bse_apply_host(bse_handle_t h, const void *hX, int64_t ldx, void *hY, int64_t ldy, int32_t k)
{
    if (!h || !hX || !hY || k < 1) return BSE_ERR_INVALID_ARG;
    const int64_t n = (h->mode == BSE_MODE_FULL) ? 2 * h->N : h->N;
    if (ldx < n || ldy < n) return BSE_ERR_INVALID_ARG;
    bse_status_t st = ensure_ws2(h, (size_t)2 * n * k * 16);
    if (st) return st;
    char *dX = (char *)h->ws2, *dY = dX + (size_t)n * k * 16;
    BSE_CUDA(cudaMemcpy2DAsync(dX, (size_t)n * 16, hX, (size_t)ldx * 16, (size_t)n * 16, (size_t)k,
                               cudaMemcpyHostToDevice, h->stream));
    st = bse_apply(h, dX, n, dY, n, k);
    if (st) return st;
    BSE_CUDA(cudaMemcpy2DAsync(hY, (size_t)ldy * 16, dY, (size_t)n * 16, (size_t)n * 16, (size_t)k,
                               cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    return BSE_OK;
}

}  // extern "C"
