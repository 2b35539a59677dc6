// bse_solve_direct: the diagonalisation scheme of PAPER.md section 2.1 (Eq. 2-4) on the GPU, for full-mode handles.
//
//   1. M_r (Eq. 3), real symmetric 2N x 2N, from the packed tiles of R and C          (build_mr_kernel)
//   2. Cholesky M_r = L L^T, blocked: 64 x 64 diagonal factor + its inverse in one CTA, panel and trailing
//      update as real GEMMs on the FP64 tensor cores (gemm_nn_kernel)
//   3. W = L^T J L, real skew-symmetric: one GEMM of L^T with the row-permuted copy J L
//   4. Householder tridiagonalisation of W in real arithmetic ("the tridiagonalization of a real matrix instead of a
//      Hermitian one"): H W H = W + tau (v p^T - p v^T) with p = W v, because v^T W v = 0 for a skew W
//   5. -i T is Hermitian tridiagonal with zero diagonal ("multiplying the result by -i allows the use of
//      Hermitian tridiagonal solvers"); D = diag((-i)^j) makes it the real symmetric S = tridiag(b, 0, b), whose even and
//      odd entries decouple: S ~ [[0, B^T], [B, 0]] with B upper bidiagonal, so omega^2 and the even half of an
//      eigenvector come from the N x N tridiagonal B^T B (host QL, as the projected problem of the iterative path),
//      the odd half is B s_E / omega
//   6. back-transformation (Eq. 4): z = H_0 ... H_{n-3} D s,  L^T y = z,  [X; Y] = Q y with Q of Eq. (2),
//      normalised X^H X - Y^H Y = 1
// Everything O(n^3) runs on the device; the host sequences kernels and solves the tridiagonal problem.
#include <algorithm>
#include <cmath>
#include <ctime>
#include <vector>

#include "bse_common.cuh"
#include "bse_internal.h"

namespace bse {

constexpr int DNB = 64;                         // block size of the Cholesky and of the triangular solve

// entry (i, j) of a packed store (lower triangle of tiles; diagonal tiles hold both triangles), as complex128
template <int ES>
__device__ __forceinline__ double2 store_entry(const char *tiles, int64_t i, int64_t j)
{
    const int64_t I = i >> 6, J = j >> 6;
    const char *p = tiles + tile_index(I, J) * tile_bytes_es(ES) + tile_offset_es((int)(i & 63), (int)(j & 63), ES);
    if (ES == 16) return *reinterpret_cast<const double2 *>(p);
    const float2 f = *reinterpret_cast<const float2 *>(p);
    return make_double2((double)f.x, (double)f.y);
}

// M_r = [[Re(R + C), Im(R - C)], [-Im(R + C), Re(R - C)]]  (Eq. 3 as printed), column-major n x n, n = 2N.
// One thread per (i, j) of the N x N blocks; R_ij = conj(R_ji), C_ij = C_ji above the diagonal.
template <int ES>
__global__ void __launch_bounds__(256) build_mr_kernel(const char *R, const char *C, int64_t N, double *M)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t j = blockIdx.y;
    if (i >= N) return;
    double2 r, c;
    if (i >= j) { r = store_entry<ES>(R, i, j); c = store_entry<ES>(C, i, j); }
    else { r = store_entry<ES>(R, j, i); r.y = -r.y; c = store_entry<ES>(C, j, i); }
    if (i == j) r.y = 0.0;                                      // the diagonal of R is real (reading S14)
    const int64_t n = 2 * N;
    M[i + j * n] = r.x + c.x;
    M[i + (j + N) * n] = r.y - c.y;
    M[i + N + j * n] = -(r.y + c.y);
    M[i + N + (j + N) * n] = r.x - c.x;
}

// The same from a real-form store (S = R + C in `R`, D = R - C in `C`, bse_to_real_form): the four blocks are stored.
template <int ES>
__global__ void __launch_bounds__(256) build_mr_real_form_kernel(const char *S, const char *D, int64_t N, double *M)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t j = blockIdx.y;
    if (i >= N) return;
    // S_ji = conj(R_ij) + C_ij: Re S_ji = Re S_ij, Im S_ji = -Im D_ij; D likewise with S and D exchanged
    double2 s, d;
    if (i >= j) { s = store_entry<ES>(S, i, j); d = store_entry<ES>(D, i, j); }
    else {
        const double2 st = store_entry<ES>(S, j, i), dt = store_entry<ES>(D, j, i);
        s = make_double2(st.x, -dt.y);
        d = make_double2(dt.x, -st.y);
    }
    const int64_t n = 2 * N;
    M[i + j * n] = s.x;
    M[i + (j + N) * n] = d.y;
    M[i + N + j * n] = -s.y;
    M[i + N + (j + N) * n] = d.x;
}

// Cholesky of the 64 x 64 diagonal block at A (column-major, lda) in shared memory, one CTA of 64 threads: thread r owns
// row r.  Writes L (lower; the strict upper part is zeroed) back and inv(L)^T, column-major 64 x 64, to invT (the B operand
// of the panel GEMM A21 inv(L)^T and, as inv(L^T), of the triangular solve).  A pivot <= 0 sets *flag (PAPER.md:49:
// "If M is positive definite ... we can perform a Cholesky decomposition").
__global__ void __launch_bounds__(DNB) potrf_diag_kernel(double *A, int64_t lda, int nb, double *invT, int *flag)
{
    __shared__ double a[DNB][DNB + 1];
    const int r = threadIdx.x;                                  // nb <= DNB rows are active (the last block of a ragged n)
    for (int c = 0; c < DNB; ++c) a[r][c] = (r < nb && c < nb) ? A[r + c * lda] : (r == c ? 1.0 : 0.0);
    __syncthreads();
    for (int j = 0; j < nb; ++j) {
        const double d = a[j][j];
        if (!(d > 0.0)) {
            if (r == 0) *flag = 1;
            return;                                             // uniform: every thread reads the same pivot
        }
        const double s = sqrt(d);
        __syncthreads();
        if (r == j) a[j][j] = s;
        else if (r > j) a[r][j] /= s;
        __syncthreads();
        if (r > j)
            for (int c = j + 1; c <= r; ++c) a[r][c] -= a[r][j] * a[c][j];
        __syncthreads();
    }
    // thread r: column r of X = inv(L) by forward substitution L x = e_r; X[i][r] lives at invT[r + i * DNB], which is
    // entry (r, i) of (inv L)^T in column-major order (written and read back by this thread only); identity beyond nb
    for (int i = 0; i < DNB; ++i) {
        double v = 0.0;
        if (i >= r) {
            v = (i == r) ? 1.0 : 0.0;
            for (int q = r; q < i; ++q) v -= a[i][q] * invT[r + q * DNB];
            v /= a[i][i];
        }
        invT[r + i * DNB] = v;
    }
    if (r < nb)
        for (int c = 0; c < nb; ++c) A[r + c * lda] = (c <= r) ? a[r][c] : 0.0;
}

// dst (cols x rows, ldd) = src (rows x cols, lds)^T, with `lower_only`: entries of src above its diagonal read as zero
__global__ void __launch_bounds__(256) transpose_kernel(const double *src, int64_t lds, int64_t rows, int64_t cols,
                                                        double *dst, int64_t ldd, int lower_only)
{
    __shared__ double t[32][33];
    const int64_t r0 = blockIdx.x * 32ll, c0 = blockIdx.y * 32ll;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int q = ty; q < 32; q += 8) {
        const int64_t r = r0 + tx, c = c0 + q;
        t[q][tx] = (r < rows && c < cols && !(lower_only && c > r)) ? src[r + c * lds] : 0.0;
    }
    __syncthreads();
    for (int q = ty; q < 32; q += 8) {
        const int64_t c = c0 + tx, r = r0 + q;
        if (r < rows && c < cols) dst[c + r * ldd] = t[tx][q];
    }
}

// JL = J L with J = [[0, I], [-I, 0]] (Eq. 2): row i of J L is row i + N of L (i < N) or minus row i - N; L lower triangular
__global__ void __launch_bounds__(256) jl_kernel(const double *L, int64_t n, int64_t N, double *JL)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t c = blockIdx.y;
    if (i >= n) return;
    const int64_t src = i < N ? i + N : i - N;
    double v = (c <= src) ? L[src + c * n] : 0.0;
    JL[i + c * n] = i < N ? v : -v;
}


// ---- skew-symmetric Householder tridiagonalisation.  Only the strict lower triangle of W is read and written (W[c][r] =
// -W[r][c]).  Step j works on the trailing block T_j = W[j+1:, j+1:] (m = n - j - 1 rows) with the reflector v_j of column j:
//     T_j <- H T_j H = T_j + tau (v p^T - p v^T),  p = T_j v      (v^T T_j v = 0 for a skew matrix)
// and that update is applied lazily: to column j + 1 by the next house_kernel, to the rest, T_{j+1}, by the next
// skew_fused_kernel in the same pass that forms p_{j+1} = T_{j+1} v_{j+1} -- every step reads and writes the lower triangle
// once (8/3 n^3 bytes in all).

// Reflector of column j: first the pending update of step j - 1 (tau_{j-1}, vp = v_{j-1}, pp = p_{j-1}, both indexed from
// row j) on x = W[j+1:, j], then beta = -sign(x_0) ||x||, tau = (beta - x_0) / beta, v = (1, x_1.. / (x_0 - beta))
// (H = I - tau v v^T, H x = beta e_0); v is written over x (kept for the back-transformation) and to vn; pn is cleared.  One CTA.
__global__ void __launch_bounds__(1024) house_kernel(double *W, int64_t n, int64_t j, double *tau, double *beta,
                                                     const double *vp, const double *pp, double *vn, double *pn)
{
    __shared__ double red[32];
    __shared__ double s_scale;
    const int64_t m = n - j - 1;
    double *x = W + (j + 1) + j * n;
    const double tp = j > 0 ? tau[j - 1] : 0.0;
    if (tp != 0.0) {
        const double p0 = pp[0];                                   // v_{j-1}[0] = 1
        for (int64_t r = threadIdx.x; r < m; r += blockDim.x) x[r] += tp * (vp[r + 1] * p0 - pp[r + 1]);
        __syncthreads();
    }
    double acc = 0.0;
    for (int64_t r = 1 + threadIdx.x; r < m; r += blockDim.x) acc += x[r] * x[r];
    for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double xnorm2 = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) xnorm2 += red[w];
        const double alpha = x[0];
        double b = alpha, t = 0.0, sc = 0.0;
        if (xnorm2 != 0.0) {
            b = -copysign(sqrt(alpha * alpha + xnorm2), alpha);
            t = (b - alpha) / b;
            sc = 1.0 / (alpha - b);
        }
        beta[j] = b;
        tau[j] = t;
        s_scale = sc;
    }
    __syncthreads();
    const double sc = s_scale;
    for (int64_t r = threadIdx.x; r < m; r += blockDim.x) {
        const double v = r == 0 ? 1.0 : x[r] * sc;
        x[r] = v;
        vn[r] = v;
        pn[r] = 0.0;
    }
}

// One 64 x 64 tile (bi >= bj) of the lower triangle of T_j, CTA of 256 threads: w = W[r][c] + tau_{j-1} (vp_r pp_c - pp_r vp_c)
// (vp, pp: v_{j-1}, p_{j-1} indexed from row j + 1), stored back, and its two contributions to pn = T_j vn:
// pn_r += w vn_c,  pn_c -= w vn_r.
__global__ void __launch_bounds__(256, 3) skew_fused_kernel(double *W, int64_t n, int64_t j, const double *tau, const double *vp,
                                                         const double *pp, const double *vn, double *pn)
{
    const int bi = blockIdx.x, bj = blockIdx.y;                  // (a linear walk of the triangle measured slower: 3.04 vs 2.69 s at n = 16384)
    if (bj > bi) return;
    __shared__ double tile[64][65];
    __shared__ double vpr[64], ppr[64], vnr[64], vpc[64], ppc[64], vnc[64];
    const int64_t m = n - j - 1, r0 = bi * 64ll, c0 = bj * 64ll;
    const double tp = j > 0 ? tau[j - 1] : 0.0;
    const int t = threadIdx.x;
    if (t < 64) {
        const bool ok = r0 + t < m;
        vpr[t] = (ok && tp != 0.0) ? vp[r0 + t] : 0.0;
        ppr[t] = (ok && tp != 0.0) ? pp[r0 + t] : 0.0;
        vnr[t] = ok ? vn[r0 + t] : 0.0;
    } else if (t < 128) {
        const int q = t - 64;
        const bool ok = c0 + q < m;
        vpc[q] = (ok && tp != 0.0) ? vp[c0 + q] : 0.0;
        ppc[q] = (ok && tp != 0.0) ? pp[c0 + q] : 0.0;
        vnc[q] = ok ? vn[c0 + q] : 0.0;
    }
    __syncthreads();
    double *w0 = W + (j + 1 + r0) + (j + 1 + c0) * n;
    const int rr = t & 63, cq = t >> 6;
    const int64_t r = r0 + rr;
    double wv[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) {                                 // all loads of this thread in flight at once
        const int cc = cq + 4 * q;
        wv[q] = (r < m && c0 + cc < m && r > c0 + cc) ? w0[rr + (int64_t)cc * n] : 0.0;
    }
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const int cc = cq + 4 * q;
        double w = wv[q];
        if (tp != 0.0 && r < m && c0 + cc < m && r > c0 + cc) {
            w += tp * (vpr[rr] * ppc[cc] - ppr[rr] * vpc[cc]);
            w0[rr + (int64_t)cc * n] = w;
        }
        tile[cc][rr] = w;
    }
    __syncthreads();
    if (t < 64) {
        double a0 = 0.0, a1 = 0.0;
        for (int cc = 0; cc < 64; cc += 2) { a0 += tile[cc][t] * vnc[cc]; a1 += tile[cc + 1][t] * vnc[cc + 1]; }
        if (r0 + t < m) atomicAdd(pn + r0 + t, a0 + a1);
    } else if (t < 128) {
        const int q = t - 64;
        double a0 = 0.0, a1 = 0.0;
        for (int r = 0; r < 64; r += 2) { a0 += tile[q][r] * vnr[r]; a1 += tile[q][r + 1] * vnr[r + 1]; }
        if (c0 + q < m) atomicAdd(pn + c0 + q, -(a0 + a1));
    }
}

// z <- H_0 H_1 ... H_{n-3} z for one column of Z per CTA of 1024 threads.  Thread t owns the absolute rows t + 1024 q
// (q < PER, n <= 1024 PER) of the column, held in shared memory, for the whole kernel: a step needs one block-wide sum (the
// dot product; partial sums double-buffered, so one barrier per step) and nothing else crosses threads.  The reflector
// v_j = W[j+1:, j] (v_0 = 1 stored) is loaded once per step into registers, all loads in flight at once.
template <int PER>
__global__ void __launch_bounds__(1024) reflect_back_kernel(const double *W, int64_t n, const double *tau, double *Z, int64_t ldz)
{
    extern __shared__ double zc[];
    __shared__ double red[2][32];
    double *z = Z + blockIdx.x * ldz;
    const int t = threadIdx.x, warp = t >> 5;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        const int64_t a = t + 1024ll * q;
        if (a < n) zc[a] = z[a];
    }
    int buf = 0;
    for (int64_t j = n - 3; j >= 0; --j) {
        const double tj = tau[j];
        if (tj == 0.0) continue;                                    // uniform
        const double *col = W + j * n;
        double vv[PER];
        double acc = 0.0;
#pragma unroll
        for (int q = 0; q < PER; ++q) {
            const int64_t a = t + 1024ll * q;
            vv[q] = (a > j && a < n) ? col[a] : 0.0;
        }
#pragma unroll
        for (int q = 0; q < PER; ++q) {
            const int64_t a = t + 1024ll * q;
            if (a > j && a < n) acc += vv[q] * zc[a];
        }
        for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if ((t & 31) == 0) red[buf][warp] = acc;
        __syncthreads();
        double d = 0.0;
#pragma unroll
        for (int w = 0; w < 32; ++w) d += red[buf][w];
        const double f = tj * d;
#pragma unroll
        for (int q = 0; q < PER; ++q) {
            const int64_t a = t + 1024ll * q;
            if (a > j && a < n) zc[a] -= f * vv[q];
        }
        buf ^= 1;
    }
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        const int64_t a = t + 1024ll * q;
        if (a < n) z[a] = zc[a];
    }
}

// z_T = D s for every wanted eigenvector, D = diag((-i)^j): from the even half s_E (SE, N x nev) of the unit eigenvector of the
// zero-diagonal tridiagonal S = tridiag(b, 0, b), its odd half s_O = B s_E / omega (B upper bidiagonal: B[o][o] = b_{2o},
// B[o][o+1] = b_{2o+1}), both scaled by 1/sqrt 2:  Z = [Re | Im] (n x 2 nev, ld n): Re z_{2o} = (-1)^o s_E[o], Im z_{2o+1} = -(-1)^o s_O[o]
__global__ void __launch_bounds__(256) build_z_kernel(const double *SE, const double *b, const double *omega, int64_t N, int nev,
                                                      double *Z)
{
    const int64_t o = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int c = blockIdx.y;
    if (o >= N) return;
    const int64_t n = 2 * N;
    const double *se = SE + (int64_t)c * N;
    const double r2 = 0.70710678118654752440;
    const double even = se[o] * r2;
    const double odd = (b[2 * o] * se[o] + (o + 1 < N ? b[2 * o + 1] * se[o + 1] : 0.0)) / omega[c] * r2;
    const double sg = (o & 1) ? -1.0 : 1.0;
    double *zr = Z + (int64_t)c * n, *zi = Z + (int64_t)(nev + c) * n;
    zr[2 * o] = sg * even;
    zr[2 * o + 1] = 0.0;
    zi[2 * o] = 0.0;
    zi[2 * o + 1] = -sg * odd;
}

// Reflector panel of the blocked back-transformation: Vp (m x nb, ld m) = the reflectors j0 .. j0 + nbk - 1 restricted to rows
// j0 .. n - 1 (m = n - j0, even; row 0 is zero, column c starts at row c + 1; columns >= nbk are zero), and VpT (nb x m, ld nb)
// its transpose.
__global__ void __launch_bounds__(256) reflector_panel_kernel(const double *W, int64_t n, int64_t j0, int nbk, int nb, double *Vp,
                                                              double *VpT)
{
    const int64_t m = n - j0;
    const int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int c = blockIdx.y;
    if (r >= m) return;
    const double v = (c < nbk && r >= c + 1) ? W[(j0 + r) + (j0 + c) * n] : 0.0;
    Vp[r + (int64_t)c * m] = v;
    VpT[c + r * (int64_t)nb] = v;
}

// [X; Y] = Q y, Q = (1/sqrt 2) [[I, -iI], [I, iI]] (Eq. 2), y = Yr + i Yi (n x nev each, real, ld n), then X^H X - Y^H Y = 1.
// One CTA per eigenvector.  sig[c] receives the Sigma-norm before scaling (must be positive for a positive omega).
__global__ void __launch_bounds__(256) assemble_direct_kernel(const double *Yr, const double *Yi, int64_t n, int64_t N,
                                                              double2 *vec, int64_t ldvec, double *sig)
{
    __shared__ double red[8];
    __shared__ double s_scale;
    const int c = blockIdx.x;
    const double *yr = Yr + c * n, *yi = Yi + c * n;
    double2 *out = vec + c * ldvec;
    double acc = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += blockDim.x) {
        const double a1 = yr[i], b1 = yi[i], a2 = yr[i + N], b2 = yi[i + N];
        // x = (y1 - i y2)/sqrt2, y = (y1 + i y2)/sqrt2  with y1 = a1 + i b1, y2 = a2 + i b2
        const double xr = a1 + b2, xi = b1 - a2, wr = a1 - b2, wi = b1 + a2;
        acc += 0.5 * ((xr * xr + xi * xi) - (wr * wr + wi * wi));
    }
    for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += red[w];
        sig[c] = s;
        s_scale = s > 0.0 ? 1.0 / sqrt(2.0 * s) : 0.0;
    }
    __syncthreads();
    const double f = s_scale;
    for (int64_t i = threadIdx.x; i < N; i += blockDim.x) {
        const double a1 = yr[i], b1 = yi[i], a2 = yr[i + N], b2 = yi[i + N];
        out[i] = make_double2(f * (a1 + b2), f * (b1 - a2));
        out[i + N] = make_double2(f * (a1 - b2), f * (b1 + a2));
    }
}

}  // namespace bse

using namespace bse;

namespace {

// C (nr x l, ldc) = alpha A (nr x K, lda) B (K x l, ldb) + beta C, all real column-major; nr, lda, ldc even, A and C
// 16-byte aligned (every caller passes multiples of the 64-row block)
bse_status_t rgemm(bse_handle_s *h, int64_t nr, int l, int K, double alpha, const double *A, int64_t lda, const double *B,
                   int64_t ldb, double beta, double *C, int64_t ldc, bool a_upper = false, bool c_lower = false)
{
    if (nr <= 0 || l <= 0 || K <= 0) return BSE_OK;
    return gemm_basis(h, A, lda / 2, K, false, B, ldb, l, nr / 2, C, ldc / 2, alpha, beta, a_upper, c_lower);
}

struct DevBuf {
    void *p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    bse_status_t alloc(size_t bytes) { return cudaMalloc(&p, bytes) == cudaSuccess ? BSE_OK : BSE_ERR_ALLOC; }
    double *d() const { return (double *)p; }
};

double now_s()
{
    timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return ts.tv_sec + 1e-9 * ts.tv_nsec;
}

}  // namespace

extern "C" bse_status_t bse_solve_direct(bse_handle_t h, int32_t nev, double *hOmega, void *dVec, int64_t ldvec,
                                         double *hSeconds)
{
    if (!h || h->mode != BSE_MODE_FULL || is_partial(h) || is_row_partitioned(h) || nev < 1 || nev > h->N || !hOmega || (dVec && ldvec < 2 * h->N))
        return BSE_ERR_INVALID_ARG;
    const int64_t N = h->N, n = 2 * N;
    if (n > BSE_DIRECT_MAX_N) return BSE_ERR_INVALID_ARG;
    cudaStream_t s = h->stream;
    bse_status_t st;
    double t0 = now_s(), t_chol = 0, t_w = 0, t_tri = 0, t_eig = 0, t_back = 0;

    DevBuf A, U, JL, invT, panel, panelT, small;
    const size_t nn = (size_t)n * n * sizeof(double);
    if ((st = A.alloc(nn)) || (st = U.alloc(nn)) || (st = JL.alloc(nn)) ||
        (st = invT.alloc((size_t)((n + DNB - 1) / DNB) * DNB * DNB * sizeof(double))) || (st = panel.alloc((size_t)n * DNB * sizeof(double))) ||
        (st = panelT.alloc((size_t)n * DNB * sizeof(double))) || (st = small.alloc((size_t)(6 * n + 64) * sizeof(double))))
        return st;
    double *tau = small.d(), *beta = tau + n, *vbuf = beta + n, *pbuf = vbuf + 2 * n;      // v, p: two buffers each
    int *flag = (int *)(pbuf + 2 * n);
    BSE_CUDA(cudaMemsetAsync(flag, 0, sizeof(int), s));

    // ---- 1. M_r
    {
        dim3 grid((unsigned)((N + 255) / 256), (unsigned)N);
        if (h->real_form) {
            if (h->es == 16) build_mr_real_form_kernel<16><<<grid, 256, 0, s>>>(h->R, h->C, N, A.d());
            else build_mr_real_form_kernel<8><<<grid, 256, 0, s>>>(h->R, h->C, N, A.d());
        } else {
            if (h->es == 16) build_mr_kernel<16><<<grid, 256, 0, s>>>(h->R, h->C, N, A.d());
            else build_mr_kernel<8><<<grid, 256, 0, s>>>(h->R, h->C, N, A.d());
        }
        count_launch();
        BSE_CUDA(cudaGetLastError());
    }
    // ---- 2. blocked Cholesky, lower: A <- L (the strict upper triangle keeps entries of M_r; never read as L)
    const int nblk = (int)((n + DNB - 1) / DNB);                  // the last block of a ragged n is shorter (n is even, so is it)
    for (int b = 0; b < nblk; ++b) {
        const int64_t k0 = (int64_t)b * DNB;
        const int nb = (int)std::min<int64_t>(DNB, n - k0);
        const int64_t rows = n - k0 - nb;
        double *Akk = A.d() + k0 + k0 * n, *inv_b = invT.d() + (size_t)b * DNB * DNB;
        potrf_diag_kernel<<<1, DNB, 0, s>>>(Akk, n, nb, inv_b, flag);
        count_launch();
        if (rows <= 0) break;
        double *A21 = Akk + DNB, *A22 = Akk + DNB + DNB * n;
        // L21 = A21 inv(L11)^T
        if ((st = rgemm(h, rows, DNB, DNB, 1.0, A21, n, inv_b, DNB, 0.0, panel.d(), n))) return st;
        BSE_CUDA(cudaMemcpy2DAsync(A21, (size_t)n * 8, panel.d(), (size_t)n * 8, (size_t)rows * 8, DNB, cudaMemcpyDeviceToDevice, s));
        transpose_kernel<<<dim3((unsigned)((rows + 31) / 32), DNB / 32), 256, 0, s>>>(panel.d(), n, rows, DNB, panelT.d(), DNB, 0);
        count_launch();
        // A22 -= L21 L21^T (tiles on and below the diagonal: the upper triangle is never used)
        if ((st = rgemm(h, rows, (int)rows, DNB, -1.0, panel.d(), n, panelT.d(), DNB, 1.0, A22, n, false, true))) return st;
    }
    BSE_CUDA(cudaGetLastError());
    int hflag = 0;
    BSE_CUDA(cudaMemcpyAsync(&hflag, flag, sizeof(int), cudaMemcpyDeviceToHost, s));
    BSE_CUDA(cudaStreamSynchronize(s));
    if (hflag) return BSE_ERR_NOT_POSITIVE_DEFINITE;
    t_chol = now_s() - t0;

    // ---- 3. W = L^T (J L)  -> A
    double t1 = now_s();
    transpose_kernel<<<dim3((unsigned)((n + 31) / 32), (unsigned)((n + 31) / 32)), 256, 0, s>>>(A.d(), n, n, n, U.d(), n, 1);
    jl_kernel<<<dim3((unsigned)((n + 255) / 256), (unsigned)n), 256, 0, s>>>(A.d(), n, N, JL.d());
    count_launch(2);
    if ((st = rgemm(h, n, (int)n, (int)n, 1.0, U.d(), n, JL.d(), n, 0.0, A.d(), n, true))) return st;      // U upper triangular
    BSE_CUDA(cudaStreamSynchronize(s));
    t_w = now_s() - t1;

    // ---- 4. skew tridiagonalisation of W (in A); sub-diagonal in beta, reflectors below it
    t1 = now_s();
    for (int64_t j = 0; j + 1 < n; ++j) {
        const int64_t m = n - j - 1;
        double *vp = vbuf + ((j + 1) & 1) * n, *pp = pbuf + ((j + 1) & 1) * n, *vn = vbuf + (j & 1) * n, *pn = pbuf + (j & 1) * n;
        house_kernel<<<1, 1024, 0, s>>>(A.d(), n, j, tau, beta, vp, pp, vn, pn);
        count_launch();
        if (m < 2) break;                                          // the last entry is its own sub-diagonal (tau = 0)
        const unsigned nbt = (unsigned)((m + 63) / 64);
        skew_fused_kernel<<<dim3(nbt, nbt), 256, 0, s>>>(A.d(), n, j, tau, vp + 1, pp + 1, vn, pn);
        count_launch();
    }
    BSE_CUDA(cudaGetLastError());
    std::vector<double> hb(n), htau(n);
    BSE_CUDA(cudaMemcpyAsync(hb.data(), beta, (size_t)(n - 1) * 8, cudaMemcpyDeviceToHost, s));
    BSE_CUDA(cudaStreamSynchronize(s));
    t_tri = now_s() - t1;

    // ---- 5. S = tridiag(b, 0, b) (n x n) = perfect shuffle of [[0, B^T], [B, 0]], B upper bidiagonal N x N with
    //         B[o][o] = b_{2o}, B[o][o+1] = b_{2o+1}:  B^T B s_E = omega^2 s_E,  s_O = B s_E / omega
    t1 = now_s();
    std::vector<double> dE(N), eE(N, 0.0), w2(nev), ZE(dVec ? (size_t)N * nev : 0);
    for (int64_t e = 0; e < N; ++e) {
        const double bd = hb[2 * e], bu = e > 0 ? hb[2 * e - 1] : 0.0;
        dE[e] = bd * bd + bu * bu;
        if (e + 1 < N) eE[e] = hb[2 * e] * hb[2 * e + 1];
    }
    if (host_stev_lowest((int)N, dE.data(), eE.data(), nev, w2.data(), dVec ? ZE.data() : nullptr, (int)N)) return BSE_ERR_INTERNAL;
    for (int c = 0; c < nev; ++c) {
        if (!(w2[c] > 0.0)) return BSE_ERR_NOT_POSITIVE_DEFINITE;
        hOmega[c] = std::sqrt(w2[c]);
    }
    t_eig = now_s() - t1;
    if (!dVec) {
        if (hSeconds) { hSeconds[0] = t_chol; hSeconds[1] = t_w; hSeconds[2] = t_tri; hSeconds[3] = t_eig; hSeconds[4] = 0.0; hSeconds[5] = now_s() - t0; }
        return BSE_OK;
    }

    // ---- 6. back-transformation.  z_T = D s with D = diag((-i)^j): Z = [Re | Im], n x 2 nev real
    t1 = now_s();
    const bool verbose = getenv("BSE_VERBOSE") != nullptr;
    double t_lap = t1;
    auto lap = [&](const char *what) {
        if (!verbose) return;
        cudaStreamSynchronize(s);
        const double t = now_s();
        fprintf(stderr, "[bse_solve_direct] %s: %.3f s\n", what, t - t_lap);
        t_lap = t;
    };
    DevBuf Z, Ytmp;
    const int l2 = 2 * nev;
    if ((st = Z.alloc((size_t)n * l2 * sizeof(double))) || (st = Ytmp.alloc((size_t)DNB * l2 * sizeof(double)))) return st;
    {
        // s_E, omega to the device (the sub-diagonal b is still there): the start vectors are formed by a kernel
        DevBuf SE, omd;
        if ((st = SE.alloc((size_t)N * nev * 8)) || (st = omd.alloc((size_t)nev * 8))) return st;
        BSE_CUDA(cudaMemcpyAsync(SE.d(), ZE.data(), (size_t)N * nev * 8, cudaMemcpyHostToDevice, s));
        BSE_CUDA(cudaMemcpyAsync(omd.d(), hOmega, (size_t)nev * 8, cudaMemcpyHostToDevice, s));
        build_z_kernel<<<dim3((unsigned)((N + 255) / 256), nev), 256, 0, s>>>(SE.d(), beta, omd.d(), N, nev, Z.d());
        count_launch();
        BSE_CUDA(cudaGetLastError());
        BSE_CUDA(cudaStreamSynchronize(s));                        // SE, omd are freed here
        lap("start vectors");
    }
    constexpr int RNB = 32;                                        // reflectors per block of the compact WY form
    // (per block: a panel kernel, a Gram, one host round trip for T, three GEMMs -- n / 32 of them; below ~256 vectors the
    //  one-CTA-per-column kernel, whose cost grows with the number of columns, is faster: 0.15 vs 0.28 s at n = 16384, nev = 100)
    if (l2 >= 512 && n > 2 * RNB) {
        // Blocked: H_j0 ... H_j0+nb-1 = I - V T V^T (forward, columnwise: T upper triangular, T_ii = tau_i,
        // T[0:i, i] = -tau_i T[0:i, 0:i] (V^T V)[0:i, i]); on the transposed block ZT = Z^T (2 nev x n) the update is three
        // row-rich real GEMMs on the tensor cores:  ZT[:, rows] -= ((ZT[:, rows] V) T^T) V^T.
        DevBuf ZT, Vp, VpT, W1, W2, Gd;
        if ((st = ZT.alloc((size_t)n * l2 * 8)) || (st = Vp.alloc((size_t)n * RNB * 8)) || (st = VpT.alloc((size_t)n * RNB * 8)) ||
            (st = W1.alloc((size_t)l2 * RNB * 8)) || (st = W2.alloc((size_t)l2 * RNB * 8)) || (st = Gd.alloc((size_t)2 * RNB * RNB * 8)))
            return st;
        transpose_kernel<<<dim3((unsigned)((n + 31) / 32), (unsigned)((l2 + 31) / 32)), 256, 0, s>>>(Z.d(), n, n, l2, ZT.d(), l2, 0);
        count_launch();
        std::vector<double> htau(n, 0.0), G((size_t)RNB * RNB), TT((size_t)RNB * RNB);
        BSE_CUDA(cudaMemcpyAsync(htau.data(), tau, (size_t)(n - 1) * 8, cudaMemcpyDeviceToHost, s));
        BSE_CUDA(cudaStreamSynchronize(s));
        const int64_t nref = n - 2;                               // reflectors j = 0 .. n - 3
        for (int64_t j0 = ((nref - 1) / RNB) * RNB; j0 >= 0; j0 -= RNB) {
            const int nbk = (int)std::min<int64_t>(RNB, nref - j0);
            const int64_t m = n - j0;                              // rows j0 .. n - 1 (even; the first row of the panel is zero)
            reflector_panel_kernel<<<dim3((unsigned)((m + 255) / 256), RNB), 256, 0, s>>>(A.d(), n, j0, nbk, RNB, Vp.d(), VpT.d());
            count_launch();
            // G = V^T V (nb x nb) with the Gram kernel of the basis (real inner product over the m rows = m / 2 complex rows)
            if ((st = gram_basis(h, Vp.d(), m / 2, RNB, Vp.d(), m / 2, RNB, false, m / 2, Gd.d()))) return st;
            BSE_CUDA(cudaMemcpyAsync(G.data(), Gd.d(), (size_t)RNB * RNB * 8, cudaMemcpyDeviceToHost, s));
            BSE_CUDA(cudaStreamSynchronize(s));
            std::fill(TT.begin(), TT.end(), 0.0);                 // TT = T^T, column-major: TT[i + a * nb] = T[a, i]
            for (int i = 0; i < nbk; ++i) {
                const double ti = htau[j0 + i];
                TT[i + (size_t)i * RNB] = ti;
                for (int a = 0; a < i; ++a) {
                    double acc = 0.0;
                    for (int q = a; q < i; ++q) acc += TT[q + (size_t)a * RNB] * G[q + (size_t)i * RNB];      // T[a, q] G[q, i]
                    TT[i + (size_t)a * RNB] = -ti * acc;
                }
            }
            BSE_CUDA(cudaMemcpyAsync(Gd.d() + RNB * RNB, TT.data(), (size_t)RNB * RNB * 8, cudaMemcpyHostToDevice, s));
            double *Zr = ZT.d() + (size_t)j0 * l2;                // columns j0 .. n - 1 of ZT
            if ((st = rgemm(h, l2, RNB, (int)m, 1.0, Zr, l2, Vp.d(), m, 0.0, W1.d(), l2))) return st;
            if ((st = rgemm(h, l2, RNB, RNB, 1.0, W1.d(), l2, Gd.d() + RNB * RNB, RNB, 0.0, W2.d(), l2))) return st;
            if ((st = rgemm(h, l2, (int)m, RNB, -1.0, W2.d(), l2, VpT.d(), RNB, 1.0, Zr, l2))) return st;
            BSE_CUDA(cudaStreamSynchronize(s));                   // TT and G are reused by the next block
        }
        transpose_kernel<<<dim3((unsigned)((l2 + 31) / 32), (unsigned)((n + 31) / 32)), 256, 0, s>>>(ZT.d(), l2, l2, n, Z.d(), n, 0);
        count_launch();
        BSE_CUDA(cudaGetLastError());
    } else {
        const int per = (int)((n + 1023) / 1024);
        auto launch = [&](auto kern) -> bse_status_t {
            BSE_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(n * 8)));
            kern<<<l2, 1024, (size_t)n * 8, s>>>(A.d(), n, tau, Z.d(), n);
            return BSE_OK;
        };
        if (per <= 4) st = launch(reflect_back_kernel<4>);
        else if (per <= 8) st = launch(reflect_back_kernel<8>);
        else if (per <= 16) st = launch(reflect_back_kernel<16>);
        else st = launch(reflect_back_kernel<24>);
        if (st) return st;
        count_launch();
        BSE_CUDA(cudaGetLastError());
    }
    lap("reflectors");
    // L^T y = z: U y = z, blocked back substitution from the last block up
    for (int b = nblk - 1; b >= 0; --b) {
        const int64_t k0 = (int64_t)b * DNB;
        const int nb = (int)std::min<int64_t>(DNB, n - k0);
        const double *inv_b = invT.d() + (size_t)b * DNB * DNB;             // inv(L_bb)^T = inv(U_bb) (identity beyond nb)
        if ((st = rgemm(h, nb, l2, nb, 1.0, inv_b, DNB, Z.d() + k0, n, 0.0, Ytmp.d(), DNB))) return st;
        BSE_CUDA(cudaMemcpy2DAsync(Z.d() + k0, (size_t)n * 8, Ytmp.d(), (size_t)DNB * 8, (size_t)nb * 8, l2, cudaMemcpyDeviceToDevice, s));
        if (k0 > 0 && (st = rgemm(h, k0, l2, nb, -1.0, U.d() + k0 * n, n, Ytmp.d(), DNB, 1.0, Z.d(), n))) return st;
    }
    lap("triangular solve");
    double *sig = pbuf;
    assemble_direct_kernel<<<nev, 256, 0, s>>>(Z.d(), Z.d() + (size_t)nev * n, n, N, (double2 *)dVec, ldvec, sig);
    count_launch();
    BSE_CUDA(cudaGetLastError());
    std::vector<double> hs(nev);
    BSE_CUDA(cudaMemcpyAsync(hs.data(), sig, (size_t)nev * 8, cudaMemcpyDeviceToHost, s));
    BSE_CUDA(cudaStreamSynchronize(s));
    for (int c = 0; c < nev; ++c)
        if (!(hs[c] > 0.0)) return BSE_ERR_INTERNAL;
    t_back = now_s() - t1;
    if (hSeconds) { hSeconds[0] = t_chol; hSeconds[1] = t_w; hSeconds[2] = t_tri; hSeconds[3] = t_eig; hSeconds[4] = t_back; hSeconds[5] = now_s() - t0; }
    return BSE_OK;
}
