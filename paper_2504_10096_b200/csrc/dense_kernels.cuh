// Tall-skinny dense kernels of the Krylov basis on the FP64 tensor cores.
//
// Every complex n x m block is viewed as a REAL 2n x m matrix (re/im interleaved down the rows, leading
// dimension 2 ld), so that
//   Re(V^H W)  = V~^T W~                      Im(V^H W)  = V~^T (-iW)~         (-iW)~: row 2i -> w_i, 2i+1 -> -w_r
//   (V S)~     = V~ Re(S) + (iV)~ Im(S)       (iV)~: row 2i -> -v_i, row 2i+1 -> v_r
// and both the complex (TDA) and the real-coefficient (full mode, reading S4) variants are real GEMMs issued
// as mma.sync m8n8k4 f64 (DMMA.8x8x4).
#pragma once
#include "bse_common.cuh"

namespace bse {

// ------------------------------------------------------------------------------------------------------
// gram:  out[a + o(n)] += sum_r A~[r, a] * Bx[r, n],   a < m,  n < ncols,  o(n) = n ldo  or  half_off + (n-k) ldo
//   Bx columns n < k      : B~[:, n]
//   Bx columns k <= n < 2k: (-iB)~[:, n - k]            (only when ncols == 2k, the complex case)
// One warp owns 8 columns of A (an M-tile) and streams a chunk of rows with 32-byte sector loads straight
// into DMMA A-fragments; B fragments come through L1/L2.  Partial sums are reduced with red.global.add.f64.
// ------------------------------------------------------------------------------------------------------
template <int NT>
__global__ void __launch_bounds__(256) gram_kernel(const double *__restrict__ A, int64_t lda2, int m,
                                                   const double *__restrict__ B, int64_t ldb2, int k, int ncols,
                                                   int64_t nr, int64_t rows_per_cta, double *__restrict__ out, int ldo,
                                                   int half_off)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, t = lane & 3;
    const int c0 = blockIdx.x * 64 + warp * 8;
    if (c0 >= m) return;
    const int64_t r_begin = (int64_t)blockIdx.y * rows_per_cta;
    const int64_t r_end = min(nr, r_begin + rows_per_cta);
    const bool aok = (c0 + g) < m;
    const double *ap = A + (int64_t)(aok ? c0 + g : 0) * lda2;

    // per n-tile B column pointer / rotation flag for this lane (n = 8 q + g)
    const double *bp[NT];
    bool bok[NT], brot[NT];
#pragma unroll
    for (int q = 0; q < NT; ++q) {
        int n = 8 * q + g;
        bok[q] = n < ncols;
        brot[q] = n >= k;
        int col = bok[q] ? (brot[q] ? n - k : n) : 0;
        bp[q] = B + (int64_t)col * ldb2;
    }
    double acc[NT][2];
#pragma unroll
    for (int q = 0; q < NT; ++q) acc[q][0] = acc[q][1] = 0.0;

    constexpr int U = 4;
    for (int64_t r = r_begin; r < r_end; r += 4 * U) {
        double a[U], b[NT][U];
#pragma unroll
        for (int s = 0; s < U; ++s) {
            int64_t row = r + 4 * s + t;
            bool rok = row < r_end;
            a[s] = (aok && rok) ? ap[row] : 0.0;
#pragma unroll
            for (int q = 0; q < NT; ++q) {
                double v = 0.0;
                if (bok[q] && rok) {
                    if (!brot[q]) v = bp[q][row];
                    else { v = bp[q][row ^ 1]; if (row & 1) v = -v; }
                }
                b[q][s] = v;
            }
        }
#pragma unroll
        for (int s = 0; s < U; ++s)
#pragma unroll
            for (int q = 0; q < NT; ++q) dmma(acc[q], a[s], b[q][s]);
    }
    // C fragment: rows (A column) c0 + g, columns n = 8 q + 2 t, + 1
    if (aok) {
#pragma unroll
        for (int q = 0; q < NT; ++q)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                int n = 8 * q + 2 * t + e;
                if (n < ncols) {
                    // coefficient layout: real part of column c at c * ldo, imaginary part at half_off + c * ldo
                    int64_t o = (n < k) ? (int64_t)n * ldo : (int64_t)half_off + (int64_t)(n - k) * ldo;
                    red_add(out + (c0 + g) + o, acc[q][e]);
                }
            }
    }
}

}  // namespace bse
