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
// One warp owns 8 columns of A (an M-tile) and streams a chunk of rows.  The contraction index of a DMMA k-step is
// free to permute, so lane (g, t) loads the FOUR consecutive rows r + 4t .. r + 4t + 3 of its column (two LDG.128,
// i.e. the four lanes of a column fetch one full 128-byte line) and k-step s uses row r + 4t + s on both operands.
// B fragments come through L1/L2.  Partial sums are reduced with red.global.add.f64.
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
    const int64_t r_begin = (int64_t)blockIdx.y * rows_per_cta;           // multiple of 16
    const int64_t r_end = min(nr, r_begin + rows_per_cta);                // even (nr = 2n)
    const bool aok = (c0 + g) < m;
    const double2 *ap = reinterpret_cast<const double2 *>(A + (int64_t)(aok ? c0 + g : 0) * lda2);

    const double2 *bp[NT];
    bool bok[NT], brot[NT];
#pragma unroll
    for (int q = 0; q < NT; ++q) {
        int n = 8 * q + g;
        bok[q] = n < ncols;
        brot[q] = n >= k;
        int col = bok[q] ? (brot[q] ? n - k : n) : 0;
        bp[q] = reinterpret_cast<const double2 *>(B + (int64_t)col * ldb2);
    }
    double acc[NT][2];
#pragma unroll
    for (int q = 0; q < NT; ++q) acc[q][0] = acc[q][1] = 0.0;

    // Software pipeline: the A loads (the HBM stream) of iteration i + 1 are issued before the DMMAs of iteration i, so
    // that every warp always has 2 x 16 rows of its 8 columns in flight; the B loads (L1 / L2 hits: all eight warps of
    // the CTA read the same rows of B) are issued just in time.
    constexpr int U = 2;                                   // 2 x 16 rows per iteration (4 x 16 measured slower: 2.5 vs 2.07 ms per bse_orth call)
    const double2 zero = make_double2(0.0, 0.0);
    auto load_a = [&](int64_t r, double2 (&a)[U][2]) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t row = r + 16 * u + 4 * t;        // first of this lane's four rows (even)
#pragma unroll
            for (int h = 0; h < 2; ++h)
                a[u][h] = (aok && (row + 2 * h) < r_end) ? __ldg(ap + ((row + 2 * h) >> 1)) : zero;
        }
    };
    double2 an[U][2];
    load_a(r_begin, an);
    for (int64_t r = r_begin; r < r_end; r += 16 * U) {
        double2 a[U][2], b[NT][U][2];
#pragma unroll
        for (int u = 0; u < U; ++u) { a[u][0] = an[u][0]; a[u][1] = an[u][1]; }
        if (r + 16 * U < r_end) load_a(r + 16 * U, an);
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t row = r + 16 * u + 4 * t;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const bool rok = (row + 2 * h) < r_end;    // pairs never straddle r_end (both even)
#pragma unroll
                for (int q = 0; q < NT; ++q) {
                    double2 v = (bok[q] && rok) ? __ldg(bp[q] + ((row + 2 * h) >> 1)) : zero;
                    if (brot[q]) v = make_double2(v.y, -v.x);          // (-i w)~ : rows (2j, 2j+1) -> (w_i, -w_r)
                    b[q][u][h] = v;
                }
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < NT; ++q) {
                    dmma(acc[q], a[u][h].x, b[q][u][h].x);
                    dmma(acc[q], a[u][h].y, b[q][u][h].y);
                }
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
