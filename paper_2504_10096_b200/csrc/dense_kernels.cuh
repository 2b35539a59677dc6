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
// One warp owns 8 columns of A (an M-tile) and streams a chunk of rows through its own ring of GRAM_DEPTH shared-memory
// stages (32 rows x 8 columns = 2 KB each) filled with cp.async: the basis is the HBM stream, and with 7 stages per warp
// in flight (112 KB per SM, one CTA of 8 warps per SM) its latency is covered without tying registers to loads.  The
// contraction index of a DMMA k-step is free to permute, so lane (g, t) takes the FOUR consecutive rows r + 4t .. r + 4t + 3
// of its column (two LDS.128; column stride == 16 (mod 128) bytes, no bank conflicts) and k-step s uses row r + 4t + s on
// both operands.  B fragments come through L1/L2.  Partial sums are reduced with red.global.add.f64.
// ------------------------------------------------------------------------------------------------------
constexpr int GRAM_WARPS = 16;                       // warps (8-column M-tiles) per CTA
constexpr int GRAM_DEPTH = 4;                        // ring stages per warp
constexpr int GRAM_COL_STRIDE = 256 + 16;            // bytes: 32 rows of one column + pad
constexpr int GRAM_STAGE_BYTES = 8 * GRAM_COL_STRIDE;
constexpr int GRAM_SMEM = GRAM_WARPS * GRAM_DEPTH * GRAM_STAGE_BYTES;

template <int NT>
__global__ void __launch_bounds__(32 * GRAM_WARPS, 1) gram_kernel(const double *__restrict__ A, int64_t lda2, int m,
                                                      const double *__restrict__ B, int64_t ldb2, int k, int ncols,
                                                      int64_t nr, int64_t rows_per_cta, double *__restrict__ out, int ldo,
                                                      int half_off)
{
    extern __shared__ __align__(16) char gram_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, t = lane & 3;
    const int c0 = (blockIdx.x * GRAM_WARPS + warp) * 8;
    if (c0 >= m) return;
    const int64_t r_begin = (int64_t)blockIdx.y * rows_per_cta;           // multiple of 32
    const int64_t r_end = min(nr, r_begin + rows_per_cta);                // even (nr = 2n)
    if (r_begin >= r_end) return;
    const bool aok = (c0 + g) < m;
    char *ring = gram_smem + warp * GRAM_DEPTH * GRAM_STAGE_BYTES;

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
    // two accumulator chains per N-tile: even and odd rows, so that the minus sign of (-i w)~ (plain FP64 instructions share
    // the issue port of the DMMAs) is applied once, at the end
    double acc[2][NT][2];
#pragma unroll
    for (int q = 0; q < NT; ++q) acc[0][q][0] = acc[0][q][1] = acc[1][q][0] = acc[1][q][1] = 0.0;

    // stage fill: 8 columns x 16 pieces of 16 bytes; half a warp covers the 256 contiguous bytes of one column
    auto fill = [&](int64_t r, int stage) {
        char *dst = ring + stage * GRAM_STAGE_BYTES;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int id = lane + 32 * j, col = id >> 4, piece = id & 15;
            const int64_t row = r + 2 * piece;
            const bool ok = (c0 + col) < m && row < r_end;                 // zero-filled otherwise
            const double *src = ok ? A + (int64_t)(c0 + col) * lda2 + row : A;
            cp_async16(dst + col * GRAM_COL_STRIDE + 16 * piece, src, ok);
        }
    };
    const int n_it = (int)((r_end - r_begin + 31) / 32);
#pragma unroll
    for (int i = 0; i < GRAM_DEPTH - 1; ++i) {
        if (i < n_it) fill(r_begin + 32 * i, i);
        cp_async_commit();
    }
    const double2 zero = make_double2(0.0, 0.0);
    constexpr int U = 2;
    // B fragments (L1 / L2 hits: all eight warps of the CTA read the same rows of B) are loaded one iteration ahead
    auto load_b = [&](int64_t r, double2 (&b)[NT][U][2]) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t row = r + 16 * u + 4 * t;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const bool rok = (row + 2 * h) < r_end;    // pairs never straddle r_end (both even)
#pragma unroll
                for (int q = 0; q < NT; ++q) b[q][u][h] = (bok[q] && rok) ? __ldg(bp[q] + ((row + 2 * h) >> 1)) : zero;
            }
        }
    };
    double2 bn[NT][U][2];
    load_b(r_begin, bn);
    for (int i = 0; i < n_it; ++i) {
        const int64_t r = r_begin + 32 * (int64_t)i;
        cp_async_wait<GRAM_DEPTH - 2>();                // this lane's pieces of stage i have landed ...
        __syncwarp();                                   // ... and so have everyone's; stage i - 1 is free again
        if (i + GRAM_DEPTH - 1 < n_it) fill(r + 32 * (GRAM_DEPTH - 1), (i + GRAM_DEPTH - 1) % GRAM_DEPTH);
        cp_async_commit();
        const char *as = ring + (i % GRAM_DEPTH) * GRAM_STAGE_BYTES + g * GRAM_COL_STRIDE + 32 * t;
        double2 a[U][2], b[NT][U][2];
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                a[u][h] = *reinterpret_cast<const double2 *>(as + 128 * u + 16 * h);
#pragma unroll
                for (int q = 0; q < NT; ++q)            // (-i w)~ : rows (2j, 2j+1) -> (w_i, -w_r); the sign is applied at the end
                    b[q][u][h] = brot[q] ? make_double2(bn[q][u][h].y, bn[q][u][h].x) : bn[q][u][h];
            }
        if (i + 1 < n_it) load_b(r + 32, bn);
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < NT; ++q) {
                    dmma(acc[0][q], a[u][h].x, b[q][u][h].x);      // chain 0: even rows (real parts of A)
                    dmma(acc[1][q], a[u][h].y, b[q][u][h].y);      // chain 1: odd rows (imaginary parts)
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
                    red_add(out + (c0 + g) + o, n < k ? acc[0][q][e] + acc[1][q][e] : acc[0][q][e] - acc[1][q][e]);
                }
            }
    }
}

}  // namespace bse
