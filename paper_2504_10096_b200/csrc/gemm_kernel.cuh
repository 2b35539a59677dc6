// C~ = alpha * op(A) * Bm + beta * C~   on the FP64 tensor cores.
//   A~  : real view (2n x m, leading dimension lda2) of a complex n x m block of basis vectors
//   op(A) = A~                      (K = m,  real coefficients: full mode)
//         = [A~ | (iA)~]            (K = 2m, complex coefficients: rows 0..m-1 of Bm = Re(S), rows m..2m-1 = Im(S); every
//                                    chunk of A is brought to shared memory once and used with both halves of Bm)
//   Bm  : real K x l, column-major (ldb);   C~ : real view 2n x l (ldc2).
// Used for the Gram-Schmidt update W -= V h (skinny: l = k), the Ritz rotation V <- V S and the eigenvector
// assembly.  Shared-memory tiled (cp.async double buffering), mma.sync m8n8k4 f64 -> DMMA.8x8x4.
#pragma once
#include "bse_common.cuh"

namespace bse {

constexpr int GEMM_KC = 16;

template <int MT, int NT, int WM, int WN>
struct GemmCfg {
    static constexpr int NS = 2;   // shared-memory stages: the skinny (HBM-bound) shape keeps 4 chunks in flight
    static constexpr int BM = 8 * MT * WM, BN = 8 * NT * WN, THREADS = 32 * WM * WN;
    static constexpr int LDA_S = BM + 8;          // == 8 (mod 16) doubles: conflict-free A fragments
    static constexpr int LDB_S = GEMM_KC + 4;     // == 4 (mod 16) doubles: conflict-free B fragments
    static constexpr int SMEM = NS * (GEMM_KC * LDA_S + 2 * BN * LDB_S) * 8;     // B tile for Re(S) and Im(S)
};

template <int MT, int NT, int WM, int WN>
__global__ void __launch_bounds__(32 * WM * WN) gemm_nn_kernel(const double *__restrict__ A, int64_t lda2, int64_t nr,
                                                               int m, int flags, const double *__restrict__ Bm,
                                                               int64_t ldb, int l, double *__restrict__ C,
                                                               int64_t ldc2, double alpha, double beta)
{
    using Cfg = GemmCfg<MT, NT, WM, WN>;
    constexpr int BM = Cfg::BM, BN = Cfg::BN, KC = GEMM_KC, LDA_S = Cfg::LDA_S, LDB_S = Cfg::LDB_S, NS = Cfg::NS;
    extern __shared__ __align__(16) double gsm[];
    double *As = gsm;                                  // [NS][KC][LDA_S]
    double *Bs = gsm + NS * KC * LDA_S;                // [NS][2][BN][LDB_S]: buffer, half (Re S / Im S)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = lane >> 2, t = lane & 3;
    const int wm = warp % WM, wn = warp / WM;
    const int64_t row0 = (int64_t)blockIdx.x * BM;
    const int col0 = blockIdx.y * BN;
    // flags & 4: only the lower triangle of a square C is wanted (the trailing update of the Cholesky factorisation): tiles
    // entirely above the diagonal do nothing
    if ((flags & 4) && (int64_t)col0 >= row0 + BM) return;
    const int nch = (m + KC - 1) / KC;
    const int total = nch;                              // every chunk of A is loaded ONCE and used with Re(S) and with Im(S)
    // flags & 2: A is upper triangular (A[row, kk] = 0 for kk < row, the L^T of the direct route): the chunks left of this
    // row tile's diagonal are skipped
    const int c_begin = (flags & 2) ? (int)min((int64_t)nch, row0 / KC) : 0;
    const int cplx = flags & 1;
    const int nhalf = cplx ? 2 : 1;

    auto load_chunk = [&](int c, int buf) {
        const int kk0 = c * KC;
        double *as = As + buf * KC * LDA_S;
        double *bs = Bs + buf * 2 * BN * LDB_S;
        for (int idx = tid; idx < KC * (BM / 2); idx += Cfg::THREADS) {
            int kk = idx / (BM / 2), r2 = idx % (BM / 2);
            bool ok = (kk0 + kk) < m && (row0 + 2 * r2) < nr;
            const double *src = ok ? A + (int64_t)(kk0 + kk) * lda2 + row0 + 2 * r2 : A;
            cp_async16(as + kk * LDA_S + 2 * r2, src, ok);
        }
        for (int idx = tid; idx < nhalf * BN * KC; idx += Cfg::THREADS) {
            int half = idx / (BN * KC), rem = idx % (BN * KC);
            int col = rem / KC, kk = rem % KC;
            bool ok = (kk0 + kk) < m && (col0 + col) < l;
            const double *src = ok ? Bm + (int64_t)half * m + kk0 + kk + (int64_t)(col0 + col) * ldb : Bm;
            cp_async8(bs + half * BN * LDB_S + col * LDB_S + kk, src, ok);
        }
    };

    // (iA)~ Im(S): rows (2i, 2i+1) of (iA)~ are (-a_i, a_r); the sign depends on the parity of the lane's row only and is
    // flipped with an integer XOR (plain FP64 instructions share the issue port of the DMMAs)
    const unsigned long long im_flip = (g & 1) ? 0ull : SIGN_BIT;
    double acc[MT][NT][2];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
    for (int c = 0; c < NS - 1; ++c) {
        if (c_begin + c < total) load_chunk(c_begin + c, c);
        cp_async_commit();
    }
    for (int c = c_begin; c < total; ++c) {
        const int buf = (c - c_begin) % NS;
        if (c + NS - 1 < total) load_chunk(c + NS - 1, (c - c_begin + NS - 1) % NS);
        cp_async_commit();
        cp_async_wait<NS - 1>();
        __syncthreads();
        const double *as = As + buf * KC * LDA_S + wm * 8 * MT;
        const double *bs = Bs + buf * 2 * BN * LDB_S + (wn * 8 * NT) * LDB_S;
#pragma unroll
        for (int ks = 0; ks < KC / 4; ++ks) {
            const int kk = 4 * ks + t;
            double a[MT], b[NT];
#pragma unroll
            for (int i = 0; i < MT; ++i) a[i] = as[kk * LDA_S + 8 * i + g];
#pragma unroll
            for (int j = 0; j < NT; ++j) b[j] = bs[(8 * j + g) * LDB_S + kk];
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) dmma(acc[i][j], a[i], b[j]);
            if (cplx) {
#pragma unroll
                for (int i = 0; i < MT; ++i) a[i] = neg_if(as[kk * LDA_S + ((8 * i + g) ^ 1)], im_flip);
#pragma unroll
                for (int j = 0; j < NT; ++j) b[j] = bs[BN * LDB_S + (8 * j + g) * LDB_S + kk];
#pragma unroll
                for (int i = 0; i < MT; ++i)
#pragma unroll
                    for (int j = 0; j < NT; ++j) dmma(acc[i][j], a[i], b[j]);
            }
        }
        __syncthreads();
    }
    // epilogue: C fragment rows 8 i + g, columns 8 j + 2 t + e
#pragma unroll
    for (int i = 0; i < MT; ++i) {
        int64_t row = row0 + wm * 8 * MT + 8 * i + g;
        if (row >= nr) continue;
#pragma unroll
        for (int j = 0; j < NT; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                int col = col0 + wn * 8 * NT + 8 * j + 2 * t + e;
                if (col < l) {
                    double *cp = C + row + (int64_t)col * ldc2;
                    double v = alpha * acc[i][j][e];
                    if (beta != 0.0) v += beta * (*cp);
                    *cp = v;
                }
            }
    }
}

}  // namespace bse
