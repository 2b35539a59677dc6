// Structured block-matvec over the packed triangular tile store: what every apply kernel shares.
//
// One tile pass computes, for a group of columns of X,
//     HERM :  Y += s * R X            (R Hermitian, lower triangle stored)
//     SYMC :  Y += s * C conj(X)      (C complex symmetric, lower triangle stored)
// (or the real-form products of apply_tiles.cuh).  Every stored tile T = T_IJ (I >= J) is brought from HBM exactly once by
// ONE TMA bulk copy (cp.async.bulk -> UBLKCP, 64 KB, contiguous) into a 3-stage shared-memory ring and used twice from there:
//     P1:  Y_I += T   x_J            (HERM)      Y_I += T   conj(x_J)   (SYMC)
//     P2:  Y_J += T^H x_I            (HERM)      Y_J += T^T conj(x_I)   (SYMC)       (skipped when I == J)
//
// Work decomposition: a unit is a run of up to L consecutive tiles of one tile row I.  A CTA (8 consumer warps + 1 producer
// warp, persistent, one per SM) walks its units.  P1 partial sums stay in registers for a whole unit; P2 results are flushed
// per tile.  Partial results are added with red.global.add.f64.
//
// The shared-memory hazard found in round 1: releasing a stage with mbarrier.arrive right after the last ld.shared of that
// stage is not enough on B200 -- the arrive orders only the ISSUE of earlier loads, and queued loads of a slow warp were
// observed to execute after the producer's next bulk copy had landed (stale fragments about once per launch).  Every kernel
// therefore makes the barrier address of the arrive data-dependent on its accumulators (`live & zero`, zero a runtime 0 the
// assembler cannot fold): all MMAs / FMAs, hence all loads, have completed before the release issues.  (A predicate
// `live != const` is NOT safe: an OR of accumulator words can reproduce any constant and would skip the arrive.)
#pragma once
#include "bse_common.cuh"

namespace bse {

constexpr int APPLY_STAGES = 3;                          // ring depth for 64 KB (complex128) tiles; 6 for 32 KB (complex64)
constexpr int APPLY_CONSUMERS = 8;                       // consumer warps
constexpr int APPLY_THREADS = (APPLY_CONSUMERS + 1) * 32;
constexpr int APPLY_SMEM = APPLY_STAGES * TILE_BYTES + 128;

enum { PASS_HERM = 0, PASS_SYMC = 1 };

// parameters of the single-column (plain FMA) kernels, which read X and add to Y directly
struct ApplyParams {
    const char *tiles;
    const double2 *X;
    int64_t ldx;
    double *Y;          // complex128 viewed as doubles
    int64_t ldy;
    int64_t N;
    int nt;             // tile rows
    int kc;             // columns in this pass (1)
    int pass;           // PASS_HERM / PASS_SYMC
    double sign;        // s
    int L;              // unit length in tiles
    int64_t u_begin;    // first unit of this handle's tile rows (0 unless the handle is a shard)
    int64_t n_units;    // one past the last unit
    int zero;           // always 0; a runtime value the assembler cannot fold (see the stage release above)
};

// parameters of the tensor-core kernels (apply_tiles.cuh): operands come as images written by the pre-pass
// (apply_prep.cuh), partial results go to the padded block Ypad; no bounds checks anywhere in the tile loop
struct TileParams {
    const char *tiles;
    const double2 *img_pair;   // [rows_pad][8] (zr, zi)
    const double *img_a;       // [rows_pad][8]
    const double *img_b;       // [rows_pad][8]
    double *Ypad;              // [rows_pad][8] complex, as doubles
    int nt;
    int kc;                    // live columns (the images of the others are zero; their results are not flushed)
    int pass;                  // PASS_HERM / PASS_SYMC (ignored by the real-form roles)
    int L;
    int64_t u_begin, n_units;
    int zero;
};

__host__ __device__ __forceinline__ int64_t apply_num_units(int nt, int L)
{
    int64_t bf = nt / L, r = nt % L;
    return (int64_t)L * bf * (bf + 1) / 2 + r * (bf + 1);
}
// first unit of tile row I (units are ordered by tile row, then by segment): the units of tile rows [I0, I1) are
// the contiguous range [apply_first_unit(I0), apply_first_unit(I1))
__host__ __device__ __forceinline__ int64_t apply_first_unit(int I, int L)
{
    int64_t b = I / L, r = I % L;
    return (int64_t)L * b * (b + 1) / 2 + r * (b + 1);
}
// unit u -> (I, J0, J1): rows I in [bL, (b+1)L) have b+1 units each.
__device__ __forceinline__ void apply_decode_unit(int64_t u, int L, int &I, int &J0, int &J1)
{
    int64_t b = (int64_t)((sqrt(1.0 + 8.0 * (double)u / (double)L) - 1.0) * 0.5);
    while ((int64_t)L * b * (b + 1) / 2 > u) --b;
    while ((int64_t)L * (b + 1) * (b + 2) / 2 <= u) ++b;
    int64_t rem = u - (int64_t)L * b * (b + 1) / 2;
    int r = (int)(rem / (b + 1)), seg = (int)(rem % (b + 1));
    I = (int)(b * L + r);
    J0 = seg * L;
    J1 = min(J0 + L, I + 1);
}

}  // namespace bse
