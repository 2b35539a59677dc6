// Structured block-matvec over the packed triangular tile store.
//
// One pass computes, for up to 4 columns of X,
//     HERM :  Y += s * R X            (R Hermitian, lower triangle stored)
//     SYMC :  Y += s * C conj(X)      (C complex symmetric, lower triangle stored)
// Every stored tile T = T_IJ (I >= J) is brought from HBM exactly once by ONE TMA bulk copy
// (cp.async.bulk -> UBLKCP, 64 KB, contiguous) into a 3-stage shared-memory ring and used twice from there:
//     P1:  Y_I += T   x_J            (HERM)      Y_I += T   conj(x_J)   (SYMC)
//     P2:  Y_J += T^H x_I            (HERM)      Y_J += T^T conj(x_I)   (SYMC)       (skipped when I == J)
// Both products run on the FP64 tensor cores (mma.sync m8n8k4 -> DMMA.8x8x4) in real arithmetic:
// with N-dimension n = 2 c + part (c = column of X, part = re/im),
//     [Yr|Yi] += Tr * Ba + Ti * Bb,   Ba, Bb = signed re/im selections of X (table below and in DESIGN.md).
//
// Work decomposition: a unit is a run of up to L consecutive tiles of one tile row I.  A CTA
// (8 consumer warps + 1 producer warp, persistent, one per SM) walks its units; consumer warp w
// owns tile columns 8w .. 8w+7 of every tile, i.e. for P1 a slice of the contraction (partial Y_I for
// all 64 rows, accumulated in registers over the whole unit) and for P2 eight output rows of Y_J
// (contraction over all 64 i, with the x_I fragments held in registers for the whole unit).
// The X fragments are read by the consumers straight from global memory (X is L2-resident: 16 N k bytes),
// x_J one tile ahead of its use.  Partial results are added to Y with red.global.add.f64 (Y must be zero or
// hold the running sum).
//
// Round-1 note: an earlier version staged the X panels through shared memory with small (1 KB) bulk copies on
// their own mbarrier; with 4 columns and one-tile units it returned stale fragments about once per launch on
// B200.  Tests at N >= 4096 (many units per CTA) cover this path now.
#pragma once
#include "bse_common.cuh"

namespace bse {

constexpr int APPLY_STAGES = 3;                          // ring depth for 64 KB (complex128) tiles; 6 for 32 KB (complex64)
constexpr int APPLY_CONSUMERS = 8;                       // consumer warps
constexpr int APPLY_THREADS = (APPLY_CONSUMERS + 1) * 32;
constexpr int APPLY_SMEM = APPLY_STAGES * TILE_BYTES + 128;

enum { PASS_HERM = 0, PASS_SYMC = 1 };

struct ApplyParams {
    const char *tiles;
    const double2 *X;
    int64_t ldx;
    double *Y;          // complex128 viewed as doubles
    int64_t ldy;
    int64_t N;
    int nt;             // tile rows
    int kc;             // columns in this pass (1..4; 5..8 for the NPC = 2 kernel)
    int pass;           // PASS_HERM / PASS_SYMC
    double sign;        // s
    int L;              // unit length in tiles
    int64_t u_begin;    // first unit of this handle's tile rows (0 unless the handle is a shard)
    int64_t n_units;    // one past the last unit
    int zero;           // always 0; a runtime value the assembler cannot fold (see the stage release below)
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

// ES = bytes per stored complex entry (bse_common.cuh): 16 -> LDS.128 fragments, 8 -> LDS.64 + conversion to FP64.
// NPC = patch columns per consumer warp.  NPC = 1: up to 4 columns of X, warp w owns tile columns 8w .. 8w+7.
// NPC = 2 (5 .. 8 columns of X in ONE pass over the operand): warp w owns tile columns 16 (w >> 1) .. +15 and the
// column half nh = w & 1 (columns 4 nh .. 4 nh + 3 of X): the same accumulators and x_I fragments as NPC = 1, twice
// the DMMAs per tile, each stored tile still read from HBM once.
template <int ES, int NPC>
__global__ void __launch_bounds__(APPLY_THREADS, 1) apply_tiles_kernel(const ApplyParams p)
{
    constexpr int TBY = TB * TB * ES;                    // tile bytes
    constexpr int PBY = 64 * ES;                         // 8 x 8 patch bytes
    constexpr int NST = APPLY_STAGES * 16 / ES;          // stages: the ring always fills the same 192 KB
    constexpr int S1 = 16 * ES, S2 = 32 * ES;            // second k-step of the P1 / P2 fragment (16 / 32 slots on)
    extern __shared__ __align__(1024) char smem[];
    char *tile_s = smem;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + NST * TBY);
    uint64_t *full = bars, *empty = bars + NST;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < NST; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], APPLY_CONSUMERS); }
        fence_barrier_init();
    }
    __syncthreads();

    if (warp == APPLY_CONSUMERS) {
        // ------------------------------ producer warp (one elected lane) ------------------------------
        if (lane == 0) {
            int st = 0;
            uint32_t ph = 0;
            const uint64_t pol = l2_policy_evict_first();     // the tile stream is read exactly once
            for (int64_t u = p.u_begin + blockIdx.x; u < p.n_units; u += gridDim.x) {
                int I, J0, J1;
                apply_decode_unit(u, p.L, I, J0, J1);
                const char *src = p.tiles + tile_index(I, J0) * (int64_t)TBY;
                for (int J = J0; J < J1; ++J, src += TBY) {
                    mbar_wait(&empty[st], ph ^ 1);
                    mbar_expect_tx(&full[st], (uint32_t)TBY);
                    bulk_g2s_hint(tile_s + st * TBY, src, TBY, &full[st], pol);
                    if (++st == NST) { st = 0; ph ^= 1; }
                }
            }
        }
        return;
    }

    // ------------------------------------ consumer warps ------------------------------------------
    const int nh = (NPC == 2) ? (warp & 1) : 0;           // which half of the (up to) 8 columns
    const int w0 = (NPC == 2) ? (warp >> 1) * 2 : warp;   // first patch column of this warp
    const int g = lane >> 2, t = lane & 3;
    const int g2 = (g >> 2) & 1, g1 = (g >> 1) & 1, g0 = g & 1, t1 = (t >> 1) & 1, t0 = t & 1;
    // fragment byte offsets inside a patch (see patch_slot): P1 reads (a = g, b = 4 s + t), P2 reads (a = 4 s + t, b = g)
    const int offP1 = (((g2 << 2) | g1) * 8 + ((g0 << 2) | (t0 << 1) | (g1 ^ t1))) * ES;   // + s * S1
    const int offP2 = (((g2 << 1) | t1) * 8 + ((t0 << 2) | (g0 << 1) | (t1 ^ g1))) * ES;   // + s * S2
    // B fragments: lane supplies B[kk = t][n = g], n = 2 c + part
    const int col = (g >> 1) + 4 * nh, part = g & 1;
    const int tc = t + 4 * nh;                            // column of X / Y this lane's accumulator entries belong to
    const bool colok = col < p.kc;
    // Ba pairs with Re(T), Bb with Im(T); value = coef * (re or im of x):
    //   HERM P1 (T x):         Ba = [xr,  xi]   Bb = [-xi,  xr]
    //   HERM P2 (T^H x):       Ba = [xr,  xi]   Bb = [ xi, -xr]
    //   SYMC P1/P2 (T conj x): Ba = [xr, -xi]   Bb = [ xi,  xr]
    double ca1, cb1, ca2, cb2;
    if (p.pass == PASS_HERM) {
        ca1 = 1.0; cb1 = part ? 1.0 : -1.0;
        ca2 = 1.0; cb2 = part ? -1.0 : 1.0;
    } else {
        ca1 = part ? -1.0 : 1.0; cb1 = 1.0;
        ca2 = ca1; cb2 = 1.0;
    }
    ca1 *= p.sign; cb1 *= p.sign; ca2 *= p.sign; cb2 *= p.sign;
    const double2 *xcol = p.X + (int64_t)(colok ? col : 0) * p.ldx;
    const int kc = p.kc;

    // x rows of tile-row K needed by this lane for P1 (rows 8 (w0 + pc) + 4s + t); zero outside the matrix / columns
    auto load_xj = [&](int K, double2 (&x)[NPC][2]) {
#pragma unroll
        for (int pc = 0; pc < NPC; ++pc)
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                int64_t row = (int64_t)K * TB + (w0 + pc) * 8 + s * 4 + t;
                x[pc][s] = (colok && row < p.N) ? __ldg(xcol + row) : make_double2(0.0, 0.0);
            }
    };

    int st = 0;
    uint32_t ph = 0;
    for (int64_t u = p.u_begin + blockIdx.x; u < p.n_units; u += gridDim.x) {
        int I, J0, J1;
        apply_decode_unit(u, p.L, I, J0, J1);

        double2 xjn[NPC][2];
        load_xj(J0, xjn);
        // x_I fragments for P2 (rows 8 ib + 4 s + t), kept in registers for the whole unit
        double BaI[8][2], BbI[8][2];
        {
            double2 xi[8][2];
#pragma unroll
            for (int ib = 0; ib < 8; ++ib)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    int64_t row = (int64_t)I * TB + ib * 8 + s * 4 + t;
                    xi[ib][s] = (colok && row < p.N) ? __ldg(xcol + row) : make_double2(0.0, 0.0);
                }
#pragma unroll
            for (int ib = 0; ib < 8; ++ib)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    BaI[ib][s] = (part ? xi[ib][s].y : xi[ib][s].x) * ca2;
                    BbI[ib][s] = (part ? xi[ib][s].x : xi[ib][s].y) * cb2;
                }
        }
        double C1[8][2];
#pragma unroll
        for (int ib = 0; ib < 8; ++ib) C1[ib][0] = C1[ib][1] = 0.0;

        for (int J = J0; J < J1; ++J) {
            double BaJ[NPC][2], BbJ[NPC][2];
#pragma unroll
            for (int pc = 0; pc < NPC; ++pc)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    BaJ[pc][s] = (part ? xjn[pc][s].y : xjn[pc][s].x) * ca1;
                    BbJ[pc][s] = (part ? xjn[pc][s].x : xjn[pc][s].y) * cb1;
                }
            if (J + 1 < J1) load_xj(J + 1, xjn);            // prefetch the next tile's x_J fragments

            mbar_wait(&full[st], ph);
            int live = 0;
            double yr[NPC], yi[NPC];
#pragma unroll
            for (int pc = 0; pc < NPC; ++pc) {
                const char *tp = tile_s + st * TBY + (w0 + pc) * 8 * PBY;
                if (I != J) {
                    double C2[4][2];
#pragma unroll
                    for (int q = 0; q < 4; ++q) C2[q][0] = C2[q][1] = 0.0;
                    // two patches at a time, four independent accumulator chains interleaved: dependent DMMAs are 4 apart
#pragma unroll
                    for (int ib = 0; ib < 8; ib += 2) {
                        const char *pp = tp + ib * PBY, *pq = pp + PBY;
                        double2 a0 = load_frag<ES>(pp + offP1);
                        double2 c0 = load_frag<ES>(pq + offP1);
                        double2 b0 = load_frag<ES>(pp + offP2);
                        double2 d0 = load_frag<ES>(pq + offP2);
                        double2 a1 = load_frag<ES>(pp + offP1 + S1);
                        double2 c1 = load_frag<ES>(pq + offP1 + S1);
                        double2 b1 = load_frag<ES>(pp + offP2 + S2);
                        double2 d1 = load_frag<ES>(pq + offP2 + S2);
                        const int q = ib & 2;
                        dmma(C1[ib], a0.x, BaJ[pc][0]);
                        dmma(C1[ib + 1], c0.x, BaJ[pc][0]);
                        dmma(C2[q], b0.x, BaI[ib][0]);
                        dmma(C2[q + 1], d0.x, BaI[ib + 1][0]);
                        dmma(C1[ib], a0.y, BbJ[pc][0]);
                        dmma(C1[ib + 1], c0.y, BbJ[pc][0]);
                        dmma(C2[q], b0.y, BbI[ib][0]);
                        dmma(C2[q + 1], d0.y, BbI[ib + 1][0]);
                        dmma(C1[ib], a1.x, BaJ[pc][1]);
                        dmma(C1[ib + 1], c1.x, BaJ[pc][1]);
                        dmma(C2[q], b1.x, BaI[ib][1]);
                        dmma(C2[q + 1], d1.x, BaI[ib + 1][1]);
                        dmma(C1[ib], a1.y, BbJ[pc][1]);
                        dmma(C1[ib + 1], c1.y, BbJ[pc][1]);
                        dmma(C2[q], b1.y, BbI[ib][1]);
                        dmma(C2[q + 1], d1.y, BbI[ib + 1][1]);
                    }
                    yr[pc] = (C2[0][0] + C2[1][0]) + (C2[2][0] + C2[3][0]);
                    yi[pc] = (C2[0][1] + C2[1][1]) + (C2[2][1] + C2[3][1]);
                    live |= __double2hiint(yr[pc]) | __double2hiint(yi[pc]);
                } else {
#pragma unroll
                    for (int ib = 0; ib < 8; ib += 4) {     // diagonal tile: P1 only, four chains interleaved
                        double2 a0[4], a1[4];
#pragma unroll
                        for (int r = 0; r < 4; ++r) {
                            a0[r] = load_frag<ES>(tp + (ib + r) * PBY + offP1);
                            a1[r] = load_frag<ES>(tp + (ib + r) * PBY + offP1 + S1);
                        }
#pragma unroll
                        for (int r = 0; r < 4; ++r) dmma(C1[ib + r], a0[r].x, BaJ[pc][0]);
#pragma unroll
                        for (int r = 0; r < 4; ++r) dmma(C1[ib + r], a0[r].y, BbJ[pc][0]);
#pragma unroll
                        for (int r = 0; r < 4; ++r) dmma(C1[ib + r], a1[r].x, BaJ[pc][1]);
#pragma unroll
                        for (int r = 0; r < 4; ++r) dmma(C1[ib + r], a1[r].y, BbJ[pc][1]);
                    }
                }
            }
            // The release must not overtake the ld.shared that feed the DMMAs above: an mbarrier arrive only orders
            // the ISSUE of earlier loads, and on B200 queued loads of a slow warp were observed to execute after the
            // producer's next bulk copy had landed (stale fragments about once per launch).  The barrier address is
            // therefore made to depend on every accumulator (live & p.zero == 0, but not foldable): all DMMAs,
            // hence all loads, have completed before the arrive can issue.  (yr, yi are sums of every C2 word.)
#pragma unroll
            for (int ib = 0; ib < 8; ++ib) live |= __double2hiint(C1[ib][0]);
            __syncwarp();
            if (lane == 0)
                mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(&empty[st]) + (live & p.zero)));
            if (I != J) {                                   // flush Y_J rows 8 (w0 + pc) + g, column tc
#pragma unroll
                for (int pc = 0; pc < NPC; ++pc) {
                    int64_t row = (int64_t)J * TB + (w0 + pc) * 8 + g;
                    if (tc < kc && row < p.N) {
                        double *y = p.Y + 2 * (row + (int64_t)tc * p.ldy);
                        red_add(y, yr[pc]);
                        red_add(y + 1, yi[pc]);
                    }
                }
            }
            if (++st == NST) { st = 0; ph ^= 1; }
        }
        // flush this warp's partial Y_I (all 64 rows, column tc)
        if (tc < kc) {
#pragma unroll
            for (int ib = 0; ib < 8; ++ib) {
                int64_t row = (int64_t)I * TB + ib * 8 + g;
                if (row < p.N) {
                    double *y = p.Y + 2 * (row + (int64_t)tc * p.ldy);
                    red_add(y, C1[ib][0]);
                    red_add(y + 1, C1[ib][1]);
                }
            }
        }
    }
}

}  // namespace bse
