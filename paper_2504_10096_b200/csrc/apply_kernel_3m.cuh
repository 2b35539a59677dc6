// 5 .. 8 columns of X in ONE pass over the operand, with three real products per complex product
// (same tile ring, same producer and same stage release as apply_tiles_kernel).
//
// With eight columns the 8-wide N dimension of a DMMA can hold the eight columns themselves (n = column) instead
// of four columns x {re, im}.  A complex product T x then needs the real products of Tr, Ti with xr, xi; the
// classical three-product form (Karatsuba / "3M") takes
//     Q1 = Tr xr,   Q2 = Ti xi,   Q3 = (Tr + Ti) (u xr + v xi)
// and recovers re and im as signed sums of Q1, Q2, Q3 (table below): 3 DMMAs per 8 x 8 x 4 real block for eight
// columns, where the four-product form of apply_tiles_kernel<ES, 2> issues 4.  Tr + Ti costs one DADD per loaded
// fragment entry (1/8 of a DMMA on the FP64 pipe).  The products are accumulated separately over a whole unit and
// combined once when they are flushed.
//
//     pass / product              xs (pairs with Tr + Ti)     re          im
//     HERM P1:  T x               xr + xi                     Q1 - Q2     Q3 - Q1 - Q2
//     HERM P2:  T^H x             xi - xr                     Q1 + Q2     Q3 + Q1 - Q2
//     SYMC P1:  T conj(x)         xr - xi                     Q1 + Q2     Q3 - Q1 + Q2
//     SYMC P2:  T^T conj(x)       xi - xr                     Q1 + Q2    -Q3 - Q1 + Q2
//
// Rounding: |error| <= c eps (|Tr| + |Ti|)(|xr| + |xi|) per term, i.e. the same normwise bound as the four-product
// form up to a factor 2 (the imaginary part is no longer componentwise accurate when it is tiny against the real
// part); the parity tolerance of the apply is normwise (reading S11).
//
// Warp roles (three accumulator sets do not fit one warp's 168 registers next to the x_I fragments):
//   warps 0..3  (P1 warps):  Y_I += T x_J.  Warp (rh = w & 1, ch = w >> 1) owns tile rows 32 rh .. +31 and tile
//                columns 32 ch .. +31: 16 patches, 12 accumulator chains kept for the whole unit.
//   warps 4..7  (P2 warps):  Y_J += T^H x_I.  Warp r = w - 4 owns tile columns 16 r .. +15 (all 64 rows):
//                16 patches, the x_I fragments (64 registers) kept for the whole unit, 6 chains per tile.
//   warp 8      producer (one elected lane), as in apply_tiles_kernel.
// One P1 and one P2 warp share each scheduler; both issue 96 DMMAs per tile.  Every fragment is read from shared
// memory by exactly one warp per role, RED counts per tile and per unit equal those of apply_tiles_kernel<ES, 2>.
#pragma once
#include "apply_kernel.cuh"

namespace bse {

template <int ES>
__global__ void __launch_bounds__(APPLY_THREADS, 1) apply_tiles_3m_kernel(const ApplyParams p)
{
    constexpr int TBY = TB * TB * ES;
    constexpr int PBY = 64 * ES;
    constexpr int NST = APPLY_STAGES * 16 / ES;
    constexpr int S1 = 16 * ES, S2 = 32 * ES;
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
        if (lane == 0) {                                   // producer: identical to apply_tiles_kernel
            int st = 0;
            uint32_t ph = 0;
            const uint64_t pol = l2_policy_evict_first();
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

    const int g = lane >> 2, t = lane & 3;
    const int g2 = (g >> 2) & 1, g1 = (g >> 1) & 1, g0 = g & 1, t1 = (t >> 1) & 1, t0 = t & 1;
    const int offP1 = (((g2 << 2) | g1) * 8 + ((g0 << 2) | (t0 << 1) | (g1 ^ t1))) * ES;   // (a = g, b = 4 s + t)
    const int offP2 = (((g2 << 1) | t1) * 8 + ((t0 << 2) | (g0 << 1) | (t1 ^ g1))) * ES;   // (a = 4 s + t, b = g)
    // B fragments: lane supplies B[kk = t][n = g], n = column of X; accumulators c[e] = C[g][2 t + e]
    const bool colok = g < p.kc;
    const double2 *xcol = p.X + (int64_t)(colok ? g : 0) * p.ldx;
    const bool herm = p.pass == PASS_HERM;
    const int kc = p.kc;
    int st = 0;
    uint32_t ph = 0;

    if (warp < 4) {
        // ------------------------------ P1 warps:  Y_I += T x_J  (or T conj(x_J)) ------------------------------
        const int rh = warp & 1, ch = warp >> 1;
        const double v = herm ? 1.0 : -1.0;                  // xs = xr + v xi
        // flush coefficients: re = s (Q1 + cr2 Q2), im = s (Q3 - Q1 + ci2 Q2)
        const double cr2 = herm ? -1.0 : 1.0, ci2 = herm ? -1.0 : 1.0;
        // x rows of tile-row K needed by this lane: 8 (4 ch + pc) + 4 s + t, column g
        auto load_xj = [&](int K, double2 (&x)[4][2]) {
#pragma unroll
            for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    int64_t row = (int64_t)K * TB + (4 * ch + pc) * 8 + s * 4 + t;
                    x[pc][s] = (colok && row < p.N) ? __ldg(xcol + row) : make_double2(0.0, 0.0);
                }
        };
        for (int64_t u = p.u_begin + blockIdx.x; u < p.n_units; u += gridDim.x) {
            int I, J0, J1;
            apply_decode_unit(u, p.L, I, J0, J1);
            double2 xjn[4][2];
            load_xj(J0, xjn);
            double Q1[4][2], Q2[4][2], Q3[4][2];
#pragma unroll
            for (int ib = 0; ib < 4; ++ib) Q1[ib][0] = Q1[ib][1] = Q2[ib][0] = Q2[ib][1] = Q3[ib][0] = Q3[ib][1] = 0.0;

            for (int J = J0; J < J1; ++J) {
                double2 xj[4][2];
#pragma unroll
                for (int pc = 0; pc < 4; ++pc) { xj[pc][0] = xjn[pc][0]; xj[pc][1] = xjn[pc][1]; }
                if (J + 1 < J1) load_xj(J + 1, xjn);          // prefetch the next tile's x_J fragments
                mbar_wait(&full[st], ph);
                const char *tp = tile_s + st * TBY + (4 * ch) * 8 * PBY + (4 * rh) * PBY;
#pragma unroll
                for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        const double xr = xj[pc][s].x, xi = xj[pc][s].y;
                        const double xs = fma(v, xi, xr);
                        double2 a[4];
#pragma unroll
                        for (int ib = 0; ib < 4; ++ib) a[ib] = load_frag<ES>(tp + (pc * 8 + ib) * PBY + offP1 + s * S1);
#pragma unroll
                        for (int ib = 0; ib < 4; ++ib) {
                            const double as = a[ib].x + a[ib].y;
                            dmma(Q1[ib], a[ib].x, xr);
                            dmma(Q2[ib], a[ib].y, xi);
                            dmma(Q3[ib], as, xs);
                        }
                    }
                // stage release: data-dependent on every accumulator (see apply_tiles_kernel)
                int live = 0;
#pragma unroll
                for (int ib = 0; ib < 4; ++ib)
                    live |= __double2hiint(Q1[ib][0]) | __double2hiint(Q2[ib][0]) | __double2hiint(Q3[ib][0]);
                __syncwarp();
                if (lane == 0)
                    mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(&empty[st]) + (live & p.zero)));
                if (++st == NST) { st = 0; ph ^= 1; }
            }
            // flush this warp's partial Y_I: rows 8 (4 rh + ib) + g, columns 2 t + e
#pragma unroll
            for (int ib = 0; ib < 4; ++ib) {
                int64_t row = (int64_t)I * TB + (4 * rh + ib) * 8 + g;
                if (row < p.N) {
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int c = 2 * t + e;
                        if (c < kc) {
                            double *y = p.Y + 2 * (row + (int64_t)c * p.ldy);
                            red_add(y, p.sign * fma(cr2, Q2[ib][e], Q1[ib][e]));
                            red_add(y + 1, p.sign * (fma(ci2, Q2[ib][e], Q3[ib][e]) - Q1[ib][e]));
                        }
                    }
                }
            }
        }
        return;
    }

    // ------------------------------ P2 warps:  Y_J += T^H x_I  (or T^T conj(x_I)) ------------------------------
    const int r = warp - 4;                                   // tile columns 16 r .. 16 r + 15
    // xs = xi - xr in both passes; re = s (Q1 + Q2); im = s (c3 Q3 + c1 (Q1 - Q2)):  HERM c3 = 1, c1 = 1; SYMC c3 = -1, c1 = -1
    const double c31 = herm ? p.sign : -p.sign;
    for (int64_t u = p.u_begin + blockIdx.x; u < p.n_units; u += gridDim.x) {
        int I, J0, J1;
        apply_decode_unit(u, p.L, I, J0, J1);
        // x_I fragments (rows 8 ib + 4 s + t, column g), kept in registers for the whole unit
        double2 xI[8][2];
#pragma unroll
        for (int ib = 0; ib < 8; ++ib)
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                int64_t row = (int64_t)I * TB + ib * 8 + s * 4 + t;
                xI[ib][s] = (colok && row < p.N) ? __ldg(xcol + row) : make_double2(0.0, 0.0);
            }
        for (int J = J0; J < J1; ++J) {
            mbar_wait(&full[st], ph);
            int live = 0;
            if (I != J) {
                double Q1[2][2], Q2[2][2], Q3[2][2];
#pragma unroll
                for (int pc = 0; pc < 2; ++pc) Q1[pc][0] = Q1[pc][1] = Q2[pc][0] = Q2[pc][1] = Q3[pc][0] = Q3[pc][1] = 0.0;
                const char *tp = tile_s + st * TBY + (2 * r) * 8 * PBY;
#pragma unroll
                for (int ib = 0; ib < 8; ib += 2) {
                    // two patch rows x two patch columns x two k-steps: 8 fragments in flight, 6 chains, dependent DMMAs 6 apart
                    double2 b[2][2][2];
#pragma unroll
                    for (int q = 0; q < 2; ++q)
#pragma unroll
                        for (int s = 0; s < 2; ++s)
#pragma unroll
                            for (int pc = 0; pc < 2; ++pc)
                                b[q][s][pc] = load_frag<ES>(tp + (pc * 8 + ib + q) * PBY + offP2 + s * S2);
#pragma unroll
                    for (int q = 0; q < 2; ++q)
#pragma unroll
                        for (int s = 0; s < 2; ++s) {
                            const double xr = xI[ib + q][s].x, xi = xI[ib + q][s].y;
                            const double xs = xi - xr;
#pragma unroll
                            for (int pc = 0; pc < 2; ++pc) {
                                const double bs = b[q][s][pc].x + b[q][s][pc].y;
                                dmma(Q1[pc], b[q][s][pc].x, xr);
                                dmma(Q2[pc], b[q][s][pc].y, xi);
                                dmma(Q3[pc], bs, xs);
                            }
                        }
                }
#pragma unroll
                for (int pc = 0; pc < 2; ++pc)
                    live |= __double2hiint(Q1[pc][0]) | __double2hiint(Q2[pc][0]) | __double2hiint(Q3[pc][0]);
                __syncwarp();
                if (lane == 0)
                    mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(&empty[st]) + (live & p.zero)));
                // flush Y_J rows 8 (2 r + pc) + g, columns 2 t + e
#pragma unroll
                for (int pc = 0; pc < 2; ++pc) {
                    int64_t row = (int64_t)J * TB + (2 * r + pc) * 8 + g;
                    if (row < p.N) {
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int c = 2 * t + e;
                            if (c < kc) {
                                double *y = p.Y + 2 * (row + (int64_t)c * p.ldy);
                                red_add(y, p.sign * (Q1[pc][e] + Q2[pc][e]));
                                red_add(y + 1, c31 * (Q3[pc][e] + (Q1[pc][e] - Q2[pc][e])));
                            }
                        }
                    }
                }
            } else {
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[st]);       // diagonal tile: P1 only, nothing was read here
            }
            if (++st == NST) { st = 0; ph ^= 1; }
        }
    }
}

}  // namespace bse
