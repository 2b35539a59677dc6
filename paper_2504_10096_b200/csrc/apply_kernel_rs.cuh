// Role-split form of apply_tiles_kernel<ES, 1> (2 .. 4 columns of X, four real products per complex product, N dimension
// n = 2 c + part): the same DMMA count per tile, but -- as in apply_tiles_3m_kernel / apply_tiles_real_kernel -- consumer
// warps 0..3 do P1 only (Y_I += T x_J; warp (rh, ch) owns tile rows 32 rh .. +31 x tile columns 32 ch .. +31, four
// accumulators kept for the unit) and warps 4..7 do P2 only (Y_J += T^H x_I; warp r owns tile columns 16 r .. +15, the
// x_I fragments in 64 registers, eight accumulator chains per tile).  64 DMMAs per tile per warp, no spills, every
// fragment read from shared memory once per role.  Under the power cap of a sustained run the SM clock drops and the
// kernel becomes DMMA-issue bound, so the utilisation of the DMMA sub-pipe (not HBM) sets the k = 4 number: this form
// keeps the pipe busier than the all-roles-per-warp form.  Sign tables as in apply_kernel.cuh.
#pragma once
#include "apply_kernel.cuh"

namespace bse {

template <int ES>
__global__ void __launch_bounds__(APPLY_THREADS, 1) apply_tiles_rs_kernel(const ApplyParams p)
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
    // B fragments: lane supplies B[kk = t][n = g], n = 2 c + part; accumulators c[0], c[1] = (re, im) of column t
    const int col = g >> 1, part = g & 1;
    const bool colok = col < p.kc;
    const double2 *xcol = p.X + (int64_t)(colok ? col : 0) * p.ldx;
    const int kc = p.kc;
    double ca1, cb1, ca2, cb2;                                // apply_kernel.cuh: Ba pairs with Re(T), Bb with Im(T)
    if (p.pass == PASS_HERM) {
        ca1 = 1.0; cb1 = part ? 1.0 : -1.0;
        ca2 = 1.0; cb2 = part ? -1.0 : 1.0;
    } else {
        ca1 = part ? -1.0 : 1.0; cb1 = 1.0;
        ca2 = ca1; cb2 = 1.0;
    }
    ca1 *= p.sign; cb1 *= p.sign; ca2 *= p.sign; cb2 *= p.sign;
    int st = 0;
    uint32_t ph = 0;

    if (warp < 4) {
        // ------------------------------ P1 warps ------------------------------
        const int rh = warp & 1, ch = warp >> 1;
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
            double C1[4][2];
#pragma unroll
            for (int ib = 0; ib < 4; ++ib) C1[ib][0] = C1[ib][1] = 0.0;
            for (int J = J0; J < J1; ++J) {
                double Ba[4][2], Bb[4][2];
#pragma unroll
                for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        Ba[pc][s] = (part ? xjn[pc][s].y : xjn[pc][s].x) * ca1;
                        Bb[pc][s] = (part ? xjn[pc][s].x : xjn[pc][s].y) * cb1;
                    }
                if (J + 1 < J1) load_xj(J + 1, xjn);
                mbar_wait(&full[st], ph);
                const char *tp = tile_s + st * TBY + (4 * ch) * 8 * PBY + (4 * rh) * PBY;
#pragma unroll
                for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        double2 a[4];
#pragma unroll
                        for (int ib = 0; ib < 4; ++ib) a[ib] = load_frag<ES>(tp + (pc * 8 + ib) * PBY + offP1 + s * S1);
#pragma unroll
                        for (int ib = 0; ib < 4; ++ib) dmma(C1[ib], a[ib].x, Ba[pc][s]);      // four independent chains,
#pragma unroll
                        for (int ib = 0; ib < 4; ++ib) dmma(C1[ib], a[ib].y, Bb[pc][s]);      // dependent DMMAs 4 apart
                    }
                int live = 0;
#pragma unroll
                for (int ib = 0; ib < 4; ++ib) live |= __double2hiint(C1[ib][0]);
                __syncwarp();
                if (lane == 0)
                    mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(&empty[st]) + (live & p.zero)));
                if (++st == NST) { st = 0; ph ^= 1; }
            }
            if (t < kc) {
#pragma unroll
                for (int ib = 0; ib < 4; ++ib) {
                    int64_t row = (int64_t)I * TB + (4 * rh + ib) * 8 + g;
                    if (row < p.N) {
                        double *y = p.Y + 2 * (row + (int64_t)t * p.ldy);
                        red_add(y, C1[ib][0]);
                        red_add(y + 1, C1[ib][1]);
                    }
                }
            }
        }
        return;
    }

    // ------------------------------ P2 warps ------------------------------
    const int r = warp - 4;
    for (int64_t u = p.u_begin + blockIdx.x; u < p.n_units; u += gridDim.x) {
        int I, J0, J1;
        apply_decode_unit(u, p.L, I, J0, J1);
        double xA[8][2], xB[8][2];                            // BaI, BbI: rows 8 ib + 4 s + t of x_I
#pragma unroll
        for (int ib = 0; ib < 8; ++ib)
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                int64_t row = (int64_t)I * TB + ib * 8 + s * 4 + t;
                double2 x = (colok && row < p.N) ? __ldg(xcol + row) : make_double2(0.0, 0.0);
                xA[ib][s] = (part ? x.y : x.x) * ca2;
                xB[ib][s] = (part ? x.x : x.y) * cb2;
            }
        for (int J = J0; J < J1; ++J) {
            mbar_wait(&full[st], ph);
            if (I != J) {
                double ZA[2][2][2], ZB[2][2][2];             // [pc][ib parity][re / im]: eight independent chains
#pragma unroll
                for (int pc = 0; pc < 2; ++pc)
#pragma unroll
                    for (int q = 0; q < 2; ++q) ZA[pc][q][0] = ZA[pc][q][1] = ZB[pc][q][0] = ZB[pc][q][1] = 0.0;
                const char *tp = tile_s + st * TBY + (2 * r) * 8 * PBY;
#pragma unroll
                for (int ib = 0; ib < 8; ib += 2) {
                    double2 b[2][2][2];
#pragma unroll
                    for (int q = 0; q < 2; ++q)
#pragma unroll
                        for (int s = 0; s < 2; ++s)
#pragma unroll
                            for (int pc = 0; pc < 2; ++pc)
                                b[q][s][pc] = load_frag<ES>(tp + (pc * 8 + ib + q) * PBY + offP2 + s * S2);
#pragma unroll
                    for (int s = 0; s < 2; ++s)
#pragma unroll
                        for (int q = 0; q < 2; ++q)
#pragma unroll
                            for (int pc = 0; pc < 2; ++pc) {
                                dmma(ZA[pc][q], b[q][s][pc].x, xA[ib + q][s]);
                                dmma(ZB[pc][q], b[q][s][pc].y, xB[ib + q][s]);
                            }
                }
                double z[2][2];
                int live = 0;
#pragma unroll
                for (int pc = 0; pc < 2; ++pc)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        z[pc][e] = (ZA[pc][0][e] + ZA[pc][1][e]) + (ZB[pc][0][e] + ZB[pc][1][e]);
                        live |= __double2hiint(z[pc][e]);
                    }
                __syncwarp();
                if (lane == 0)
                    mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(&empty[st]) + (live & p.zero)));
                if (t < kc) {
#pragma unroll
                    for (int pc = 0; pc < 2; ++pc) {
                        int64_t row = (int64_t)J * TB + (2 * r + pc) * 8 + g;
                        if (row < p.N) {
                            double *y = p.Y + 2 * (row + (int64_t)t * p.ldy);
                            red_add(y, z[pc][0]);
                            red_add(y + 1, z[pc][1]);
                        }
                    }
                }
            } else {
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[st]);       // diagonal tile: stored in full, P1 only
            }
            if (++st == NST) { st = 0; ph ^= 1; }
        }
    }
}

}  // namespace bse
