// Single-column variant of apply_tiles_kernel (k = 1: the paper's own iteration generates its vectors "one by one",
// PAPER.md:71, and the Lanczos-with-quadrature solver is a single-vector recurrence).
//
// With one column the 8-wide N dimension of a DMMA is 3/4 empty, so the tensor-core kernel pays the FP64 work (and
// the power) of k = 4.  Here the same tile ring and the same two conflict-free fragment reads feed plain complex
// FMAs instead: 128 DFMA per tile per warp, about a fifth of the FP64 pipe at the HBM rate, so the kernel is bound by
// the tile stream alone.  Lane (g, t) of consumer warp w handles, per 8 x 8 patch (ib, jb = w):
//     P1:  a = T[8 ib + g][8 w + 4 s + t]   acc1[ib] += a * xj[s]          (xj = x_J or conj(x_J))
//     P2:  b = T[8 ib + 4 s + t][8 w + g]   acc2     += b * conj(x_I[8 ib + 4 s + t])
// acc1 is summed over the four t-lanes once per unit, acc2 once per tile (warp shuffles), then added to Y with
// red.global.add.f64.  HERM: Y_J += conj(acc2) (= T^H x_I);  SYMC: Y_J += acc2 (= T^T conj(x_I)).
#pragma once
#include "apply_kernel.cuh"

namespace bse {

__device__ __forceinline__ void cfma(double2 &acc, const double2 a, const double2 x)
{
    acc.x = fma(a.x, x.x, acc.x); acc.x = fma(-a.y, x.y, acc.x);
    acc.y = fma(a.x, x.y, acc.y); acc.y = fma(a.y, x.x, acc.y);
}

template <int ES>
__global__ void __launch_bounds__(APPLY_THREADS, 1) apply_tiles_k1_kernel(const ApplyParams p)
{
    constexpr int TBY = TB * TB * ES, PBY = 64 * ES, NST = APPLY_STAGES * 16 / ES, S1 = 16 * ES, S2 = 32 * ES;
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
        if (lane == 0) {                                   // producer: identical to the tensor-core kernel
            int st = 0;
            uint32_t ph = 0;
            const uint64_t pol = l2_policy_evict_first();
            for (int64_t u = blockIdx.x; u < p.n_units; u += gridDim.x) {
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

    const int w = warp;
    const int g = lane >> 2, t = lane & 3;
    const int g2 = (g >> 2) & 1, g1 = (g >> 1) & 1, g0 = g & 1, t1 = (t >> 1) & 1, t0 = t & 1;
    const int offP1 = (((g2 << 2) | g1) * 8 + ((g0 << 2) | (t0 << 1) | (g1 ^ t1))) * ES;   // + s * S1
    const int offP2 = (((g2 << 1) | t1) * 8 + ((t0 << 2) | (g0 << 1) | (t1 ^ g1))) * ES;   // + s * S2
    const bool herm = (p.pass == PASS_HERM);
    const double sgn = p.sign;
    const double2 zero2 = make_double2(0.0, 0.0);
    const double2 *x = p.X;

    // x_J rows 8w + 4s + t, as the P1 operand: x_J (HERM) or conj(x_J) (SYMC), times the pass sign
    auto load_xj = [&](int K, double2 (&v)[2]) {
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            int64_t row = (int64_t)K * TB + w * 8 + s * 4 + t;
            double2 a = row < p.N ? __ldg(x + row) : zero2;
            v[s] = make_double2(sgn * a.x, herm ? sgn * a.y : -sgn * a.y);
        }
    };

    int st = 0;
    uint32_t ph = 0;
    for (int64_t u = blockIdx.x; u < p.n_units; u += gridDim.x) {
        int I, J0, J1;
        apply_decode_unit(u, p.L, I, J0, J1);

        double2 xjn[2];
        load_xj(J0, xjn);
        // conj(x_I) for rows 8 ib + 4 s + t, times the pass sign: the P2 operand, in registers for the whole unit
        double2 xi[8][2];
#pragma unroll
        for (int ib = 0; ib < 8; ++ib)
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                int64_t row = (int64_t)I * TB + ib * 8 + s * 4 + t;
                double2 a = row < p.N ? __ldg(x + row) : zero2;
                xi[ib][s] = make_double2(sgn * a.x, -sgn * a.y);
            }
        double2 acc1[8];
#pragma unroll
        for (int ib = 0; ib < 8; ++ib) acc1[ib] = zero2;

        for (int J = J0; J < J1; ++J) {
            const double2 xj0 = xjn[0], xj1 = xjn[1];
            if (J + 1 < J1) load_xj(J + 1, xjn);            // prefetch the next tile's x_J rows

            mbar_wait(&full[st], ph);
            const char *tp = tile_s + st * TBY + w * 8 * PBY;
            int live = 0;
            if (I != J) {
                double2 acc2[2] = {zero2, zero2};
#pragma unroll
                for (int ib = 0; ib < 8; ++ib) {
                    const char *pp = tp + ib * PBY;
                    const double2 a0 = load_frag<ES>(pp + offP1);
                    const double2 a1 = load_frag<ES>(pp + offP1 + S1);
                    const double2 b0 = load_frag<ES>(pp + offP2);
                    const double2 b1 = load_frag<ES>(pp + offP2 + S2);
                    cfma(acc1[ib], a0, xj0);
                    cfma(acc2[0], b0, xi[ib][0]);
                    cfma(acc1[ib], a1, xj1);
                    cfma(acc2[1], b1, xi[ib][1]);
                }
                double yr = acc2[0].x + acc2[1].x, yi = acc2[0].y + acc2[1].y;
                // dependent release (see apply_kernel.cuh): values computed from every load of this stage
#pragma unroll
                for (int ib = 0; ib < 8; ++ib) live |= __double2hiint(acc1[ib].x);
                live |= __double2hiint(yr) | __double2hiint(yi);
                __syncwarp();
                if (lane == 0)
                    mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(&empty[st]) + (live & p.zero)));
                // sum over the four t-lanes, then Y_J[8w + g] += conj(acc2) (HERM) or acc2 (SYMC)
                yr += __shfl_xor_sync(0xffffffffu, yr, 1); yi += __shfl_xor_sync(0xffffffffu, yi, 1);
                yr += __shfl_xor_sync(0xffffffffu, yr, 2); yi += __shfl_xor_sync(0xffffffffu, yi, 2);
                const int64_t row = (int64_t)J * TB + w * 8 + g;
                if (t == 0 && row < p.N) {
                    double *y = p.Y + 2 * row;
                    red_add(y, yr);
                    red_add(y + 1, herm ? -yi : yi);
                }
            } else {
#pragma unroll
                for (int ib = 0; ib < 8; ++ib) {
                    const char *pp = tp + ib * PBY;
                    const double2 a0 = load_frag<ES>(pp + offP1);
                    const double2 a1 = load_frag<ES>(pp + offP1 + S1);
                    cfma(acc1[ib], a0, xj0);
                    cfma(acc1[ib], a1, xj1);
                }
#pragma unroll
                for (int ib = 0; ib < 8; ++ib) live |= __double2hiint(acc1[ib].x);
                __syncwarp();
                if (lane == 0)
                    mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(&empty[st]) + (live & p.zero)));
            }
            if (++st == NST) { st = 0; ph ^= 1; }
        }
        // flush this warp's partial Y_I: sum over the four t-lanes, lane t == 0 adds rows 8 ib + g
#pragma unroll
        for (int ib = 0; ib < 8; ++ib) {
            double yr = acc1[ib].x, yi = acc1[ib].y;
            yr += __shfl_xor_sync(0xffffffffu, yr, 1); yi += __shfl_xor_sync(0xffffffffu, yi, 1);
            yr += __shfl_xor_sync(0xffffffffu, yr, 2); yi += __shfl_xor_sync(0xffffffffu, yi, 2);
            const int64_t row = (int64_t)I * TB + ib * 8 + g;
            if (t == 0 && row < p.N) {
                double *y = p.Y + 2 * row;
                red_add(y, yr);
                red_add(y + 1, yi);
            }
        }
    }
}

}  // namespace bse
