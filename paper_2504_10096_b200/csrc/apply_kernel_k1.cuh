// Single-column variant of apply_tiles_kernel (k = 1: the paper's own iteration generates its vectors "one by one",
// PAPER.md:71, and the Lanczos-with-quadrature solver is a single-vector recurrence).
//
// With one column the 8-wide N dimension of a DMMA is 3/4 empty, so the tensor-core kernel pays the FP64 work (and
// the power) of k = 4.  Here the same tile ring feeds plain complex FMAs, and -- with no MMA fragment layout to
// honour -- every entry is loaded (and, for the complex64 store, widened) ONCE and used for both products.  Lane
// (g, t) of consumer warp w reads, per 8 x 8 patch (ib, jb = w) and s = 0, 1, the entry
//     a = T[r][c],  r = 8 ib + g,  c = 8 w + 4 s + t          (the conflict-free P1 fragment read)
//     P1:  acc1[ib] += a * xj[s]            (xj = x_J[c] or conj(x_J[c]))          -> Y_I[r], summed over t and s
//     P2:  acc2[s]  += a * conj(x_I[r])                                           -> Y_J[c], summed over ib and g
// acc1 is summed over the four t-lanes once per unit, acc2 over the eight g-lanes once per tile (warp shuffles),
// then added to Y with red.global.add.f64.  HERM: Y_J += conj(acc2) (= T^H x_I);  SYMC: Y_J += acc2 (= T^T conj(x_I)).
// 128 DFMA and 16 shared-memory loads per tile per warp.
#pragma once
#include "apply_kernel.cuh"

namespace bse {

__device__ __forceinline__ void cfma(double2 &acc, const double2 a, const double2 x)
{
    acc.x = fma(a.x, x.x, acc.x); acc.x = fma(-a.y, x.y, acc.x);
    acc.y = fma(a.x, x.y, acc.y); acc.y = fma(a.y, x.x, acc.y);
}

// NW consumer warps (8 or 16) + the producer warp.  NW = 16 (warp w owns tile columns 4w .. 4w+3: half a patch
// column, s = w & 1 of patch column jb = w >> 1; four consumer warps per scheduler, 96 registers) was measured
// SLOWER than NW = 8 at N = 98304 (complex64 store 7.6 vs 7.0 ms, complex128 12.1 vs 11.1 ms): only NW = 8 is
// instantiated.
template <int ES, int NW>
__global__ void __launch_bounds__((NW + 1) * 32, 1) apply_tiles_k1_kernel(const ApplyParams p)
{
    constexpr int TBY = TB * TB * ES, PBY = 64 * ES, NST = APPLY_STAGES * 16 / ES, S1 = 16 * ES;
    constexpr int NS = 16 / NW;                          // k-halves (s) of a patch column handled by one warp: 2 or 1
    extern __shared__ __align__(1024) char smem[];
    char *tile_s = smem;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + NST * TBY);
    uint64_t *full = bars, *empty = bars + NST;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < NST; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NW); }
        fence_barrier_init();
    }
    __syncthreads();

    if (warp == NW) {
        if (lane == 0) {                                   // producer: identical to the tensor-core kernel
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

    const int jb = (NW == 8) ? warp : (warp >> 1);        // patch column
    const int s0 = (NW == 8) ? 0 : (warp & 1);            // first k-half
    const int c0 = jb * 8 + s0 * 4;                       // first tile column of this warp (lane adds t, s adds 4)
    const int g = lane >> 2, t = lane & 3;
    const int g2 = (g >> 2) & 1, g1 = (g >> 1) & 1, g0 = g & 1, t1 = (t >> 1) & 1, t0 = t & 1;
    const int offP1 = (((g2 << 2) | g1) * 8 + ((g0 << 2) | (t0 << 1) | (g1 ^ t1))) * ES + s0 * S1;   // + s * S1
    const bool herm = (p.pass == PASS_HERM);
    const double sgn = p.sign;
    const double2 zero2 = make_double2(0.0, 0.0);
    const double2 *x = p.X;

    // x_J rows c0 + 4s + t, RAW: the loads are issued one tile ahead, so nothing may touch the values here (a
    // multiply at this point would wait out the L2 latency at every tile -- 14 % of all stall samples in round 1)
    auto load_xj = [&](int K, double2 (&v)[NS]) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            int64_t row = (int64_t)K * TB + c0 + s * 4 + t;
            v[s] = row < p.N ? __ldg(x + row) : zero2;
        }
    };
    const double sgn_im = herm ? sgn : -sgn;             // P1 operand: x_J (HERM) or conj(x_J) (SYMC), times the pass sign

    int st = 0;
    uint32_t ph = 0;
    for (int64_t u = p.u_begin + blockIdx.x; u < p.n_units; u += gridDim.x) {
        int I, J0, J1;
        apply_decode_unit(u, p.L, I, J0, J1);

        double2 xjn[NS];
        load_xj(J0, xjn);
        // conj(x_I[8 ib + g]) times the pass sign: the P2 operand, in registers for the whole unit
        double2 xi[8];
#pragma unroll
        for (int ib = 0; ib < 8; ++ib) {
            int64_t row = (int64_t)I * TB + ib * 8 + g;
            double2 a = row < p.N ? __ldg(x + row) : zero2;
            xi[ib] = make_double2(sgn * a.x, -sgn * a.y);
        }
        double2 acc1[8];
#pragma unroll
        for (int ib = 0; ib < 8; ++ib) acc1[ib] = zero2;

        for (int J = J0; J < J1; ++J) {
            double2 xj[NS];
#pragma unroll
            for (int s = 0; s < NS; ++s) xj[s] = make_double2(sgn * xjn[s].x, sgn_im * xjn[s].y);
            if (J + 1 < J1) load_xj(J + 1, xjn);            // prefetch the next tile's x_J rows

            mbar_wait(&full[st], ph);
            const char *tp = tile_s + st * TBY + jb * 8 * PBY + offP1;
            int live = 0;
            if (I != J) {
                double2 acc2[NS];
#pragma unroll
                for (int s = 0; s < NS; ++s) acc2[s] = zero2;
#pragma unroll
                for (int h = 0; h < 8; h += 4) {             // four patch rows at a time (register budget)
                    double2 a[4][NS];
#pragma unroll
                    for (int r = 0; r < 4; ++r)
#pragma unroll
                        for (int s = 0; s < NS; ++s) a[r][s] = load_frag<ES>(tp + (h + r) * PBY + s * S1);
#pragma unroll
                    for (int r = 0; r < 4; ++r)
#pragma unroll
                        for (int s = 0; s < NS; ++s) {
                            cfma(acc1[h + r], a[r][s], xj[s]);
                            cfma(acc2[s], a[r][s], xi[h + r]);
                        }
                }
                // dependent release (see apply_kernel.cuh): values computed from every load of this stage
#pragma unroll
                for (int ib = 0; ib < 8; ++ib) live |= __double2hiint(acc1[ib].x);
#pragma unroll
                for (int s = 0; s < NS; ++s) live |= __double2hiint(acc2[s].x);
                __syncwarp();
                if (lane == 0)
                    mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(&empty[st]) + (live & p.zero)));
                // sum over the eight g-lanes (lane bits 2..4), then lanes g == 0 add Y_J[c0 + 4s + t]
#pragma unroll
                for (int s = 0; s < NS; ++s) {
                    double yr = acc2[s].x, yi = acc2[s].y;
#pragma unroll
                    for (int m = 4; m < 32; m <<= 1) {
                        yr += __shfl_xor_sync(0xffffffffu, yr, m);
                        yi += __shfl_xor_sync(0xffffffffu, yi, m);
                    }
                    const int64_t row = (int64_t)J * TB + c0 + s * 4 + t;
                    if (g == 0 && row < p.N) {
                        double *y = p.Y + 2 * row;
                        red_add(y, yr);
                        red_add(y + 1, herm ? -yi : yi);
                    }
                }
            } else {
#pragma unroll
                for (int h = 0; h < 8; h += 4) {
                    double2 a[4][NS];
#pragma unroll
                    for (int r = 0; r < 4; ++r)
#pragma unroll
                        for (int s = 0; s < NS; ++s) a[r][s] = load_frag<ES>(tp + (h + r) * PBY + s * S1);
#pragma unroll
                    for (int r = 0; r < 4; ++r)
#pragma unroll
                        for (int s = 0; s < NS; ++s) cfma(acc1[h + r], a[r][s], xj[s]);
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
