// Single-column kernels of the real-form store (Eq. 3; roles and modes as RoleReal in apply_tiles.cuh).
#pragma once
#include "apply_kernel_k1.cuh"

namespace bse {

// Single-column variant of apply_tiles_kernel<ES, RoleReal<MODE>> (plain FMAs, every entry loaded once and used for both products, as in
// apply_kernel_k1.cuh): per stored entry (Ar, Ai) two FMAs for P1 and two for P2 -- half of the complex single-column
// kernel -- so that the binary32-plane store, whose DMMA kernel is bound by the tensor pipe for every k, streams at the
// HBM rate when k = 1 (the full-mode quadrature recurrence at the paper's precision).
//   MODE 0:  (re_I, im_I) += (Ar, Ai) a_J;    re_J += Ar a_I + Ai b_I
//   MODE 1:  (re_I, im_I) += (-Ai, Ar) b_J;   im_J += Ar b_I - Ai a_I
template <int MODE> __device__ __forceinline__ void rfma1(double2 &acc, const double2 a, const double xs)
{
    if (MODE == 0) { acc.x = fma(a.x, xs, acc.x); acc.y = fma(a.y, xs, acc.y); }
    else { acc.x = fma(-a.y, xs, acc.x); acc.y = fma(a.x, xs, acc.y); }
}

template <int ES, int MODE>
__global__ void __launch_bounds__(APPLY_THREADS, 1) apply_tiles_real_k1_kernel(const ApplyParams p)
{
    constexpr int NW = 8;
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

    int st = 0;
    uint32_t ph = 0;
    for (int64_t u = p.u_begin + blockIdx.x; u < p.n_units; u += gridDim.x) {
        int I, J0, J1;
        apply_decode_unit(u, p.L, I, J0, J1);

        double2 xjn[NS];
        load_xj(J0, xjn);
        // P2 operands (u, v) pairing with (Ar, Ai): MODE 0 (a_I, b_I), MODE 1 (b_I, -a_I); in registers for the whole unit
        double2 xi[8];
#pragma unroll
        for (int ib = 0; ib < 8; ++ib) {
            int64_t row = (int64_t)I * TB + ib * 8 + g;
            double2 a = row < p.N ? __ldg(x + row) : zero2;
            xi[ib] = MODE == 0 ? a : make_double2(a.y, -a.x);
        }
        double2 acc1[8];
#pragma unroll
        for (int ib = 0; ib < 8; ++ib) acc1[ib] = zero2;

        for (int J = J0; J < J1; ++J) {
            double xj[NS];                                  // a_J (MODE 0) or b_J (MODE 1)
#pragma unroll
            for (int s = 0; s < NS; ++s) xj[s] = MODE == 0 ? xjn[s].x : xjn[s].y;
            if (J + 1 < J1) load_xj(J + 1, xjn);            // prefetch the next tile's x_J rows

            mbar_wait(&full[st], ph);
            const char *tp = tile_s + st * TBY + jb * 8 * PBY + offP1;
            int live = 0;
            if (I != J) {
                double acc2[NS];
#pragma unroll
                for (int s = 0; s < NS; ++s) acc2[s] = 0.0;
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
                            rfma1<MODE>(acc1[h + r], a[r][s], xj[s]);
                            acc2[s] = fma(a[r][s].x, xi[h + r].x, acc2[s]);
                            acc2[s] = fma(a[r][s].y, xi[h + r].y, acc2[s]);
                        }
                }
                // dependent release (see apply_common.cuh): values computed from every load of this stage
#pragma unroll
                for (int ib = 0; ib < 8; ++ib) live |= __double2hiint(acc1[ib].x);
#pragma unroll
                for (int s = 0; s < NS; ++s) live |= __double2hiint(acc2[s]);
                __syncwarp();
                if (lane == 0)
                    mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(&empty[st]) + (live & p.zero)));
                // sum over the eight g-lanes (lane bits 2..4), then lanes g == 0 add Y_J[c0 + 4s + t]
#pragma unroll
                for (int s = 0; s < NS; ++s) {
                    double yr = acc2[s];
#pragma unroll
                    for (int m = 4; m < 32; m <<= 1) yr += __shfl_xor_sync(0xffffffffu, yr, m);
                    const int64_t row = (int64_t)J * TB + c0 + s * 4 + t;
                    if (g == 0 && row < p.N) red_add(p.Y + 2 * row + MODE, yr);      // re_J (MODE 0) / im_J (MODE 1)
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
                        for (int s = 0; s < NS; ++s) rfma1<MODE>(acc1[h + r], a[r][s], xj[s]);
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
