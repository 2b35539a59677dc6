// Packed triangular tile store: pack / unpack / on-device generators.
#pragma once
#include "bse_common.cuh"
#include "rng.cuh"

namespace bse {

// One thread per stored complex entry: grid.x covers the 4096 entries of a tile, blockIdx.y/z the tiles.
// Source entry functor f(gi, gj) is only evaluated for gj <= gi < N (the lower triangle).
// es = 16: complex128 entries; es = 8: each component rounded to nearest-even float (cvt.rn.f32.f64).
template <class F>
__device__ __forceinline__ void store_tile_entry(char *tiles, int es, int64_t N, int which, int64_t tile, int I, int J,
                                                 int il, int jl, F f)
{
    int64_t gi = (int64_t)I * TB + il, gj = (int64_t)J * TB + jl;
    double2 v = make_double2(0.0, 0.0);
    if (gi < N && gj < N) {
        if (gj <= gi) {
            v = f(gi, gj);
            if (gi == gj && which == 0) v.y = 0.0;            // Hermitian: real diagonal
        } else {                                               // only reached in diagonal tiles: mirror
            v = f(gj, gi);
            if (which == 0) v.y = -v.y;
        }
    }
    char *dst = tiles + tile * tile_bytes_es(es) + tile_offset_es(il, jl, es);
    if (es == ES_C128) *reinterpret_cast<double2 *>(dst) = v;
    else *reinterpret_cast<float2 *>(dst) = make_float2(__double2float_rn(v.x), __double2float_rn(v.y));
}

__device__ __forceinline__ void tile_from_linear(int64_t tile, int &I, int &J)
{
    // I = floor((sqrt(8 t + 1) - 1) / 2), with integer fix-up
    int64_t i = (int64_t)((sqrt(8.0 * (double)tile + 1.0) - 1.0) * 0.5);
    while (i * (i + 1) / 2 > tile) --i;
    while ((i + 1) * (i + 2) / 2 <= tile) ++i;
    I = (int)i;
    J = (int)(tile - i * (i + 1) / 2);
}

__global__ void __launch_bounds__(256) pack_from_dense_kernel(const double2 *__restrict__ dense, int64_t ld,
                                                              int64_t N, int which, char *__restrict__ tiles,
                                                              int es, int64_t n_tiles)
{
    int64_t tile = blockIdx.y + (int64_t)blockIdx.z * gridDim.y;
    if (tile >= n_tiles) return;
    int I, J;
    tile_from_linear(tile, I, J);
    int e = blockIdx.x * blockDim.x + threadIdx.x;   // 0..4095, il fastest (coalesced dense reads)
    int il = e & 63, jl = e >> 6;
    store_tile_entry(tiles, es, N, which, tile, I, J, il, jl,
                     [&](int64_t gi, int64_t gj) { return dense[gi + gj * ld]; });
}

__global__ void __launch_bounds__(256) unpack_to_dense_kernel(const char *__restrict__ tiles, int es, int64_t N, int which,
                                                              double2 *__restrict__ dense, int64_t ld, int64_t n_tiles)
{
    int64_t tile = blockIdx.y + (int64_t)blockIdx.z * gridDim.y;
    if (tile >= n_tiles) return;
    int I, J;
    tile_from_linear(tile, I, J);
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    int il = e & 63, jl = e >> 6;
    int64_t gi = (int64_t)I * TB + il, gj = (int64_t)J * TB + jl;
    if (gi >= N || gj >= N) return;
    const char *src = tiles + tile * tile_bytes_es(es) + tile_offset_es(il, jl, es);
    double2 v;
    if (es == ES_C128) v = *reinterpret_cast<const double2 *>(src);
    else { float2 f = *reinterpret_cast<const float2 *>(src); v = make_double2((double)f.x, (double)f.y); }
    dense[gi + gj * ld] = v;
    if (I != J) {   // mirror image of an off-diagonal tile
        if (which == 0) v.y = -v.y;
        dense[gj + gi * ld] = v;
    }
}

// d_eps_i ~ U[1,10] sorted ascending inside each group (one thread per group; group <= 64)
__global__ void transition_energies_kernel(double *__restrict__ d, int64_t N, int group, uint64_t h0)
{
    int64_t gidx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int64_t base = gidx * group;
    if (base >= N) return;
    double v[64];
    for (int a = 0; a < group; ++a) {
        uint64_t h2, h3;
        hash2(h0, (uint64_t)(base + a), 0, h2, h3);
        v[a] = 1.0 + 9.0 * u01(h2);
    }
    for (int a = 1; a < group; ++a) {   // insertion sort
        double x = v[a];
        int b = a - 1;
        while (b >= 0 && v[b] > x) { v[b + 1] = v[b]; --b; }
        v[b + 1] = x;
    }
    for (int a = 0; a < group; ++a) d[base + a] = v[a];
}

__global__ void __launch_bounds__(256) fill_synthetic_kernel(char *__restrict__ tiles, int es, int64_t N, int which,
                                                             uint64_t h0, double sigma,
                                                             const double *__restrict__ deps, int64_t tile0,
                                                             int64_t tile1)
{
    int64_t tile = tile0 + blockIdx.y + (int64_t)blockIdx.z * gridDim.y;      // global tile number, [tile0, tile1)
    if (tile >= tile1) return;
    int I, J;
    tile_from_linear(tile, I, J);
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    int il = e & 63, jl = e >> 6;
    store_tile_entry(tiles, es, N, which, tile, I, J, il, jl, [&](int64_t gi, int64_t gj) {
        double2 g = normal_pair(h0, (uint64_t)gi, (uint64_t)gj);
        double dec = 1.0 + fabs((double)gi - (double)gj) / 64.0;
        if (which == 0) {
            if (gi == gj) return make_double2(0.1 * g.x + deps[gi] + sigma, 0.0);
            return make_double2(0.1 * g.x / dec, 0.1 * g.y / dec);
        }
        return make_double2(0.05 * g.x / dec, 0.05 * g.y / dec);
    });
}

// R_ij = lam_i d_ij - 2 u_i conj(u_j) (lam_i + lam_j - 2 s)
__global__ void __launch_bounds__(256) fill_closed_tda_kernel(char *__restrict__ tiles, int es, int64_t N,
                                                              const double *__restrict__ lam,
                                                              const double2 *__restrict__ u, double s, int64_t n_tiles)
{
    int64_t tile = blockIdx.y + (int64_t)blockIdx.z * gridDim.y;
    if (tile >= n_tiles) return;
    int I, J;
    tile_from_linear(tile, I, J);
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    int il = e & 63, jl = e >> 6;
    store_tile_entry(tiles, es, N, 0, tile, I, J, il, jl, [&](int64_t gi, int64_t gj) {
        double2 a = u[gi], b = u[gj];
        double pr = a.x * b.x + a.y * b.y, pi = a.y * b.x - a.x * b.y;   // u_i conj(u_j)
        double f = -2.0 * (lam[gi] + lam[gj] - 2.0 * s);
        double2 v = make_double2(f * pr, f * pi);
        if (gi == gj) v.x += lam[gi];
        return v;
    });
}

// R = U (M+ + M-)/2 U^H, C = U (M+ - M-)/2 U^T, M+- real closed forms as above with real u.
__global__ void __launch_bounds__(256) fill_closed_full_kernel(char *__restrict__ tiles, int es, int64_t N, int which,
                                                               const double *__restrict__ d1,
                                                               const double *__restrict__ d2,
                                                               const double *__restrict__ ur,
                                                               const double *__restrict__ phi, double s1, double s2,
                                                               int64_t n_tiles)
{
    int64_t tile = blockIdx.y + (int64_t)blockIdx.z * gridDim.y;
    if (tile >= n_tiles) return;
    int I, J;
    tile_from_linear(tile, I, J);
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    int il = e & 63, jl = e >> 6;
    store_tile_entry(tiles, es, N, which, tile, I, J, il, jl, [&](int64_t gi, int64_t gj) {
        double uu = ur[gi] * ur[gj];
        double mp = -2.0 * uu * (d1[gi] + d1[gj] - 2.0 * s1);
        double mm = -2.0 * uu * (d2[gi] + d2[gj] - 2.0 * s2);
        if (gi == gj) { mp += d1[gi]; mm += d2[gi]; }
        double val = (which == 0) ? 0.5 * (mp + mm) : 0.5 * (mp - mm);
        double ang = (which == 0) ? (phi[gi] - phi[gj]) : (phi[gi] + phi[gj]);
        double sn, cs;
        sincos(ang, &sn, &cs);
        return make_double2(val * cs, val * sn);
    });
}

}  // namespace bse
