// Pre- and post-pass of the tensor-core apply kernels (apply_tiles.cuh): O(N k) elementwise work that takes every bounds
// check, conjugation, sign and re/im selection out of the O(N^2 k) tile loop.
//
// prep: reads up to 8 columns of the caller's X (each with its own pointer, optionally conjugated on the way in -- the general
// full-mode apply feeds conj(X2) and X1 side by side) and writes the operand IMAGES, [rows_pad][8] arrays
// with rows >= N and columns >= kc zero, for one or two operand sets (a half apply over complex stores needs the HERM images
// for R and the SYMC images for C).  With z = s x (HERM, real form) or z = s conj(x) (SYMC), s the pass sign:
//     IMG_4M :  img_a[row][2 c + part] = Ba = (zr, zi),   img_b[row][2 c + part] = Bb = (-zi, zr)          (c < 4)
//               i.e. HERM: Ba = [xr, xi], Bb = [-xi, xr];  SYMC: Ba = [xr, -xi], Bb = [xi, xr]  -- [Yr | Yi] += Tr Ba + Ti Bb
//     IMG_3M :  img_pair[row][c] = (zr, zi);   img_a[row][c] = z2r + z2i with z2 = s conj(x) (the P2 operand sum)
//     IMG_REAL: img_pair[row][c] = (xr, xi)
// and zeroes Ypad.  post: Y(:, c) = Ypad[:, c] (or -conj of it) for the live columns, rows < N.
#pragma once
#include "apply_common.cuh"

namespace bse {

enum { IMG_4M = 0, IMG_3M = 1, IMG_REAL = 2 };

struct PrepSet {
    const double2 *src[8];     // source column c (n rows), NULL beyond kc
    unsigned conj_in;          // bit c: conjugate source column c on the way in
    int kind, pass, kc;
    double sign;
    double2 *img_pair;
    double *img_a, *img_b;
};
struct PrepParams {
    PrepSet set[2];
    int n_sets;
    int64_t N, rows_pad;
    double *Ypad;              // zeroed when non-NULL
};

__global__ void __launch_bounds__(256) apply_prep_kernel(const PrepParams p)
{
    const int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (idx >= p.rows_pad * 8) return;
    const int64_t row = idx >> 3;
    const int n = (int)(idx & 7);
    if (p.Ypad) { p.Ypad[2 * idx] = 0.0; p.Ypad[2 * idx + 1] = 0.0; }
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        if (q >= p.n_sets) break;
        const PrepSet &s = p.set[q];
        const int c = s.kind == IMG_4M ? (n >> 1) : n;
        double2 x = make_double2(0.0, 0.0);
        if (row < p.N && c < s.kc) {
            x = s.src[c][row];
            if ((s.conj_in >> c) & 1) x.y = -x.y;
        }
        // z = s x (HERM, real form) or s conj(x) (SYMC)
        const double zr = s.sign * x.x, zi = (s.pass == PASS_SYMC && s.kind != IMG_REAL) ? -s.sign * x.y : s.sign * x.y;
        if (s.kind == IMG_4M) {
            const int part = n & 1;
            s.img_a[idx] = part ? zi : zr;
            s.img_b[idx] = part ? zr : -zi;
        } else {
            s.img_pair[idx] = make_double2(zr, zi);
            // z2 = s conj(x):  HERM (zr, -zi), SYMC (zr, zi)
            if (s.kind == IMG_3M) s.img_a[idx] = s.pass == PASS_HERM ? zr - zi : zr + zi;
        }
    }
}

struct PostParams {
    const double2 *Ypad;
    double2 *dst[8];           // destination column c (n rows)
    unsigned neg_conj;         // bit c: store -conj(value)
    int kc;
    int64_t N;
};

__global__ void __launch_bounds__(256) apply_post_kernel(const PostParams p)
{
    const int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (idx >= p.N * 8) return;
    const int64_t row = idx >> 3;
    const int c = (int)(idx & 7);
    if (c >= p.kc) return;
    double2 v = p.Ypad[idx];
    if ((p.neg_conj >> c) & 1) v.x = -v.x;
    p.dst[c][row] = v;
}

}  // namespace bse
