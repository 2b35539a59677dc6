// The tensor-core apply kernels: ONE skeleton -- tile ring, producer lane, unit walk, dependent stage
// release (apply_common.cuh) -- and three ROLES that supply the arithmetic of the two products of a stored tile,
//     P1 warps (0..3):  Y_I += T x_J       warp (rh, ch) owns tile rows 32 rh .. +31 x tile columns 32 ch .. +31 (16 patches),
//                                          accumulators kept in registers for a whole unit (a run of tiles of one tile row);
//     P2 warps (4..7):  Y_J += T^H x_I     warp r owns tile columns 16 r .. +15 (16 patches, all 64 rows), the x_I fragments in
//                                          registers for a whole unit, results flushed per tile.
// One P1 and one P2 warp share each scheduler.  The inner loops are LEAN: the B operands of the DMMAs come ready-made from the
// pre-pass (apply_prep.cuh: conjugation, pass sign, re/im selection, zero padding to whole tiles), results go to the padded
// block Ypad, so a tile costs its DMMAs, its fragment loads and a dozen bookkeeping instructions -- no bounds checks, no
// selects, and no plain FP64 arithmetic beyond what the method itself needs (a plain FP64 instruction costs issue cycles of
// the FP64 tensor pipe it shares: bse_selftest_peak measures 30 instead of 37 TFLOP/s with 8 DADDs per 12 DMMAs; round 1's
// kernels kept the DMMA pipe 76-81 % busy with everything resident).
//
//   Role4M   (1..4 columns, complex stores): four real products per complex product with N dimension n = 2 c + part,
//            [Yr | Yi] += Tr Ba + Ti Bb.  Images: img_a = Ba, img_b = Bb of the P1 product (sign tables in apply_prep.cuh); the
//            P2 product uses the same Ba and, for HERM, -Bb.  64 DMMAs per tile per warp.
//   Role3M   (5..8 columns, complex stores): three real products per complex product (Karatsuba) with n = column:
//            Q1 = Tr zr, Q2 = Ti zi, Q3 = (Tr + Ti)(zr + zi);  re = Q1 - Q2, im = Q3 - Q1 - Q2.  Image: img_pair = z (x, or
//            conj x for SYMC, times the pass sign).  P2 forms T^T conj(x) the same way from z2 = conj(x) (img_pair with the
//            imaginary part negated for HERM; img_a = z2r + z2i) and conjugates the result for HERM (T^H x = conj(T^T conj x)).
//            96 DMMAs and 32 DADDs (Tr + Ti, once per loaded fragment entry) per tile per warp.
//   RoleReal<MODE> (1..8 columns, real-form stores S = R + C, D = R - C; Eq. 3): tiles A = Ar + i Ai,
//            MODE 0:  P1: re_I += Ar a_J, im_I += Ai a_J;   P2: re_J += Ar^T a_I + Ai^T b_I
//            MODE 1:  P1: re_I -= Ai b_J, im_I += Ar b_J;   P2: im_J += Ar^T b_I - Ai^T a_I
//            (P = MODE 0 over S + MODE 1 over D;  M = MODE 0 over D + MODE 1 over S).  Image: img_pair = (a, b) = x.
// Rounding of the three-product form: |error| <= c eps (|Tr| + |Ti|)(|xr| + |xi|) per term, the normwise bound of the
// four-product form up to a factor 2; the parity tolerance of the apply is normwise (reading S11).
#pragma once
#include "apply_common.cuh"

namespace bse {

template <int ES> struct TileGeom {
    static constexpr int TBY = TB * TB * ES;              // tile bytes
    static constexpr int PBY = 64 * ES;                   // 8 x 8 patch bytes
    static constexpr int NST = APPLY_STAGES * 16 / ES;    // stages: the ring always fills the same 192 KB
    static constexpr int S1 = 16 * ES, S2 = 32 * ES;      // second k-step of the P1 / P2 fragment (16 / 32 slots on)
};

struct Lane {
    int g, t, offP1, offP2;                               // lane = 4 g + t; fragment byte offsets inside a patch (patch_slot)
};
template <int ES> __device__ __forceinline__ Lane make_lane(int lane)
{
    Lane l;
    l.g = lane >> 2; l.t = lane & 3;
    const int g2 = (l.g >> 2) & 1, g1 = (l.g >> 1) & 1, g0 = l.g & 1, t1 = (l.t >> 1) & 1, t0 = l.t & 1;
    l.offP1 = (((g2 << 2) | g1) * 8 + ((g0 << 2) | (t0 << 1) | (g1 ^ t1))) * ES;   // P1 reads (a = g, b = 4 s + t)
    l.offP2 = (((g2 << 1) | t1) * 8 + ((t0 << 2) | (g0 << 1) | (t1 ^ g1))) * ES;   // P2 reads (a = 4 s + t, b = g)
    return l;
}
constexpr int IMG_ROW = 8;                                 // image entries per matrix row
constexpr int IMG_TILE = TB * IMG_ROW;                     // image entries per tile row

// ------------------------------------------------------------------------------------------------------------------
// Role4M
// ------------------------------------------------------------------------------------------------------------------
struct Role4M {
    template <int ES> struct P1 {
        using G = TileGeom<ES>;
        double Ba[4][2], Bb[4][2], Ban[4][2], Bbn[4][2], C1[4][2];
        const double *xa, *xb;
        int frag, rh, lane_off;
        __device__ __forceinline__ P1(const TileParams &, const Lane &l, int rh_, int ch)
            : frag((4 * ch) * 8 * G::PBY + (4 * rh_) * G::PBY + l.offP1), rh(rh_), lane_off(((4 * ch) * 8 + l.t) * IMG_ROW + l.g) {}
        __device__ __forceinline__ void fetch()
        {
#pragma unroll
            for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    Ban[pc][s] = __ldg(xa + (pc * 8 + 4 * s) * IMG_ROW);
                    Bbn[pc][s] = __ldg(xb + (pc * 8 + 4 * s) * IMG_ROW);
                }
        }
        __device__ __forceinline__ void begin_unit(const TileParams &p, int, int J0)
        {
            xa = p.img_a + (int64_t)J0 * IMG_TILE + lane_off;
            xb = p.img_b + (int64_t)J0 * IMG_TILE + lane_off;
            fetch();
#pragma unroll
            for (int ib = 0; ib < 4; ++ib) C1[ib][0] = C1[ib][1] = 0.0;
        }
        __device__ __forceinline__ void next_operands(bool more)      // x_J of this tile in, x_J of the next tile requested
        {
#pragma unroll
            for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                for (int s = 0; s < 2; ++s) { Ba[pc][s] = Ban[pc][s]; Bb[pc][s] = Bbn[pc][s]; }
            if (more) { xa += IMG_TILE; xb += IMG_TILE; fetch(); }
        }
        __device__ __forceinline__ int tile(const char *stage)
        {
            const char *tp = stage + frag;
#pragma unroll
            for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    double2 a[4];
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) a[ib] = load_frag<ES>(tp + (pc * 8 + ib) * G::PBY + s * G::S1);
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) dmma(C1[ib], a[ib].x, Ba[pc][s]);      // four independent chains,
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) dmma(C1[ib], a[ib].y, Bb[pc][s]);      // dependent DMMAs 4 apart
                }
            int live = 0;
#pragma unroll
            for (int ib = 0; ib < 4; ++ib) live |= __double2hiint(C1[ib][0]);
            return live;
        }
        __device__ __forceinline__ void end_unit(const TileParams &p, const Lane &l, int I)
        {
            if (l.t < p.kc) {                              // accumulator entries = (re, im) of column t
                double *y = p.Ypad + (((int64_t)I * TB + (4 * rh) * 8 + l.g) * IMG_ROW + l.t) * 2;
#pragma unroll
                for (int ib = 0; ib < 4; ++ib) {
                    red_add(y + ib * 8 * IMG_ROW * 2, C1[ib][0]);
                    red_add(y + ib * 8 * IMG_ROW * 2 + 1, C1[ib][1]);
                }
            }
        }
    };
    template <int ES> struct P2 {
        using G = TileGeom<ES>;
        double xA[8][2], xB[8][2], Z[2][2];
        int frag, r;
        unsigned long long flip;
        __device__ __forceinline__ P2(const TileParams &p, const Lane &l, int r_)
            : frag((2 * r_) * 8 * G::PBY + l.offP2), r(r_), flip(p.pass == PASS_HERM ? SIGN_BIT : 0ull) {}
        __device__ __forceinline__ void begin_unit(const TileParams &p, const Lane &l, int I)
        {
            const double *xa = p.img_a + ((int64_t)I * TB + l.t) * IMG_ROW + l.g, *xb = p.img_b + ((int64_t)I * TB + l.t) * IMG_ROW + l.g;
#pragma unroll
            for (int ib = 0; ib < 8; ++ib)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    xA[ib][s] = __ldg(xa + (ib * 8 + 4 * s) * IMG_ROW);
                    xB[ib][s] = neg_if(__ldg(xb + (ib * 8 + 4 * s) * IMG_ROW), flip);     // HERM: Bb of T^H x = -Bb of T x
                }
        }
        __device__ __forceinline__ int tile(const TileParams &, const char *stage)
        {
            Z[0][0] = Z[0][1] = Z[1][0] = Z[1][1] = 0.0;
            const char *tp = stage + frag;
#pragma unroll
            for (int ib = 0; ib < 8; ib += 2) {
                double2 b[2][2][2];
#pragma unroll
                for (int q = 0; q < 2; ++q)
#pragma unroll
                    for (int s = 0; s < 2; ++s)
#pragma unroll
                        for (int pc = 0; pc < 2; ++pc) b[q][s][pc] = load_frag<ES>(tp + (pc * 8 + ib + q) * G::PBY + s * G::S2);
#pragma unroll
                for (int q = 0; q < 2; ++q)
#pragma unroll
                    for (int s = 0; s < 2; ++s) {                                         // two chains, dependent DMMAs 2 apart
                        dmma(Z[0], b[q][s][0].x, xA[ib + q][s]);
                        dmma(Z[1], b[q][s][1].x, xA[ib + q][s]);
                        dmma(Z[0], b[q][s][0].y, xB[ib + q][s]);
                        dmma(Z[1], b[q][s][1].y, xB[ib + q][s]);
                    }
            }
            return __double2hiint(Z[0][0]) | __double2hiint(Z[0][1]) | __double2hiint(Z[1][0]) | __double2hiint(Z[1][1]);
        }
        __device__ __forceinline__ void flush(const TileParams &p, const Lane &l, int J)
        {
            if (l.t < p.kc) {
                double *y = p.Ypad + (((int64_t)J * TB + (2 * r) * 8 + l.g) * IMG_ROW + l.t) * 2;
                red_add(y, Z[0][0]);
                red_add(y + 1, Z[0][1]);
                red_add(y + 8 * IMG_ROW * 2, Z[1][0]);
                red_add(y + 8 * IMG_ROW * 2 + 1, Z[1][1]);
            }
        }
    };
};

// ------------------------------------------------------------------------------------------------------------------
// Role3M
// ------------------------------------------------------------------------------------------------------------------
struct Role3M {
    template <int ES> struct P1 {
        using G = TileGeom<ES>;
        double2 z[4][2], zn[4][2];
        double Q1[4][2], Q2[4][2], Q3[4][2];
        const double2 *zp;
        int frag, rh, lane_off;
        __device__ __forceinline__ P1(const TileParams &, const Lane &l, int rh_, int ch)
            : frag((4 * ch) * 8 * G::PBY + (4 * rh_) * G::PBY + l.offP1), rh(rh_), lane_off(((4 * ch) * 8 + l.t) * IMG_ROW + l.g) {}
        __device__ __forceinline__ void fetch()
        {
#pragma unroll
            for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                for (int s = 0; s < 2; ++s) zn[pc][s] = __ldg(zp + (pc * 8 + 4 * s) * IMG_ROW);
        }
        __device__ __forceinline__ void begin_unit(const TileParams &p, int, int J0)
        {
            zp = p.img_pair + (int64_t)J0 * IMG_TILE + lane_off;
            fetch();
#pragma unroll
            for (int ib = 0; ib < 4; ++ib) Q1[ib][0] = Q1[ib][1] = Q2[ib][0] = Q2[ib][1] = Q3[ib][0] = Q3[ib][1] = 0.0;
        }
        __device__ __forceinline__ void next_operands(bool more)
        {
#pragma unroll
            for (int pc = 0; pc < 4; ++pc) { z[pc][0] = zn[pc][0]; z[pc][1] = zn[pc][1]; }
            if (more) { zp += IMG_TILE; fetch(); }
        }
        __device__ __forceinline__ int tile(const char *stage)
        {
            const char *tp = stage + frag;
#pragma unroll
            for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    const double zr = z[pc][s].x, zi = z[pc][s].y, zs = zr + zi;
                    double2 a[4];
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) a[ib] = load_frag<ES>(tp + (pc * 8 + ib) * G::PBY + s * G::S1);
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) {       // twelve independent chains
                        const double as = a[ib].x + a[ib].y;
                        dmma(Q1[ib], a[ib].x, zr);
                        dmma(Q2[ib], a[ib].y, zi);
                        dmma(Q3[ib], as, zs);
                    }
                }
            int live = 0;
#pragma unroll
            for (int ib = 0; ib < 4; ++ib) live |= __double2hiint(Q1[ib][0]) | __double2hiint(Q2[ib][0]) | __double2hiint(Q3[ib][0]);
            return live;
        }
        __device__ __forceinline__ void end_unit(const TileParams &p, const Lane &l, int I)
        {
            // accumulator entries e = 0, 1 belong to columns 2 t + e;  re = Q1 - Q2, im = Q3 - Q1 - Q2
            double *y = p.Ypad + (((int64_t)I * TB + (4 * rh) * 8 + l.g) * IMG_ROW + 2 * l.t) * 2;
#pragma unroll
            for (int e = 0; e < 2; ++e)
                if (2 * l.t + e < p.kc) {
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) {
                        red_add(y + ib * 8 * IMG_ROW * 2 + 2 * e, Q1[ib][e] - Q2[ib][e]);
                        red_add(y + ib * 8 * IMG_ROW * 2 + 2 * e + 1, (Q3[ib][e] - Q1[ib][e]) - Q2[ib][e]);
                    }
                }
        }
    };
    template <int ES> struct P2 {
        using G = TileGeom<ES>;
        double2 z2[8][2];                                    // conj(x_I) (times the pass sign), rows 8 ib + 4 s + t, column g
        double zs[8][2];                                     // z2r + z2i of the same rows (from the pre-pass: no FP64 add here)
        double Q1[2][2], Q2[2][2], Q3[2][2];
        int frag, r;
        unsigned long long eflip;                            // HERM: the result is conjugated
        __device__ __forceinline__ P2(const TileParams &p, const Lane &l, int r_)
            : frag((2 * r_) * 8 * G::PBY + l.offP2), r(r_), eflip(p.pass == PASS_HERM ? SIGN_BIT : 0ull) {}
        __device__ __forceinline__ void begin_unit(const TileParams &p, const Lane &l, int I)
        {
            const unsigned long long flip = p.pass == PASS_HERM ? SIGN_BIT : 0ull;          // img_pair holds x for HERM: conjugate it
            const double2 *zp = p.img_pair + ((int64_t)I * TB + l.t) * IMG_ROW + l.g;
            const double *zs2 = p.img_a + ((int64_t)I * TB + l.t) * IMG_ROW + l.g;
#pragma unroll
            for (int ib = 0; ib < 8; ++ib)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    const double2 v = __ldg(zp + (ib * 8 + 4 * s) * IMG_ROW);
                    z2[ib][s] = make_double2(v.x, neg_if(v.y, flip));
                    zs[ib][s] = __ldg(zs2 + (ib * 8 + 4 * s) * IMG_ROW);
                }
        }
        __device__ __forceinline__ int tile(const TileParams &, const char *stage)
        {
#pragma unroll
            for (int pc = 0; pc < 2; ++pc) Q1[pc][0] = Q1[pc][1] = Q2[pc][0] = Q2[pc][1] = Q3[pc][0] = Q3[pc][1] = 0.0;
            const char *tp = stage + frag;
#pragma unroll
            for (int ib = 0; ib < 8; ib += 2) {
                double2 b[2][2][2];
#pragma unroll
                for (int q = 0; q < 2; ++q)
#pragma unroll
                    for (int s = 0; s < 2; ++s)
#pragma unroll
                        for (int pc = 0; pc < 2; ++pc) b[q][s][pc] = load_frag<ES>(tp + (pc * 8 + ib + q) * G::PBY + s * G::S2);
#pragma unroll
                for (int q = 0; q < 2; ++q)
#pragma unroll
                    for (int s = 0; s < 2; ++s)
#pragma unroll
                        for (int pc = 0; pc < 2; ++pc) {                                    // six independent chains
                            const double bs = b[q][s][pc].x + b[q][s][pc].y;
                            dmma(Q1[pc], b[q][s][pc].x, z2[ib + q][s].x);
                            dmma(Q2[pc], b[q][s][pc].y, z2[ib + q][s].y);
                            dmma(Q3[pc], bs, zs[ib + q][s]);
                        }
            }
            int live = 0;
#pragma unroll
            for (int pc = 0; pc < 2; ++pc) live |= __double2hiint(Q1[pc][0]) | __double2hiint(Q2[pc][0]) | __double2hiint(Q3[pc][0]);
            return live;
        }
        __device__ __forceinline__ void flush(const TileParams &p, const Lane &l, int J)
        {
            // T^T z2:  re = Q1 - Q2, im = Q3 - Q1 - Q2;  HERM adds its conjugate (T^H x = conj(T^T conj x))
            double *y = p.Ypad + (((int64_t)J * TB + (2 * r) * 8 + l.g) * IMG_ROW + 2 * l.t) * 2;
#pragma unroll
            for (int e = 0; e < 2; ++e)
                if (2 * l.t + e < p.kc) {
#pragma unroll
                    for (int pc = 0; pc < 2; ++pc) {
                        red_add(y + pc * 8 * IMG_ROW * 2 + 2 * e, Q1[pc][e] - Q2[pc][e]);
                        red_add(y + pc * 8 * IMG_ROW * 2 + 2 * e + 1, neg_if((Q3[pc][e] - Q1[pc][e]) - Q2[pc][e], eflip));
                    }
                }
        }
    };
};

// ------------------------------------------------------------------------------------------------------------------
// RoleReal<MODE>
// ------------------------------------------------------------------------------------------------------------------
template <int MODE> struct RoleReal {
    template <int ES> struct P1 {
        using G = TileGeom<ES>;
        double x[4][2], xn[4][2];                            // a_J (MODE 0) or b_J (MODE 1)
        double U[4][2], W[4][2];                             // U = Ar x, W = Ai x
        const double *xp;
        int frag, rh, lane_off;
        __device__ __forceinline__ P1(const TileParams &, const Lane &l, int rh_, int ch)
            : frag((4 * ch) * 8 * G::PBY + (4 * rh_) * G::PBY + l.offP1), rh(rh_),
              lane_off((((4 * ch) * 8 + l.t) * IMG_ROW + l.g) * 2 + MODE) {}
        __device__ __forceinline__ void fetch()
        {
#pragma unroll
            for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                for (int s = 0; s < 2; ++s) xn[pc][s] = __ldg(xp + (pc * 8 + 4 * s) * IMG_ROW * 2);
        }
        __device__ __forceinline__ void begin_unit(const TileParams &p, int, int J0)
        {
            xp = reinterpret_cast<const double *>(p.img_pair) + (int64_t)J0 * IMG_TILE * 2 + lane_off;
            fetch();
#pragma unroll
            for (int ib = 0; ib < 4; ++ib) U[ib][0] = U[ib][1] = W[ib][0] = W[ib][1] = 0.0;
        }
        __device__ __forceinline__ void next_operands(bool more)
        {
#pragma unroll
            for (int pc = 0; pc < 4; ++pc) { x[pc][0] = xn[pc][0]; x[pc][1] = xn[pc][1]; }
            if (more) { xp += IMG_TILE * 2; fetch(); }
        }
        __device__ __forceinline__ int tile(const char *stage)
        {
            const char *tp = stage + frag;
#pragma unroll
            for (int pc = 0; pc < 4; ++pc)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    double2 a[4];
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) a[ib] = load_frag<ES>(tp + (pc * 8 + ib) * G::PBY + s * G::S1);
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) {       // eight independent chains
                        dmma(U[ib], a[ib].x, x[pc][s]);
                        dmma(W[ib], a[ib].y, x[pc][s]);
                    }
                }
            int live = 0;
#pragma unroll
            for (int ib = 0; ib < 4; ++ib) live |= __double2hiint(U[ib][0]) | __double2hiint(W[ib][0]);
            return live;
        }
        __device__ __forceinline__ void end_unit(const TileParams &p, const Lane &l, int I)
        {
            double *y = p.Ypad + (((int64_t)I * TB + (4 * rh) * 8 + l.g) * IMG_ROW + 2 * l.t) * 2;
#pragma unroll
            for (int e = 0; e < 2; ++e)
                if (2 * l.t + e < p.kc) {
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) {
                        double *yy = y + ib * 8 * IMG_ROW * 2 + 2 * e;
                        if (MODE == 0) { red_add(yy, U[ib][e]); red_add(yy + 1, W[ib][e]); }
                        else { red_add(yy, neg_if(W[ib][e], SIGN_BIT)); red_add(yy + 1, U[ib][e]); }
                    }
                }
        }
    };
    template <int ES> struct P2 {
        using G = TileGeom<ES>;
        double xA[8][2], xB[8][2], Z[2][2];                  // xA pairs with Ar^T, xB with Ai^T:  MODE 0 (a_I, b_I), MODE 1 (b_I, -a_I)
        int frag, r;
        __device__ __forceinline__ P2(const TileParams &, const Lane &l, int r_) : frag((2 * r_) * 8 * G::PBY + l.offP2), r(r_) {}
        __device__ __forceinline__ void begin_unit(const TileParams &p, const Lane &l, int I)
        {
            const double2 *zp = p.img_pair + ((int64_t)I * TB + l.t) * IMG_ROW + l.g;
#pragma unroll
            for (int ib = 0; ib < 8; ++ib)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    const double2 v = __ldg(zp + (ib * 8 + 4 * s) * IMG_ROW);
                    xA[ib][s] = MODE == 0 ? v.x : v.y;
                    xB[ib][s] = MODE == 0 ? v.y : neg_if(v.x, SIGN_BIT);
                }
        }
        __device__ __forceinline__ int tile(const TileParams &, const char *stage)
        {
            Z[0][0] = Z[0][1] = Z[1][0] = Z[1][1] = 0.0;
            const char *tp = stage + frag;
#pragma unroll
            for (int ib = 0; ib < 8; ib += 2) {
                double2 b[2][2][2];
#pragma unroll
                for (int q = 0; q < 2; ++q)
#pragma unroll
                    for (int s = 0; s < 2; ++s)
#pragma unroll
                        for (int pc = 0; pc < 2; ++pc) b[q][s][pc] = load_frag<ES>(tp + (pc * 8 + ib + q) * G::PBY + s * G::S2);
#pragma unroll
                for (int q = 0; q < 2; ++q)
#pragma unroll
                    for (int s = 0; s < 2; ++s) {                                         // two chains, dependent DMMAs 2 apart
                        dmma(Z[0], b[q][s][0].x, xA[ib + q][s]);
                        dmma(Z[1], b[q][s][1].x, xA[ib + q][s]);
                        dmma(Z[0], b[q][s][0].y, xB[ib + q][s]);
                        dmma(Z[1], b[q][s][1].y, xB[ib + q][s]);
                    }
            }
            return __double2hiint(Z[0][0]) | __double2hiint(Z[0][1]) | __double2hiint(Z[1][0]) | __double2hiint(Z[1][1]);
        }
        __device__ __forceinline__ void flush(const TileParams &p, const Lane &l, int J)
        {
            double *y = p.Ypad + (((int64_t)J * TB + (2 * r) * 8 + l.g) * IMG_ROW + 2 * l.t) * 2 + MODE;     // re_J (MODE 0) / im_J (MODE 1)
#pragma unroll
            for (int e = 0; e < 2; ++e)
                if (2 * l.t + e < p.kc) {
                    red_add(y + 2 * e, Z[0][e]);
                    red_add(y + 8 * IMG_ROW * 2 + 2 * e, Z[1][e]);
                }
        }
    };
};

// ------------------------------------------------------------------------------------------------------------------
// The skeleton.  ES = bytes per stored complex entry (bse_common.cuh): 16 -> LDS.128 fragments, 8 -> LDS.64 + conversion.
// ------------------------------------------------------------------------------------------------------------------
template <int ES, class Role>
__global__ void __launch_bounds__(APPLY_THREADS, 1) apply_tiles_kernel(const TileParams p)
{
    using G = TileGeom<ES>;
    extern __shared__ __align__(1024) char smem[];
    char *tile_s = smem;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + G::NST * G::TBY);
    uint64_t *full = bars, *empty = bars + G::NST;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < G::NST; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], APPLY_CONSUMERS); }
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
                const char *src = p.tiles + tile_index(I, J0) * (int64_t)G::TBY;
                for (int J = J0; J < J1; ++J, src += G::TBY) {
                    mbar_wait(&empty[st], ph ^ 1);
                    mbar_expect_tx(&full[st], (uint32_t)G::TBY);
                    bulk_g2s_hint(tile_s + st * G::TBY, src, G::TBY, &full[st], pol);
                    if (++st == G::NST) { st = 0; ph ^= 1; }
                }
            }
        }
        return;
    }

    const Lane l = make_lane<ES>(lane);
    const char *stage = tile_s;
    int st = 0;
    uint32_t ph = 0;
    // stage release: data-dependent on the accumulators (apply_common.cuh); then on to the next stage of the ring
    auto release = [&](int live) {
        __syncwarp();
        if (lane == 0) mbar_arrive(reinterpret_cast<uint64_t *>(reinterpret_cast<char *>(&empty[st]) + (live & p.zero)));
        stage += G::TBY;
        if (++st == G::NST) { st = 0; ph ^= 1; stage = tile_s; }
    };

    if (warp < 4) {
        typename Role::template P1<ES> w(p, l, warp & 1, warp >> 1);
        for (int64_t u = p.u_begin + blockIdx.x; u < p.n_units; u += gridDim.x) {
            int I, J0, J1;
            apply_decode_unit(u, p.L, I, J0, J1);
            w.begin_unit(p, I, J0);
            for (int J = J0; J < J1; ++J) {
                w.next_operands(J + 1 < J1);
                mbar_wait(&full[st], ph);
                release(w.tile(stage));
            }
            w.end_unit(p, l, I);
        }
    } else {
        typename Role::template P2<ES> w(p, l, warp - 4);
        for (int64_t u = p.u_begin + blockIdx.x; u < p.n_units; u += gridDim.x) {
            int I, J0, J1;
            apply_decode_unit(u, p.L, I, J0, J1);
            w.begin_unit(p, l, I);
            for (int J = J0; J < J1; ++J) {
                mbar_wait(&full[st], ph);
                if (I != J) {
                    release(w.tile(p, stage));
                    w.flush(p, l, J);
                } else {
                    release(0);                             // diagonal tile: stored in full, P1 only -- nothing was read here
                }
            }
        }
    }
}

}  // namespace bse
