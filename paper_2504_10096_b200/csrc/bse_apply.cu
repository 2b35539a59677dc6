// The operator applies: handle set-up of the tile kernels, the launch layer that turns a block
// of columns into groups (pre-pass -> tile passes -> post-pass, or the single-column kernels), and the C-ABI entry points
// bse_apply, bse_apply_half, bse_apply_host.
#include <cstdlib>

#include "apply_kernel_k1.cuh"
#include "apply_kernel_real_k1.cuh"
#include "apply_prep.cuh"
#include "apply_tiles.cuh"
#include "bse_internal.h"

namespace bse {

// ---------------------------------------------------------------------------------------------------------------------
// handle set-up
// ---------------------------------------------------------------------------------------------------------------------
template <class K> static cudaError_t big_smem(K kernel)
{
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, APPLY_SMEM);
}

static bse_status_t apply_kernel_attributes()
{
    // cudaFuncSetAttribute is per device: remember which devices of this process have been set up
    static std::atomic<uint64_t> attr_devices{0};
    int dev = 0;
    BSE_CUDA(cudaGetDevice(&dev));
    if (dev >= 64 || !(attr_devices.load(std::memory_order_acquire) & (1ull << dev))) {
        BSE_CUDA(big_smem(apply_tiles_kernel<16, Role4M>));
        BSE_CUDA(big_smem(apply_tiles_kernel<8, Role4M>));
        BSE_CUDA(big_smem(apply_tiles_kernel<16, Role3M>));
        BSE_CUDA(big_smem(apply_tiles_kernel<8, Role3M>));
        BSE_CUDA(big_smem(apply_tiles_kernel<16, RoleReal<0>>));
        BSE_CUDA(big_smem(apply_tiles_kernel<16, RoleReal<1>>));
        BSE_CUDA(big_smem(apply_tiles_kernel<8, RoleReal<0>>));
        BSE_CUDA(big_smem(apply_tiles_kernel<8, RoleReal<1>>));
        BSE_CUDA(big_smem(apply_tiles_k1_kernel<16, 8>));
        BSE_CUDA(big_smem(apply_tiles_k1_kernel<8, 8>));
        BSE_CUDA(big_smem(apply_tiles_real_k1_kernel<16, 0>));
        BSE_CUDA(big_smem(apply_tiles_real_k1_kernel<16, 1>));
        BSE_CUDA(big_smem(apply_tiles_real_k1_kernel<8, 0>));
        BSE_CUDA(big_smem(apply_tiles_real_k1_kernel<8, 1>));
        if (dev < 64) attr_devices.fetch_or(1ull << dev, std::memory_order_release);
    }
    return BSE_OK;
}

// operand workspace: two image sets (pair [16 doubles per row], a, b [8 each]) + Ypad [16] = 80 doubles per padded row,
// and, for real-form handles, the four blocks U, V, P(U), M(V) of the general apply (8 columns each)
static inline int64_t rows_pad_of(const bse_handle_s *h) { return (int64_t)h->nt * TB; }
static inline size_t op_doubles(const bse_handle_s *h) { return (size_t)rows_pad_of(h) * 80; }

bse_status_t handle_finalize(bse_handle_s *h)
{
    bse_status_t st = apply_kernel_attributes();
    if (st) return st;
    // knobs are read here, once: BSE_APPLY_UNIT (tiles per unit), BSE_APPLY_K1=0 (tensor-core kernels for single columns too)
    const int64_t total_tiles = (int64_t)h->nt * (h->nt + 1) / 2;
    int64_t L = total_tiles / ((int64_t)h->num_sms * 12);
    if (L < 1) L = 1;
    if (L > 32) L = 32;
    if (const char *e = getenv("BSE_APPLY_UNIT")) { int v = atoi(e); if (v >= 1 && v <= 4096) L = v; }
    h->unit_L = (int)L;
    h->u_begin = apply_first_unit(h->row_begin, h->unit_L);
    h->n_units = apply_first_unit(h->row_end, h->unit_L);          // == apply_num_units(nt, L) for row_end == nt
    const int64_t count = h->n_units - h->u_begin;
    h->grid = (int)(count < h->num_sms ? (count > 0 ? count : 1) : h->num_sms);
    h->use_k1 = 1;
    if (const char *e = getenv("BSE_APPLY_K1")) h->use_k1 = atoi(e) != 0;
    if (!h->ws_op) {
        size_t bytes = op_doubles(h) * 8;
        if (h->real_form) bytes += (size_t)4 * h->N * 8 * 16;
        if (cudaMalloc(&h->ws_op, bytes) != cudaSuccess) { cudaGetLastError(); h->ws_op = nullptr; return BSE_ERR_ALLOC; }
        h->ws_op_bytes = bytes;
    }
    return BSE_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// one group of up to 8 operand columns through the tensor-core kernels
// ---------------------------------------------------------------------------------------------------------------------
enum { ROLE_4M = 0, ROLE_3M = 1, ROLE_REAL0 = 2, ROLE_REAL1 = 3 };

struct Term {
    const char *tiles;     // this handle's slice of the store
    int role, pass, set;
};
struct Group {
    int kc = 0;                  // operand / result columns (<= 8; <= 4 for ROLE_4M)
    int n_sets = 0, n_terms = 0;
    PrepSet set[2];              // src, conj_in, kind, pass, sign filled by the caller; images assigned by run_group
    Term term[2];
    double2 *dst[8];
    unsigned neg_conj = 0;
};

template <int ES> static void launch_role(const bse_handle_s *h, int role, const TileParams &p)
{
    switch (role) {
        case ROLE_4M: apply_tiles_kernel<ES, Role4M><<<h->grid, APPLY_THREADS, APPLY_SMEM, h->stream>>>(p); break;
        case ROLE_3M: apply_tiles_kernel<ES, Role3M><<<h->grid, APPLY_THREADS, APPLY_SMEM, h->stream>>>(p); break;
        case ROLE_REAL0: apply_tiles_kernel<ES, RoleReal<0>><<<h->grid, APPLY_THREADS, APPLY_SMEM, h->stream>>>(p); break;
        default: apply_tiles_kernel<ES, RoleReal<1>><<<h->grid, APPLY_THREADS, APPLY_SMEM, h->stream>>>(p); break;
    }
}

static bse_status_t run_group(bse_handle_s *h, Group &g)
{
    const int64_t rows_pad = rows_pad_of(h);
    double *base = (double *)h->ws_op;
    double *Ypad = base + (size_t)rows_pad * 64;
    PrepParams pp;
    pp.n_sets = g.n_sets;
    pp.N = h->N;
    pp.rows_pad = rows_pad;
    pp.Ypad = Ypad;
    for (int q = 0; q < g.n_sets; ++q) {
        double *sb = base + (size_t)rows_pad * 32 * q;
        g.set[q].img_pair = (double2 *)sb;
        g.set[q].img_a = sb + (size_t)rows_pad * 16;
        g.set[q].img_b = sb + (size_t)rows_pad * 24;
        g.set[q].kc = g.kc;
        pp.set[q] = g.set[q];
    }
    if (g.n_sets < 2) pp.set[1] = pp.set[0];
    apply_prep_kernel<<<(unsigned)((rows_pad * 8 + 255) / 256), 256, 0, h->stream>>>(pp);
    for (int i = 0; i < g.n_terms; ++i) {
        const Term &t = g.term[i];
        TileParams p;
        p.tiles = t.tiles - tile_index(h->row_begin, 0) * tile_bytes_es(h->es);   // virtual base of the whole packed store
        p.img_pair = g.set[t.set].img_pair;
        p.img_a = g.set[t.set].img_a;
        p.img_b = g.set[t.set].img_b;
        p.Ypad = Ypad;
        p.nt = h->nt;
        p.kc = g.kc;
        p.pass = t.pass;
        p.L = h->unit_L;
        p.u_begin = h->u_begin;
        p.n_units = h->n_units;
        p.zero = 0;
        if (h->es == ES_C128) launch_role<16>(h, t.role, p);
        else launch_role<8>(h, t.role, p);
    }
    PostParams po;
    po.Ypad = (const double2 *)Ypad;
    po.kc = g.kc;
    po.N = h->N;
    po.neg_conj = g.neg_conj;
    for (int c = 0; c < 8; ++c) po.dst[c] = c < g.kc ? g.dst[c] : nullptr;
    apply_post_kernel<<<(unsigned)((h->N * 8 + 255) / 256), 256, 0, h->stream>>>(po);
    count_launch(2 + g.n_terms);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

// single column through the plain-FMA kernels: y += s * (R x) or s * (C conj x) [real form: mode 0 / 1]; y zeroed by the caller
static bse_status_t run_k1(bse_handle_s *h, const char *tiles, bool real, int pass_or_mode, double sign, const double2 *x, double2 *y)
{
    ApplyParams p;
    p.tiles = tiles - tile_index(h->row_begin, 0) * tile_bytes_es(h->es);
    p.X = x; p.ldx = h->N;
    p.Y = (double *)y; p.ldy = h->N;
    p.N = h->N; p.nt = h->nt; p.kc = 1; p.pass = pass_or_mode; p.sign = sign;
    p.L = h->unit_L; p.u_begin = h->u_begin; p.n_units = h->n_units; p.zero = 0;
    const int g = h->grid;
    cudaStream_t s = h->stream;
    if (!real) {
        if (h->es == ES_C128) apply_tiles_k1_kernel<16, 8><<<g, APPLY_THREADS, APPLY_SMEM, s>>>(p);
        else apply_tiles_k1_kernel<8, 8><<<g, APPLY_THREADS, APPLY_SMEM, s>>>(p);
    } else if (h->es == ES_C128) {
        if (pass_or_mode == 0) apply_tiles_real_k1_kernel<16, 0><<<g, APPLY_THREADS, APPLY_SMEM, s>>>(p);
        else apply_tiles_real_k1_kernel<16, 1><<<g, APPLY_THREADS, APPLY_SMEM, s>>>(p);
    } else {
        if (pass_or_mode == 0) apply_tiles_real_k1_kernel<8, 0><<<g, APPLY_THREADS, APPLY_SMEM, s>>>(p);
        else apply_tiles_real_k1_kernel<8, 1><<<g, APPLY_THREADS, APPLY_SMEM, s>>>(p);
    }
    count_launch();
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

// columns of a group: 5 .. 8 at a time while more than 4 are left (three-product role), else up to 4 (four-product role)
static inline int group_width(int left) { return left > 4 ? (left < 8 ? left : 8) : left; }

// ---------------------------------------------------------------------------------------------------------------------
// the products of this handle's tile rows (no sum over the other slices)
// ---------------------------------------------------------------------------------------------------------------------
bse_status_t apply_tda_local(bse_handle_s *h, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k)
{
    const double2 *X = (const double2 *)dX;
    double2 *Y = (double2 *)dY;
    for (int32_t c0 = 0; c0 < k;) {
        const int kc = group_width(k - c0);
        bse_status_t st;
        if (kc == 1 && h->use_k1) {
            if ((st = zero_block(h, Y + (int64_t)c0 * ldy, ldy, h->N, 1))) return st;
            if ((st = run_k1(h, h->R, false, PASS_HERM, 1.0, X + (int64_t)c0 * ldx, Y + (int64_t)c0 * ldy))) return st;
        } else {
            Group g;
            g.kc = kc;
            g.n_sets = 1;
            g.set[0].kind = kc > 4 ? IMG_3M : IMG_4M;
            g.set[0].pass = PASS_HERM;
            g.set[0].sign = 1.0;
            g.set[0].conj_in = 0;
            for (int c = 0; c < 8; ++c) {
                g.set[0].src[c] = c < kc ? X + (int64_t)(c0 + c) * ldx : nullptr;
                g.dst[c] = c < kc ? Y + (int64_t)(c0 + c) * ldy : nullptr;
            }
            g.n_terms = 1;
            g.term[0] = Term{h->R, kc > 4 ? ROLE_3M : ROLE_4M, PASS_HERM, 0};
            if ((st = run_group(h, g))) return st;
        }
        c0 += kc;
    }
    return BSE_OK;
}

bse_status_t apply_half_local(bse_handle_s *h, int sign, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k)
{
    const double2 *X = (const double2 *)dX;
    double2 *Y = (double2 *)dY;
    // real-form stores hold S = R + C (h->R) and D = R - C (h->C):  P = mode 0 over S + mode 1 over D,  M = mode 0 over D + mode 1 over S
    const char *first = sign > 0 ? h->R : h->C, *second = sign > 0 ? h->C : h->R;
    for (int32_t c0 = 0; c0 < k;) {
        const int left = k - c0;
        const int kc = h->real_form ? (left < 8 ? left : 8) : group_width(left);
        const double2 *x = X + (int64_t)c0 * ldx;
        double2 *y = Y + (int64_t)c0 * ldy;
        bse_status_t st;
        if (kc == 1 && h->use_k1) {
            if ((st = zero_block(h, y, ldy, h->N, 1))) return st;
            if (h->real_form) {
                if ((st = run_k1(h, first, true, 0, 1.0, x, y))) return st;
                if ((st = run_k1(h, second, true, 1, 1.0, x, y))) return st;
            } else {
                if ((st = run_k1(h, h->R, false, PASS_HERM, 1.0, x, y))) return st;
                if ((st = run_k1(h, h->C, false, PASS_SYMC, (double)sign, x, y))) return st;
            }
            c0 += kc;
            continue;
        }
        Group g;
        g.kc = kc;
        for (int c = 0; c < 8; ++c) g.dst[c] = c < kc ? y + (int64_t)c * ldy : nullptr;
        if (h->real_form) {
            g.n_sets = 1;
            g.set[0].kind = IMG_REAL; g.set[0].pass = PASS_HERM; g.set[0].sign = 1.0; g.set[0].conj_in = 0;
            for (int c = 0; c < 8; ++c) g.set[0].src[c] = c < kc ? x + (int64_t)c * ldx : nullptr;
            g.n_terms = 2;
            g.term[0] = Term{first, ROLE_REAL0, 0, 0};
            g.term[1] = Term{second, ROLE_REAL1, 1, 0};
        } else {
            const int kind = kc > 4 ? IMG_3M : IMG_4M, role = kc > 4 ? ROLE_3M : ROLE_4M;
            g.n_sets = 2;
            for (int q = 0; q < 2; ++q) {
                g.set[q].kind = kind;
                g.set[q].pass = q == 0 ? PASS_HERM : PASS_SYMC;
                g.set[q].sign = q == 0 ? 1.0 : (double)sign;
                g.set[q].conj_in = 0;
                for (int c = 0; c < 8; ++c) g.set[q].src[c] = c < kc ? x + (int64_t)c * ldx : nullptr;
            }
            g.n_terms = 2;
            g.term[0] = Term{h->R, role, PASS_HERM, 0};
            g.term[1] = Term{h->C, role, PASS_SYMC, 1};
        }
        if ((st = run_group(h, g))) return st;
        c0 += kc;
    }
    return BSE_OK;
}

// u = (x1 + conj x2) / 2,  v = (x1 - conj x2) / 2
__global__ void split_uv_kernel(const double2 *__restrict__ x1, const double2 *__restrict__ x2, int64_t ldx,
                                double2 *__restrict__ u, double2 *__restrict__ v, int64_t n, int k)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (i < n && c < k) {
        double2 a = x1[i + c * ldx], b = x2[i + c * ldx];
        u[i + c * n] = make_double2(0.5 * (a.x + b.x), 0.5 * (a.y - b.y));
        v[i + c * n] = make_double2(0.5 * (a.x - b.x), 0.5 * (a.y + b.y));
    }
}
// y1 = pu + mv,  y2 = -conj(pu - mv)
__global__ void combine_uv_kernel(const double2 *__restrict__ pu, const double2 *__restrict__ mv, double2 *__restrict__ y1,
                                  double2 *__restrict__ y2, int64_t ldy, int64_t n, int k)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int c = blockIdx.y;
    if (i < n && c < k) {
        double2 a = pu[i + c * n], b = mv[i + c * n];
        y1[i + c * ldy] = make_double2(a.x + b.x, a.y + b.y);
        y2[i + c * ldy] = make_double2(-(a.x - b.x), a.y - b.y);
    }
}

// [Y1; Y2] = H [X1; X2] for this handle's tile rows (Eq. 1 with A = R^*, C = C^T):
//   Y1 = R X1 + C X2,   Y2 = -conj( R conj(X2) + C conj(X1) ).
// Complex stores: ONE pass over R and ONE over C with 2 kk operand columns -- the HERM pass sees [X1 | conj X2], the SYMC pass
// (which conjugates its operand) [conj X2 | X1]; the first kk result columns are Y1, the other kk are stored as -conj.
// Real-form stores: U = (X1 + conj X2)/2, V = (X1 - conj X2)/2, Y1 = P(U) + M(V), Y2 = -conj(P(U) - M(V)).
static bse_status_t apply_general_local(bse_handle_s *h, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k)
{
    const int64_t N = h->N;
    const double2 *X1 = (const double2 *)dX, *X2 = X1 + N;
    double2 *Y1 = (double2 *)dY, *Y2 = Y1 + N;
    bse_status_t st;
    if (h->real_form) {
        double2 *U = (double2 *)((double *)h->ws_op + op_doubles(h)), *V = U + (size_t)N * 8, *PU = V + (size_t)N * 8,
                *MV = PU + (size_t)N * 8;
        for (int32_t c0 = 0; c0 < k; c0 += 8) {
            const int kc = k - c0 < 8 ? k - c0 : 8;
            dim3 grid((unsigned)((N + 255) / 256), (unsigned)kc);
            split_uv_kernel<<<grid, 256, 0, h->stream>>>(X1 + (int64_t)c0 * ldx, X2 + (int64_t)c0 * ldx, ldx, U, V, N, kc);
            count_launch();
            if ((st = apply_half_local(h, +1, U, N, PU, N, kc))) return st;
            if ((st = apply_half_local(h, -1, V, N, MV, N, kc))) return st;
            combine_uv_kernel<<<grid, 256, 0, h->stream>>>(PU, MV, Y1 + (int64_t)c0 * ldy, Y2 + (int64_t)c0 * ldy, ldy, N, kc);
            count_launch();
        }
        BSE_CUDA(cudaGetLastError());
        return BSE_OK;
    }
    for (int32_t c0 = 0; c0 < k;) {
        const int left = k - c0, kk = left < 4 ? left : 4;
        Group g;
        g.kc = 2 * kk;
        const int kind = g.kc > 4 ? IMG_3M : IMG_4M, role = g.kc > 4 ? ROLE_3M : ROLE_4M;
        g.n_sets = 2;
        g.set[0].kind = g.set[1].kind = kind;
        g.set[0].pass = PASS_HERM; g.set[1].pass = PASS_SYMC;
        g.set[0].sign = g.set[1].sign = 1.0;
        g.set[0].conj_in = g.set[1].conj_in = 0;
        for (int c = 0; c < 8; ++c) { g.set[0].src[c] = g.set[1].src[c] = nullptr; g.dst[c] = nullptr; }
        for (int c = 0; c < kk; ++c) {
            const double2 *x1 = X1 + (int64_t)(c0 + c) * ldx, *x2 = X2 + (int64_t)(c0 + c) * ldx;
            g.set[0].src[c] = x1;                                                 // R X1
            g.set[0].src[kk + c] = x2; g.set[0].conj_in |= 1u << (kk + c);        // R conj(X2)
            g.set[1].src[c] = x2; g.set[1].conj_in |= 1u << c;                    // C conj(conj X2) = C X2
            g.set[1].src[kk + c] = x1;                                            // C conj(X1)
            g.dst[c] = Y1 + (int64_t)(c0 + c) * ldy;
            g.dst[kk + c] = Y2 + (int64_t)(c0 + c) * ldy;
            g.neg_conj |= 1u << (kk + c);
        }
        g.n_terms = 2;
        g.term[0] = Term{h->R, role, PASS_HERM, 0};
        g.term[1] = Term{h->C, role, PASS_SYMC, 1};
        if ((st = run_group(h, g))) return st;
        c0 += kk;
    }
    return BSE_OK;
}

bse_status_t apply_vec(bse_handle_s *h, int sign, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k)
{
    const int64_t N = h->N;
    bse_status_t st;
    if (!is_row_partitioned(h)) {
        st = sign == 0 ? apply_tda_local(h, dX, ldx, dY, ldy, k) : apply_half_local(h, sign, dX, ldx, dY, ldy, k);
        if (st) return st;
        return comm_sum_block(h, dY, ldy, N, k);
    }
    // row-partitioned vectors: all-gather of the operand block as a zero-padded sum, product with this rank's tile rows,
    // sum of the partial results, this rank's rows copied out (2 x 16 N k bytes through the hook per product)
    if (!h->comm) return BSE_ERR_INVALID_ARG;
    const size_t need = (size_t)2 * N * k * 16;
    if (h->rp_buf_bytes < need) {
        if (h->rp_buf) cudaFree(h->rp_buf);
        h->rp_buf = nullptr;
        h->rp_buf_bytes = 0;
        if (cudaMalloc(&h->rp_buf, need) != cudaSuccess) { cudaGetLastError(); return BSE_ERR_ALLOC; }
        h->rp_buf_bytes = need;
    }
    char *Xf = (char *)h->rp_buf, *Yf = Xf + (size_t)N * k * 16;
    const int64_t rows = vec_rows(h);
    BSE_CUDA(cudaMemsetAsync(Xf, 0, (size_t)N * k * 16, h->stream));
    BSE_CUDA(cudaMemcpy2DAsync(Xf + (size_t)h->vr_begin * 16, (size_t)N * 16, dX, (size_t)ldx * 16, (size_t)rows * 16, (size_t)k,
                               cudaMemcpyDeviceToDevice, h->stream));
    if ((st = comm_sum_block(h, Xf, N, N, k))) return st;
    st = sign == 0 ? apply_tda_local(h, Xf, N, Yf, N, k) : apply_half_local(h, sign, Xf, N, Yf, N, k);
    if (st) return st;
    if ((st = comm_sum_block(h, Yf, N, N, k))) return st;
    BSE_CUDA(cudaMemcpy2DAsync(dY, (size_t)ldy * 16, Yf + (size_t)h->vr_begin * 16, (size_t)N * 16, (size_t)rows * 16, (size_t)k,
                               cudaMemcpyDeviceToDevice, h->stream));
    return BSE_OK;
}

}  // namespace bse

using namespace bse;

extern "C" {

bse_status_t bse_apply(bse_handle_t h, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k)
{
    if (!h || !dX || !dY || k < 1 || dX == dY) return BSE_ERR_INVALID_ARG;
    const int64_t N = h->N;
    if (h->mode == BSE_MODE_TDA) {
        if (ldx < N || ldy < N) return BSE_ERR_INVALID_ARG;
        bse_status_t st = apply_tda_local(h, dX, ldx, dY, ldy, k);
        if (st) return st;
        return comm_sum_block(h, dY, ldy, N, k);
    }
    if (ldx < 2 * N || ldy < 2 * N) return BSE_ERR_INVALID_ARG;
    bse_status_t st = apply_general_local(h, dX, ldx, dY, ldy, k);
    if (st) return st;
    return comm_sum_block(h, dY, ldy, 2 * N, k);
}

bse_status_t bse_apply_half(bse_handle_t h, int32_t sign, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k)
{
    if (!h || !dX || !dY || k < 1 || ldx < h->N || ldy < h->N || (sign != 1 && sign != -1) || dX == dY) return BSE_ERR_INVALID_ARG;
    if (h->mode != BSE_MODE_FULL) return BSE_ERR_INVALID_ARG;
    bse_status_t st = apply_half_local(h, sign, dX, ldx, dY, ldy, k);
    if (st) return st;
    return comm_sum_block(h, dY, ldy, h->N, k);
}

bse_status_t bse_apply_host(bse_handle_t h, const void *hX, int64_t ldx, void *hY, int64_t ldy, int32_t k)
{
    if (!h || !hX || !hY || k < 1) return BSE_ERR_INVALID_ARG;
    const int64_t n = (h->mode == BSE_MODE_FULL) ? 2 * h->N : h->N;
    if (ldx < n || ldy < n) return BSE_ERR_INVALID_ARG;
    bse_status_t st = ensure_ws2(h, (size_t)2 * n * k * 16);
    if (st) return st;
    char *dX = (char *)h->ws2, *dY = dX + (size_t)n * k * 16;
    BSE_CUDA(cudaMemcpy2DAsync(dX, (size_t)n * 16, hX, (size_t)ldx * 16, (size_t)n * 16, (size_t)k,
                               cudaMemcpyHostToDevice, h->stream));
    st = bse_apply(h, dX, n, dY, n, k);
    if (st) return st;
    BSE_CUDA(cudaMemcpy2DAsync(hY, (size_t)ldy * 16, dY, (size_t)n * 16, (size_t)n * 16, (size_t)k,
                               cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    return BSE_OK;
}

}  // extern "C"
