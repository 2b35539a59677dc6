// Internal declarations shared by the translation units of libbse_b200.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <atomic>
#include <cstdio>
#include <cstdlib>

#include "../../include/bse.h"

struct bse_handle_s {
    int32_t mode;
    int64_t N;
    int nt;
    int es;              // bytes per stored complex entry: 16 (BSE_STORE_C128) or 8 (BSE_STORE_C64)
    int row_begin, row_end;   // tile rows [row_begin, row_end) this handle's stores hold (0, nt unless created by bse_create_shard)
    bse_comm_fn comm;    // bse_set_comm: sum / broadcast over the ranks that hold the other slices (NULL: none)
    void *comm_user;
    void *comm_buf;      // device staging for host-side broadcasts
    size_t comm_buf_bytes;
    // bse_set_row_partition: the solver-level calls hold rows [vr_begin, vr_end) of every vector (0, N: replicated vectors)
    int64_t vr_begin, vr_end;
    void *rp_buf;        // full-length operand and result blocks of a row-partitioned product
    size_t rp_buf_bytes;
    int real_form;       // BSE_STORE_REAL_FORM: R holds S = R + C, C holds D = R - C (full mode only, complex128)
    const char *R;
    const char *C;
    cudaStream_t stream;
    int num_sms;
    // apply kernels: unit walk of this handle's tile rows and the operand workspace (images + Ypad, apply_prep.cuh),
    // all fixed by handle_finalize at creation: the apply calls themselves never allocate and read no environment
    int unit_L;
    int64_t u_begin, n_units;
    int grid;
    int use_k1;          // single columns take the plain-FMA kernels (BSE_APPLY_K1=0 at creation: tensor-core kernels)
    void *ws_op;
    size_t ws_op_bytes;
    // lazily grown scratch (device)
    void *ws;
    size_t ws_bytes;
    // second scratch used by the solver / orth (device)
    void *ws2;
    size_t ws2_bytes;
    // pinned host staging for small results
    void *hpin;
    size_t hpin_bytes;
};

namespace bse {

// a handle created by bse_create_shard over part of the tile rows: apply / apply_half only
inline bool is_partial(const bse_handle_s *h) { return h->row_begin != 0 || h->row_end != h->nt; }
// partial handle that cannot complete its products: the solver-level calls refuse it
inline bool is_incomplete(const bse_handle_s *h) { return is_partial(h) && !h->comm; }
// vectors of the solver-level calls partitioned by rows over the ranks behind the hook
inline bool is_row_partitioned(const bse_handle_s *h) { return h->vr_begin != 0 || h->vr_end != h->N; }
inline int64_t vec_rows(const bse_handle_s *h) { return h->vr_end - h->vr_begin; }
// communication through the hook (no-ops without one).  ld, rows in complex elements.
bse_status_t comm_sum_block(bse_handle_s *h, void *dY, int64_t ld, int64_t rows, int k);
bse_status_t comm_bcast_dev(bse_handle_s *h, void *dBuf, int64_t n_doubles);
bse_status_t comm_sum_dev(bse_handle_s *h, void *dBuf, int64_t n_doubles);
bse_status_t comm_bcast_host(bse_handle_s *h, void *hBuf, size_t bytes);

extern std::atomic<int64_t> g_launches;
inline void count_launch(int n = 1) { g_launches.fetch_add(n, std::memory_order_relaxed); }

// BSE_VERBOSE=1 prints the failing CUDA call (status codes alone cannot say which one it was)
#define BSE_CUDA(call)                                                                                   \
    do {                                                                                                 \
        cudaError_t e__ = (call);                                                                        \
        if (e__ != cudaSuccess) {                                                                        \
            if (getenv("BSE_VERBOSE"))                                                                   \
                fprintf(stderr, "[bse] %s:%d %s -> %s\n", __FILE__, __LINE__, #call, cudaGetErrorString(e__)); \
            return BSE_ERR_CUDA;                                                                         \
        }                                                                                                \
    } while (0)

bse_status_t ensure_ws(bse_handle_s *h, size_t bytes);
bse_status_t ensure_ws2(bse_handle_s *h, size_t bytes);
bse_status_t ensure_pin(bse_handle_s *h, size_t bytes);

// unit walk parameters and operand workspace of a handle (bse_create / bse_create_shard)
bse_status_t handle_finalize(bse_handle_s *h);
// The products of this handle's tile rows WITHOUT the sum over the other slices (callers add comm_sum_block):
//   apply_tda_local : Y = R X                       (N x k, TDA handles)
//   apply_half_local: Y = R X + sign C conj(X)      (N x k, full-mode handles; complex or real-form stores)
bse_status_t apply_tda_local(bse_handle_s *h, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k);
bse_status_t apply_half_local(bse_handle_s *h, int sign, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k);
bse_status_t zero_block(bse_handle_s *h, void *dY, int64_t ldy, int64_t rows, int32_t k);
// The COMPLETE product on this handle's vector rows, as the solver-level calls need it: sign = 0: Y = R X (TDA), +-1:
// Y = R X + sign C conj(X).  Replicated vectors: local product + sum over the slices.  Row-partitioned vectors (X, Y hold
// rows [vr_begin, vr_end)): the operand block is gathered (zero-padded sum), multiplied by this rank's tile rows, summed, and
// this rank's rows of the result are copied out.
bse_status_t apply_vec(bse_handle_s *h, int sign, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k);


// ---- dense basis kernels (dense_ops.cu).  Complex blocks are column-major; *_cplx selects complex coefficients.
// out (device, doubles): coefficient matrix in the layout gemm_basis consumes: out[a + half*m + col*ldo],
// ldo = cplx ? 2m : m, half = 0 (real part) / 1 (imaginary part).  out is zeroed first.
bse_status_t gram_basis(bse_handle_s *h, const void *A, int64_t lda, int m, const void *B, int64_t ldb, int k,
                        bool cplx, int64_t n, double *out);
// C(n x l) = alpha * A(n x m) * S + beta * C,  S given as coefficient matrix `coef` (layout above, ld = ldo).
// a_upper: A~ (real view) is upper triangular, A~[row, col] = 0 for col < row: the zero part of the contraction is skipped;
// c_lower: only the lower triangle of the (square) C~ is wanted: tiles above the diagonal are left alone
bse_status_t gemm_basis(bse_handle_s *h, const void *A, int64_t lda, int m, bool cplx, const double *coef,
                        int64_t ldo, int l, int64_t n, void *C, int64_t ldc, double alpha, double beta, bool a_upper = false,
                        bool c_lower = false);
bse_status_t fill_random_block(bse_handle_s *h, void *W, int64_t ldw, int64_t n, int k, uint64_t seed,
                               uint64_t counter);
bse_status_t copy_block(bse_handle_s *h, const void *src, int64_t lds, void *dst, int64_t ldd, int64_t n, int k);
// dst[a + col*m] (complex) = c1 + c2 in coefficient layout (c2 may be NULL)
bse_status_t coef_to_complex(bse_handle_s *h, const double *c1, const double *c2, int m, int k, bool cplx,
                             void *dst);
// v (2N x nev) from x, px (N x nev each): v = [x + px/w; conj(x - px/w)] * sqrt(w)/2   (reading S4)
bse_status_t assemble_full_vectors(bse_handle_s *h, const void *x, const void *px, int64_t N, int nev,
                                   const double *d_omega, void *vec, int64_t ldvec);

// orthogonalisation core shared by bse_orth and bse_solve (bse_orth.cu).  hcoef_host: m x k complex (ld m),
// bfac_host: k x k complex (ld k); both host, nullable.  rng_counter advances when columns are replaced.
bse_status_t orth_block(bse_handle_s *h, const void *V, int64_t ldv, int m, const void *PV, int64_t ldpv, void *W,
                        int64_t ldw, int k, void *PW, int64_t ldpw, void *hcoef_host, void *bfac_host, int *rank,
                        uint64_t seed, uint64_t *rng_counter);

bse_status_t orth_reserve(bse_handle_s *h, int m_max, int k);
// The pieces of orth_block, for callers that recompute P(W) between projection and normalisation.  All asynchronous on the
// handle's stream except normalize_block, which ends with the block step's ONE host synchronisation and hands back the
// projection coefficients h1 + h2 (hcoef_host, m x k, out), the k x k factor and the rank.  Device scalar slots of
// block_norm_scale: ORTH_E_IN (opens a block step: clears the flags), ORTH_E_AFTER, ORTH_G; normalize_block's scale_mode 0
// takes the incoming block's norm scale from ORTH_E_IN (same inner product), 1 from ORTH_G * ORTH_E_IN / ORTH_E_AFTER.
enum { ORTH_E_IN = 0, ORTH_E_AFTER = 1, ORTH_G = 2 };
bse_status_t project_block(bse_handle_s *h, const void *V, int64_t ldv, int m, const void *PV, int64_t ldpv, void *W,
                           int64_t ldw, int k, void *PW, int64_t ldpw, bool cplx);
bse_status_t block_norm_scale(bse_handle_s *h, const void *W, int64_t ldw, const void *PW, int64_t ldpw, int k,
                              bool cplx, int slot);
bse_status_t normalize_block(bse_handle_s *h, const void *V, int64_t ldv, int m, const void *PV, int64_t ldpv, void *W,
                             int64_t ldw, int k, void *PW, int64_t ldpw, bool cplx, int scale_mode, void *hcoef_host,
                             void *bfac_host, int *rank_out, uint64_t seed, uint64_t *rng_counter, int image_sign = +1);
// (image_sign: which half apply gives the image PW of a replacement column in the real inner product: +1 P, -1 M)

// host eigensolver (host_eig.cpp)
int host_heev(int m, void *A, int lda, double *w, void *Z, int ldz, int nz);
// real symmetric variant (full mode's projected matrix): A, Z real
int host_syev(int m, double *A, int lda, double *w, double *Z, int ldz, int nz);
// real symmetric tridiagonal (d, e): all eigenvalues ascending, eigenvectors of the nz lowest
int host_stev(int m, double *d, double *e, double *w, double *Z, int ldz, int nz);
// the nz lowest eigenpairs only (w: nz values; Z nullable): bisection + inverse iteration when nz is a small part of m
int host_stev_lowest(int m, double *d, double *e, int nz, double *w, double *Z, int ldz);

}  // namespace bse
