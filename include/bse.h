/*
 * bse.h -- C ABI of the B200-native BSE hot path (arXiv 2504.10096, iterative solution).
 *
 * What the library computes (citations are PAPER.md line + equation/section):
 *   * the structured operator of Eq. (1) in the optical case A = R^*, C = C^T
 *      applied to a block of k vectors -- "the most expensive step ... are the
 *     matrix-vector products";  TDA: C = 0, Y = R X with R Hermitian;
 *   * block classical Gram-Schmidt with reorthogonalisation of new vectors against the stored
 *     Krylov basis;
 *   * thick-restart Lanczos: Hermitian for TDA, structure-preserving (works on H^2 with the lower
 *     blocks of matrix and basis implicit, final step recovers +omega and eigenvectors) for the
 *     full case.
 *
 * Conventions
 *   - every pointer named d* is a DEVICE pointer in the caller's current CUDA context, every pointer
 *     named h* is a HOST pointer; complex128 = interleaved (re, im) doubles, 16-byte aligned;
 *   - dense matrices and vector blocks are COLUMN-MAJOR with an explicit leading dimension
 *     (in complex elements);  sizes are int64_t / int32_t;
 *   - all device work is enqueued on the `stream` given to bse_create (a cudaStream_t passed as
 *     void*; NULL = the legacy default stream).  bse_apply / bse_apply_half / bse_gram / bse_update are
 *     asynchronous with respect to the host; bse_orth synchronises the stream once (it returns the rank on the host; the
 *     k x k factorisations run on the device); bse_solve, bse_lanczos_quadrature and the *_host calls are synchronous;
 *   - bse_apply / bse_apply_half only enqueue kernel launches (and a memset for single columns) into a workspace sized at
 *     bse_create: they allocate nothing, read no environment variable (BSE_APPLY_UNIT, BSE_APPLY_K1 are read once, at
 *     bse_create) and can be captured in a CUDA graph on the handle's stream and replayed, for any mode, store and k
 *     (tests/test_gpu_apply.py).  Not once bse_set_comm is active: the calls then issue collectives through the hook;
 *   - no call throws or exits; every call returns a bse_status_t;
 *   - there is no CPU fallback: without a CUDA device every compute call returns BSE_ERR_CUDA.
 *
 * Packed triangular tile storage (north_star: "R lower triangle ... stored as packed triangular
 * tiles").  With TB = 64 and nt = ceil(N / 64), a matrix is nt (nt + 1) / 2 tiles of 64 x 64
 * complex128 (65536 bytes each, contiguous); tile (I, J), J <= I, is tile number I (I + 1) / 2 + J.
 * Rows/columns >= N of the last tile row are zero.  Diagonal tiles are stored in full, the strictly
 * upper part holding the Hermitian (R) or symmetric (C) mirror image; the diagonal of R is real.
 * Inside a tile the 64 x 64 entries are ordered in 8 x 8 patches, patch (ib, jb) at byte
 * (jb * 8 + ib) * 1024, entry (a, b) of a patch at slot
 *     ((a>>2)<<2 | (b>>2)<<1 | (a>>1 & 1)) * 8 + ((a&1)<<2 | (b&1)<<1 | ((a>>1 ^ b>>1) & 1))
 * of 16 bytes -- the order in which the FP64 tensor-core fragments of the apply kernel read it
 * from shared memory without bank conflicts, both as T and as T^H.  The layout is opaque to
 * callers: fill it with bse_pack_from_dense / bse_fill_synthetic / bse_fill_closed_form_*.
 *
 * Storage type (`storage` argument): BSE_STORE_C128 keeps the entries as complex128 (the layout
 * above).  BSE_STORE_C64 keeps each entry as two IEEE binary32 values (the paper's matrices are
 * single precision, PAPER.md:111 and the caption of Table 2): every size above
 * halves (32768-byte tiles, 512-byte patches, 8-byte slots, same order), entries are rounded to
 * nearest-even when the store is written, and the operator every later call works with IS the
 * rounded matrix: fragments are widened to FP64 on load and all arithmetic, vectors and results
 * stay complex128.  Half the HBM bytes per apply, twice the N per GPU.
 * BSE_STORE_REAL_FORM (full mode, bse_layout and bse_create only): the two complex128 stores hold S = R + C and
 * D = R - C -- the blocks Re(R+C), Im(R+C), Re(R-C), Im(R-C) of the real symmetric M_r of Eq. (3) --
 * written by bse_to_real_form from stores of R and C.  The half applies then run in real arithmetic,
 * P(x): re = Sr a - Di b, im = Si a + Dr b;  M(x): re = Dr a - Si b, im = Di a + Sr b  (x = a + i b),
 * with half the flops of the complex form; every result is the same operator's to rounding.
 * BSE_STORE_REAL_FORM_C64: the same with binary32 planes, written by bse_to_real_form from BSE_STORE_C64 stores:
 * S32 = fl32(R32 + C32), D32 = fl32(R32 - C32) (exact sum, one rounding to nearest-even).  The operator every later
 * call works with is then R' = (S32 + D32)/2, C' = (S32 - D32)/2 (exact in FP64) -- within one binary32 ulp of the
 * single-precision R32, C32, i.e. inside the precision of the data; arithmetic stays FP64.
 */
#ifndef BSE_B200_H
#define BSE_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bse_handle_s *bse_handle_t;

typedef enum {
    BSE_OK = 0,
    BSE_ERR_INVALID_ARG = 1,
    BSE_ERR_CUDA = 2,               /* a CUDA runtime call failed (or no device)                  */
    BSE_ERR_ALLOC = 3,
    BSE_ERR_NOT_CONVERGED = 4,      /* bse_solve: outputs hold the best estimates, see info.nconv */
    BSE_ERR_NOT_POSITIVE_DEFINITE = 5, /* full mode: Re(w^H P(w)) <= 0 met (PAPER.md:49 precondition) */
    BSE_ERR_INTERNAL = 6,
    BSE_ERR_STATIC_LIMIT = 7        /* bse_lanczos_quadrature_static: N or steps beyond the fixed scratch array */
} bse_status_t;

enum { BSE_MODE_TDA = 0, BSE_MODE_FULL = 1 };
enum { BSE_MATRIX_R = 0, BSE_MATRIX_C = 1 };
enum { BSE_STORE_C128 = 0, BSE_STORE_C64 = 1, BSE_STORE_REAL_FORM = 2, BSE_STORE_REAL_FORM_C64 = 3 };

typedef struct {
    int32_t n_apply;        /* operator applications (block applies; a full-mode step counts 2 half applies) */
    int32_t n_restart;      /* thick restarts performed                                                   */
    int32_t nconv;          /* wanted Ritz pairs that met the tolerance                                    */
    int32_t ncv;            /* basis size used                                                              */
    double  seconds_apply, seconds_orth, seconds_project, seconds_restart, seconds_total;
                            /* apply: every operator application (in full mode both half applies of a step, also the
                               P(W) that follows the projection); orth: projection + normalisation only            */
    double  norm_est;       /* estimate of ||H|| (largest |Ritz value| seen; sqrt of it in full mode)      */
    double  basis_orth_err; /* || <V, V> - I ||_F of the final Krylov basis in the active inner product:
                               V^H V (TDA) or Re(X^H P(X)) (full mode, reading S10); north_star bound 1e-12    */
} bse_info_t;

const char *bse_status_string(bse_status_t s);

/* Tile geometry for an N x N matrix: *tile = 64, *n_tiles = nt (nt+1)/2, *bytes = n_tiles * 65536
 * (BSE_STORE_C128) or n_tiles * 32768 (BSE_STORE_C64).  N < 1 or an unknown storage ->
 * BSE_ERR_INVALID_ARG (every call below with a `storage` argument rejects unknown values the same
 * way).  Output pointers may be NULL. */
bse_status_t bse_layout(int64_t N, int32_t storage, int32_t *tile, int64_t *n_tiles,
                        int64_t *bytes_per_matrix);

/* dTiles <- lower triangle of the dense column-major N x N matrix dDense (leading dimension ld);
 * which = BSE_MATRIX_R (Hermitian: mirror is the conjugate, diagonal imaginary part dropped) or
 * BSE_MATRIX_C (symmetric: mirror is a copy).  Only entries (i, j) with j <= i are read.  dDense is
 * complex128 for both storage types. */
bse_status_t bse_pack_from_dense(const void *dDense, int64_t ld, int64_t N, int32_t which,
                                 void *dTiles, int32_t storage, void *stream);

/* dDense (column-major, ld) <- the full N x N matrix the tiles represent (both triangles). Test helper. */
bse_status_t bse_unpack_to_dense(const void *dTiles, int32_t storage, int64_t N, int32_t which,
                                 void *dDense, int64_t ld, void *stream);

/* The synthetic "BSE-shaped" generator of BASELINE.json, evaluated on the device
 * with the same counter-based generator as bse_inputs/ (matches it to a few ulp):
 *   R = diag(d_eps + sigma) + K,  K_ij = 0.1 (g1 + i g2) / (1 + |i-j|/64), d_eps ~ U[1,10] sorted in
 *   groups of `group` indices;  C_ij = C_ji = 0.05 (g1 + i g2) / (1 + |i-j|/64).
 * N % group != 0 -> BSE_ERR_INVALID_ARG (which = R only). */
bse_status_t bse_fill_synthetic(void *dTiles, int32_t storage, int64_t N, int32_t which, uint64_t seed,
                                double sigma, int32_t group, void *stream);

/* Closed-form instance with a prescribed spectrum: R = Q diag(lam) Q^H, Q = I - 2 u u^H,
 *   R_ij = lam_i d_ij - 2 u_i conj(u_j) (lam_i + lam_j - 2 s),  s = sum_l lam_l |u_l|^2.
 * dLam: N doubles (device), dU: N complex128 (device, unit 2-norm).  which=BSE_MATRIX_R only. */
bse_status_t bse_fill_closed_form_tda(void *dTiles, int32_t storage, int64_t N, const double *dLam,
                                      const void *dU, double s, void *stream);

/* Closed-form pair with omega_i = sqrt(d1_i d2_i): M+- = Q diag(d1|d2) Q^T (real Householder, dUr real
 * unit vector), R = U (M+ + M-)/2 U^H, C = U (M+ - M-)/2 U^T, U = diag(exp(i phi)).
 * All inputs are device arrays of N doubles; s1 = sum d1 u^2, s2 = sum d2 u^2. */
bse_status_t bse_fill_closed_form_full(void *dRTiles, void *dCTiles, int32_t storage, int64_t N,
                                       const double *dD1, const double *dD2, const double *dUr,
                                       const double *dPhi, double s1, double s2, void *stream);

/* Creates a handle.  BORROWS dRTiles (and dCTiles in full mode): the caller keeps them alive and
 * unmodified until bse_destroy.  mode = BSE_MODE_TDA (dCTiles ignored, may be NULL) or BSE_MODE_FULL
 * (dCTiles required); `storage` is the type both stores were written with.  Does not verify
 * Hermitian / symmetric / positive-definite structure.  Workspace O(N k) is allocated lazily by
 * later calls with cudaMalloc. */
bse_status_t bse_create(bse_handle_t *h, int32_t mode, int32_t storage, int64_t N, const void *dRTiles,
                        const void *dCTiles, void *stream);
bse_status_t bse_destroy(bse_handle_t h);

/* In place, on two stores (or two slices of stores, see bse_shard_layout) of n_tiles tiles each and the same
 * `storage` (BSE_STORE_C128 or BSE_STORE_C64):  dRTiles <- S = R + C,
 * dCTiles <- D = R - C (every stored entry, mirrored halves and padding included; binary32 planes are summed exactly
 * and rounded once).  Afterwards pass both to bse_create with BSE_STORE_REAL_FORM / BSE_STORE_REAL_FORM_C64 (mode
 * FULL); they no longer represent R and C for any other call.  Asynchronous on `stream`. */
bse_status_t bse_to_real_form(void *dRTiles, void *dCTiles, int32_t storage, int64_t n_tiles, void *stream);

/* ---- Sharding of the tile stream (the paper partitions matrices by rows). ----
 * The packed store is ordered by tile row, so a range of tile rows [tile_row_begin, tile_row_end) is one contiguous
 * slice of it.  bse_shard_layout splits the nt tile rows into n_shards ranges of (nearly) equal TILE COUNT
 * (boundary r = the smallest I with I (I+1)/2 >= r * total / n_shards) and reports, for `shard`, the range, the number
 * of its first tile in the whole store, its tile count and its size in bytes.  Output pointers may be NULL. */
bse_status_t bse_shard_layout(int64_t N, int32_t storage, int32_t n_shards, int32_t shard, int32_t *tile_row_begin,
                              int32_t *tile_row_end, int64_t *first_tile, int64_t *n_tiles, int64_t *bytes);

/* bse_fill_synthetic for one slice: dTiles points at the slice (tile row tile_row_begin, column 0 first). */
bse_status_t bse_fill_synthetic_shard(void *dTiles, int32_t storage, int64_t N, int32_t which, uint64_t seed,
                                      double sigma, int32_t group, int32_t tile_row_begin, int32_t tile_row_end,
                                      void *stream);

/* A handle over ONE slice: dRSlice (and dCSlice) hold only the tiles of tile rows [tile_row_begin, tile_row_end).
 * bse_apply and bse_apply_half on such a handle compute this slice's CONTRIBUTION to Y -- rows of the slice's tile rows
 * from T X (P1) and rows of all tile columns J <= I from T^H X (P2) -- over the full length N: the sum over the
 * shards of a partition is Y = H X.  X must be the whole block on every shard (16 N k bytes); the partial Y are
 * summed by the caller (one all-reduce of 16 N k bytes per apply over NVLink when shards live on different GPUs:
 * paper_2504_10096_b200.ShardedBse).  bse_solve, bse_orth and bse_lanczos_quadrature need the whole operator and
 * return BSE_ERR_INVALID_ARG on a partial handle that has no communication hook (bse_set_comm).  The general FULL-mode bse_apply is real-linear in the stores as
 * well (its elementwise pre/post steps commute with the sum), for every storage type. */
bse_status_t bse_create_shard(bse_handle_t *h, int32_t mode, int32_t storage, int64_t N, int32_t tile_row_begin,
                              int32_t tile_row_end, const void *dRSlice, const void *dCSlice, void *stream);

/* Communication hook for partial handles (one process per GPU; the library itself links no communication library).
 * fn(user, op, dBuf, n_doubles) must, on the handle's stream order, either
 *   BSE_COMM_SUM  : replace dBuf[0 .. n_doubles) (device, FP64) by its sum over all ranks (an all-reduce), or
 *   BSE_COMM_BCAST: replace it by rank 0's copy (a broadcast),
 * and return 0 (anything else aborts the calling library function with BSE_ERR_INTERNAL).  With a hook installed
 *   - bse_apply / bse_apply_half on a partial handle return the COMPLETE product (local contribution + one SUM of
 *     16 N k bytes);
 *   - bse_solve and bse_lanczos_quadrature run on partial handles: every rank executes the same host loop on
 *     replicated vectors; each operator application is summed over the ranks, and every quantity the kernels
 *     accumulate with floating-point atomics (projection coefficients, Gram matrices, recurrence scalars) as well as
 *     the projected eigen-decomposition is broadcast from rank 0 before it is used, so that all ranks hold bitwise
 *     identical bases and take identical decisions (same number of steps and restarts: no rank can fall out of the
 *     collective sequence).  Vectors, orthogonalisation and restart are replicated (O(N ncv) per rank), the O(N^2)
 *     tile stream is divided.
 * fn = NULL removes the hook.  The hook is called from the thread that called the library function. */
typedef int32_t (*bse_comm_fn)(void *user, int32_t op, void *dBuf, int64_t n_doubles);
enum { BSE_COMM_SUM = 0, BSE_COMM_BCAST = 1 };
bse_status_t bse_set_comm(bse_handle_t h, bse_comm_fn fn, void *user);

/* Vectors partitioned by rows as well ("the matrices and vectors are distributed by rows"): after this call the
 * solver-level calls bse_solve / bse_solve_variant(BSE_VARIANT_SHAO) and bse_orth treat every vector block they are given or
 * hold as rows [row_begin, row_end) of the full-length block (leading dimensions >= row_end - row_begin).  Needs a hook
 * (bse_set_comm) and disjoint row ranges that cover [0, N) over the ranks.  Then
 *   - the Krylov bases, the Gram / update / rotation kernels and the restart work on the local rows only (O(N ncv / G) memory
 *     and work per rank); every Gram matrix and norm is the SUM over the ranks (one BSE_COMM_SUM of the small matrix);
 *   - every operator application gathers the operand block (a zero-padded SUM of 16 N k bytes), multiplies it by this rank's
 *     tile rows, sums the partial results and keeps its own rows (two SUMs of 16 N k bytes per product);
 *   - start and replacement vectors are functions of the GLOBAL row index (the partitioned block is the slice of the
 *     replicated one); the projected eigen-decomposition is still rank 0's, broadcast;
 *   - bse_solve returns the eigenvectors at FULL length on every rank (dVec N x nev / 2N x nev, gathered at the end).
 * bse_apply / bse_apply_half keep taking full-length blocks.  row_begin = 0, row_end = N restores replicated vectors.
 * Errors: BSE_ERR_INVALID_ARG (empty or out-of-range rows); the solver calls return BSE_ERR_INVALID_ARG on a row-partitioned
 * handle without a hook, and bse_lanczos_quadrature*, bse_solve_direct and BSE_VARIANT_GRUNING do not take one. */
bse_status_t bse_set_row_partition(bse_handle_t h, int64_t row_begin, int64_t row_end);

/* Y = H X for a block of k >= 1 vectors.
 *   TDA : X, Y are N x k;   Y = R X.
 *   FULL: X, Y are 2N x k, rows [X1; X2];  Y1 = R X1 + C X2,  Y2 = -(C^H X1 + R^* X2).
 * X and Y must not alias.  Asynchronous on the handle's stream.  TDA: each stored tile of R is read from HBM once
 * per group of up to 8 columns (one column: plain-FMA kernel; 2..4: four real products per complex product on the
 * FP64 tensor cores; 5..8: three).  FULL: four such passes per group (R and C, twice), or two half applies on a
 * real-form store.  On a partial handle (bse_create_shard) the result is that slice's contribution, or the complete
 * product when a communication hook is installed (bse_set_comm). */
bse_status_t bse_apply(bse_handle_t h, const void *dX, int64_t ldx, void *dY, int64_t ldy, int32_t k);

/* FULL mode only, N-row half vectors:  Y = R X + sign * C conj(X),  sign = +1 (P) or -1 (M).
 * This is the upper half of H [x; sign*conj(x)] -- "working implicitly with the lower blocks of the
 * matrix and vector basis".  The structured solver uses only this call. */
bse_status_t bse_apply_half(bse_handle_t h, int32_t sign, const void *dX, int64_t ldx, void *dY,
                            int64_t ldy, int32_t k);

/* Same as bse_apply with HOST buffers (pageable or pinned): copies X to the device, applies, copies
 * Y back and synchronises the stream.  The end-to-end entry point measured by bench.py's "e2e". */
bse_status_t bse_apply_host(bse_handle_t h, const void *hX, int64_t ldx, void *hY, int64_t ldy, int32_t k);

/* Block classical Gram-Schmidt with one reorthogonalisation, then orthonormalises
 * the block in place:   W_in = V hcoef + W_out Bfac,   <V, W_out> = 0,  <W_out, W_out> = I.
 *   dV   : n x m basis (m >= 0), orthonormal in the inner product below; ldv
 *   dBV  : NULL -> Euclidean complex inner product <x, y> = x^H y (TDA);
 *          else the n x m block P(V) and the REAL inner product <x, y> = Re(x^H P(y)) with real
 *          coefficients (full mode, reading S4); then dBW (n x k, = P(W) on entry) is
 *          required and is updated by the same linear combination as W, so dBW_out = P(W_out) up
 *          to kappa(W_in) * eps: for an ill-conditioned block re-apply P afterwards (bse_solve
 *          does, reading R3);
 *   dW   : n x k block, overwritten with the orthonormalised block;
 *   dHcoef: m x k (ld = m) device output, complex128 (imaginary parts 0 in the real case), nullable;
 *   dBfac : k x k (ld = k) device output, upper triangular, positive real diagonal, nullable;
 *   hRank : host int, numerical rank of the block; columns found dependent (diagonal of Bfac below
 *           1e-13 * the largest column norm of W_in) are replaced by orthonormalised pseudo-random
 *           vectors and their Bfac row/column entries set to 0.  Reading it synchronises the stream.
 * n is N for both modes (half vectors in full mode). Returns BSE_ERR_NOT_POSITIVE_DEFINITE if a
 * P-norm is not positive. */
bse_status_t bse_orth(bse_handle_t h, const void *dV, int64_t ldv, int32_t m, const void *dBV,
                      int64_t ldbv, void *dW, int64_t ldw, int32_t k, void *dBW, int64_t ldbw,
                      void *dHcoef, void *dBfac, int32_t *hRank);

/* Thick-restart block Lanczos.
 *   TDA : the nev algebraically smallest eigenvalues of R, ascending, and orthonormal eigenvectors
 *         (N x nev, column-major, ldvec) in dVec.
 *   FULL: the nev smallest positive omega of H, ascending, and right eigenvectors [X_I; Y_I]
 *         (2N x nev) normalised X^H X - Y^H Y = 1.  The -omega partner is [conj(Y); conj(X)].
 *   k    : block size (>= 1; >= 2 recommended in full mode);  ncv: maximum basis
 *          size, 0 -> default max(2 nev, nev + 15) (doubled in full mode) and at least (wanted Ritz values) + 8 k,
 *          rounded up to a multiple of k;
 *   tol  : a Ritz pair is converged when ||H v - w v||_2 <= tol * ||H||_est * ||v||_2 (accepted at 0.9 of that: ||H||_est is a
 *          lower bound of ||H||; reading S7).  TDA: converged leading pairs are locked at restarts (kept in the basis,
 *          left out of the projected eigenproblem);
 *   hOmega: nev doubles (host);  hResid: nev doubles (host, nullable): the residual estimates;
 *   info : nullable.
 * Synchronous.  Errors: BSE_ERR_NOT_CONVERGED after max_restarts, BSE_ERR_NOT_POSITIVE_DEFINITE,
 * BSE_ERR_INVALID_ARG (nev < 1, nev + k > N, ...), BSE_ERR_ALLOC, BSE_ERR_CUDA. */
bse_status_t bse_solve(bse_handle_t h, int32_t nev, int32_t k, int32_t ncv, double tol,
                       int32_t max_restarts, uint64_t seed, double *hOmega, void *dVec, int64_t ldvec,
                       double *hResid, bse_info_t *info);

/* bse_solve with a choice among the structure-preserving variants of PAPER.md:65-67 ("three variations of a structure-preserving
 * Lanczos iteration with a thick restart ... very similar in terms of operations"); full mode only (TDA handles run the
 * Hermitian iteration whatever `variant` says).  Same outputs, tolerances and errors as bse_solve.
 *   BSE_VARIANT_SHAO    (= bse_solve): Lanczos on H^2 through G = M o P in the inner product Re(x^H P(z)) (reading S4);
 *   BSE_VARIANT_GRUNING : Lanczos on H itself in the Omega inner product (reading R9): the Lanczos vectors alternate
 *                         between [x; conj x] and [y; -conj y]; both families are stored with their images (X, P(X), Y, M(Y):
 *                         twice the basis memory), the projected matrix is [[0, Bm^T], [Bm, 0]] with P(X) = Y Bm, and its positive
 *                         eigenvalues approximate omega directly (no square root of a Ritz value of H^2).  Two half applies per
 *                         block step, as BSE_VARIANT_SHAO; twice the orthogonalisation work.
 * The third variant the paper names (ProjectedBSE) is not built: see DESIGN.md section 2, reading R10. */
enum { BSE_VARIANT_SHAO = 0, BSE_VARIANT_GRUNING = 1 };
bse_status_t bse_solve_variant(bse_handle_t h, int32_t variant, int32_t nev, int32_t k, int32_t ncv, double tol,
                               int32_t max_restarts, uint64_t seed, double *hOmega, void *dVec, int64_t ldvec,
                               double *hResid, bse_info_t *info);

/* Lanczos with quadrature rules (the optical absorption spectrum "directly, without explicitly computing
 * the eigenpairs").  No reorthogonalisation, no stored basis; dStart: N complex128, device, not modified.  Synchronous;
 * all scalars stay on the device until the end.
 *   TDA handle:  `steps` steps of the three-term Lanczos recurrence of R started at d / |d|:
 *     hAlpha[0..steps)  diagonal of the Jacobi matrix T;  hBeta[0..steps]: hBeta[0] = |d|_2, hBeta[j] couples steps
 *     j-1, j.  Each step is one bse_apply with k = 1 plus three O(N) kernels.
 *   FULL handle (operator of Eq. 1, with A = R^*, C = C^T): the recurrence of G = M o P,
 *     P(x) = R x + C conj(x), M(y) = R y - C conj(y), in the inner product <a, b>_P = Re(a^H P(b)) (the structured
 *     iteration of bse_solve with k = 1), started at d / sqrt(<d, d>_P): hBeta[0] = sqrt(Re(d^H P(d))).  For
 *     u = [d; conj d], Sigma = diag(I, -I):  u^H Sigma (z - H)^{-1} u = 2 hBeta[0]^2 [(z^2 - T)^{-1}]_00
 *     (bse_quadrature_resolvent_full).  The other start vector of the structure, [y; -conj y], is d = i y.  Each
 *     step is two half applies with k = 1 (R and C streamed once each) plus five O(N) kernels.
 *     BSE_ERR_NOT_POSITIVE_DEFINITE when Re(w^H P(w)) < 0 is met (PAPER.md:49's precondition fails).
 * *hDone (nullable) = number of valid steps (smaller than `steps` only on an exact breakdown). */
bse_status_t bse_lanczos_quadrature(bse_handle_t h, const void *dStart, int32_t steps, double *hAlpha,
                                    double *hBeta, int32_t *hDone);

/* Host utility: d^H (omega_i + i eta - R)^{-1} d  ~=  hBeta[0]^2 [(z - T)^{-1}]_00 by the continued fraction of the
 * Jacobi matrix T(hAlpha, hBeta).  hOut: n_omega complex128 (host).  -Im(...)/pi is the broadened spectral function. */
bse_status_t bse_quadrature_resolvent(int32_t steps, const double *hAlpha, const double *hBeta, int32_t n_omega,
                                      const double *hOmega, double eta, void *hOut);

/* Host utility, full mode: u^H Sigma (omega_i + i eta - H)^{-1} u ~= 2 hBeta[0]^2 [(z^2 - T)^{-1}]_00, u = [d; conj d],
 * from the coefficients a FULL handle's bse_lanczos_quadrature returned.  hOut: n_omega complex128 (host). */
bse_status_t bse_quadrature_resolvent_full(int32_t steps, const double *hAlpha, const double *hBeta, int32_t n_omega,
                                           const double *hOmega, double eta, void *hOut);

/* Host utility (no device work): eigen-decomposition of the m x m complex Hermitian matrix hA (column-major, lda,
 * lower triangle read, destroyed) -- the "small projected eigenproblem" of PAPER.md:67, which bse_solve keeps on
 * the host.  hW: m eigenvalues ascending; hZ (m x nz, ldz): the first nz eigenvectors.  Returns BSE_ERR_INTERNAL
 * if the QL iteration fails. */
bse_status_t bse_host_heev(int32_t m, void *hA, int32_t lda, double *hW, void *hZ, int32_t ldz, int32_t nz);

/* The same for a REAL symmetric matrix (hA, hZ: doubles) -- the projected matrix of the full-mode iteration is real
 * symmetric (real coefficients in the inner product Re(x^H P(y))): a quarter of the flops of the complex driver in the
 * reduction and the back-transformation. */
bse_status_t bse_host_syev(int32_t m, double *hA, int32_t lda, double *hW, double *hZ, int32_t ldz, int32_t nz);

/* bse_lanczos_quadrature (TDA handles) for callers that cannot allocate: code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc.  Same arguments, same recurrence, same results; the scratch
 * (three N-vectors and the recurrence scalars) is a file-scope device array of fixed size inside the library, so the call
 * performs no cudaMalloc / cudaFree and no host allocation.  Limits: N <= BSE_STATIC_QUADRATURE_MAX_N and
 * steps <= BSE_STATIC_QUADRATURE_MAX_STEPS, else BSE_ERR_STATIC_LIMIT ("size exceeds the static scratch limit") and nothing
 * is launched.  Every GPU that loads the library holds the array (1.5 MiB + 16 KiB) until exit.  All calls on one device
 * share it: each call clears the scalars it accumulates into and overwrites the vectors before reading them, but two calls
 * that overlap on the same GPU (different streams or threads) race -- serialise them.  hAlpha: steps doubles, hBeta:
 * steps + 1 doubles (host, written directly).  Synchronous on the handle's stream.  Full-mode and incomplete partial handles:
 * BSE_ERR_INVALID_ARG. */
#define BSE_STATIC_QUADRATURE_MAX_N 32768
#define BSE_STATIC_QUADRATURE_MAX_STEPS 1024
bse_status_t bse_lanczos_quadrature_static(bse_handle_t h, const void *dStart, int32_t steps, double *hAlpha,
                                           double *hBeta, int32_t *hDone);

/* The diagonalisation scheme of PAPER.md section 2.1 (Eq. 2-4) on the device, for full-mode handles (any
 * store): M_r of Eq. (3) from the packed tiles -> real Cholesky M_r = L L^T -> W = L^T J L (real skew-symmetric) -> Householder
 * tridiagonalisation of W in real arithmetic -> the Hermitian tridiagonal -iT (zero diagonal) solved on the host through its
 * N x N bidiagonal factor -> back-transformation [X; Y] = Q L^-T z.  "If eigenvectors for more than 5% of the spectrum are
 * required, direct diagonalization routines are recommended": nev may be anything up to N (the whole positive
 * spectrum).  O(N^3) work and three real 2N x 2N matrices of device memory, allocated and freed inside the call.
 *   hOmega  : nev doubles (host): the nev smallest positive omega, ascending;
 *   dVec    : 2N x nev complex128 (device, column-major, ldvec >= 2N): right eigenvectors [X_I; Y_I] with
 *             X^H X - Y^H Y = 1; NULL: eigenvalues only (the back-transformation is skipped);
 *   hSeconds: 6 doubles (host, nullable): Cholesky (with M_r), W, tridiagonalisation, host tridiagonal solve,
 *             back-transformation, total.
 * Synchronous.  Errors: BSE_ERR_NOT_POSITIVE_DEFINITE (a Cholesky pivot <= 0: the precondition of PAPER.md:49 fails),
 * BSE_ERR_INVALID_ARG (TDA or partial handle, nev < 1, nev > N, 2N > BSE_DIRECT_MAX_N), BSE_ERR_ALLOC, BSE_ERR_CUDA. */
#define BSE_DIRECT_MAX_N 24576
bse_status_t bse_solve_direct(bse_handle_t h, int32_t nev, double *hOmega, void *dVec, int64_t ldvec, double *hSeconds);

/* Real symmetric tridiagonal eigenproblem on the host (hD: m diagonal, hE: m - 1 sub-diagonal entries; both untouched): all
 * eigenvalues ascending in hW, eigenvectors of the nz lowest in hZ (m x nz, ldz).  The last stage of bse_solve_direct. */
bse_status_t bse_host_stev(int32_t m, const double *hD, const double *hE, double *hW, double *hZ, int32_t ldz, int32_t nz);
/* The nz lowest eigenpairs only (hW: nz values, hZ nullable): a small part of the spectrum (8 nz <= m) is found by bisection on
 * the Sturm count plus inverse iteration, O(m nz), without the O(m^2) sweep over the whole matrix; otherwise as bse_host_stev. */
bse_status_t bse_host_stev_lowest(int32_t m, const double *hD, const double *hE, int32_t nz, double *hW, double *hZ, int32_t ldz);

/* The eigenvectors that "can be obtained trivially" from the right eigenvectors v_I = [X_I; Y_I] of the positive omega_I that
 * bse_solve returns (full mode, dVec / dOut 2N x nev column-major, must not alias):
 *   which = BSE_PARTNER_RIGHT_NEGATIVE : right eigenvectors of -omega_I,  [conj(Y_I); conj(X_I)]
 *   which = BSE_PARTNER_LEFT_POSITIVE  : left eigenvectors of +omega_I,   Sigma v_I = [X_I; -Y_I]      (u^H H = omega u^H)
 *   which = BSE_PARTNER_LEFT_NEGATIVE  : left eigenvectors of -omega_I,   [conj(Y_I); -conj(X_I)]
 * With v_I^H Sigma v_J = delta_IJ the left and right sets are bi-orthonormal: u_I^H v_J = delta_IJ (+omega), = -delta_IJ (-omega).
 * Asynchronous on the handle's stream.  Errors: BSE_ERR_INVALID_ARG (TDA handle, aliasing, sizes). */
enum { BSE_PARTNER_RIGHT_NEGATIVE = 0, BSE_PARTNER_LEFT_POSITIVE = 1, BSE_PARTNER_LEFT_NEGATIVE = 2 };
bse_status_t bse_partner_vectors(bse_handle_t h, const void *dVec, int64_t ldvec, int32_t nev, int32_t which, void *dOut,
                                 int64_t ldout);

/* The two dense basis kernels of the orthogonalisation and the restart on their own (
 * PAPER.md:71, 67) -- what bse_orth and bse_solve are built from, exported so that they can be driven and timed directly.
 *   bse_gram  : G = A^H B for A (n x m, lda) and B (n x k, ldb), n = N of the handle.  real_ip = 0: the complex Gram
 *               matrix, written to dG (m x k complex128, ld = m).  real_ip = 1: Re(A^H B) only -- the real inner product of
 *               the full-mode iteration (reading S4) -- written as complex128 with zero imaginary parts.  HBM-bound on A.
 *   bse_update: C = alpha * A S + beta * C for A (n x m, lda), S (m x l complex128 device, ld = m; imaginary parts ignored
 *               when real_ip = 1) and C (n x l, ldc; must not alias A).  l <= 8: the projection update W -= V h (HBM-bound);
 *               large l: the Ritz rotation V <- V S (FP64-tensor-bound).
 * Asynchronous on the handle's stream; dG / dS scratch conversions use the handle's workspace.  Errors: BSE_ERR_INVALID_ARG. */
bse_status_t bse_gram(bse_handle_t h, const void *dA, int64_t lda, int32_t m, const void *dB, int64_t ldb, int32_t k,
                      int32_t real_ip, void *dG);
bse_status_t bse_update(bse_handle_t h, const void *dA, int64_t lda, int32_t m, const void *dS, int32_t l, int32_t real_ip,
                        void *dC, int64_t ldc, double alpha, double beta);

/* Microbenchmarks behind the roofline denominators (north_star: "achieved HBM GB/s and FP64 pipe utilisation ... against
 * the chip's peaks"; MEASURED_PEAKS.json has no FP64 figure).  Each runs one warm-up and one timed launch of a kernel that
 * does nothing else, on one CTA per SM, timed with CUDA events on `stream`; synchronous.
 *   BSE_PEAK_DMMA           : FP64 tensor pipe, mma.sync m8n8k4 f64 (DMMA.8x8x4); p1 = warps per SM (default 8), p2 =
 *                             independent accumulator chains per warp (1, 2, 4, 8 or 12; default 8); p2 = -1: twelve chains
 *                             with the three-product role's mix of plain FP64 adds (8 DADD per 12 DMMA); TFLOP/s of the DMMAs
 *   BSE_PEAK_DFMA           : plain FP64 FMA, 8 chains per thread; p1 = warps per SM (default 32); result TFLOP/s
 *   BSE_PEAK_BULK_READ      : read-only stream of dBuf (device, buf_bytes) through cp.async.bulk into a shared-memory ring
 *                             of p2 stages (default 3) of p1 bytes (default 65536) -- the apply kernels' data path; GB/s
 *   BSE_PEAK_BULK_READ_SMEM : the same with every byte read back from shared memory by the consumer warp; GB/s
 *   BSE_PEAK_RED            : red.global.add.f64 scattered over dBuf (buf_bytes / 8 doubles, which it modifies); G atomics/s
 * hMs (nullable): duration of the timed launch in ms.  Errors: BSE_ERR_INVALID_ARG, BSE_ERR_CUDA. */
enum { BSE_PEAK_DMMA = 0, BSE_PEAK_DFMA = 1, BSE_PEAK_BULK_READ = 2, BSE_PEAK_BULK_READ_SMEM = 3, BSE_PEAK_RED = 4 };
bse_status_t bse_selftest_peak(int32_t what, int32_t p1, int32_t p2, void *dBuf, int64_t buf_bytes, void *stream,
                               double *hResult, double *hMs);

/* Number of kernels this library has launched on the calling process's device since load (bench.py's
 * "gpu_launches" claim). */
int64_t bse_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* BSE_B200_H */
