"""Thin Python binding of libbse_b200.so (include/bse.h).  Argument marshalling only: every step of the
path runs in the library's CUDA kernels.  torch is used for device memory and streams, nothing else.

The binding fails loudly if the CUDA library is missing or a call returns an error; there is no CPU
fallback and this package never imports `oracle`.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libbse_b200.so")
_lib = None

MODE_TDA, MODE_FULL = 0, 1
VARIANT_SHAO, VARIANT_GRUNING = 0, 1                                         # bse_solve_variant
STORE_C128, STORE_C64, STORE_REAL_FORM, STORE_REAL_FORM_C64 = 0, 1, 2, 3      # storage type of the tile store (include/bse.h)
MATRIX_R, MATRIX_C = 0, 1
TILE = 64
TILE_BYTES = 65536

STATUS = {0: "BSE_OK", 1: "BSE_ERR_INVALID_ARG", 2: "BSE_ERR_CUDA", 3: "BSE_ERR_ALLOC", 4: "BSE_ERR_NOT_CONVERGED",
          5: "BSE_ERR_NOT_POSITIVE_DEFINITE", 6: "BSE_ERR_INTERNAL", 7: "BSE_ERR_STATIC_LIMIT"}
STATIC_QUADRATURE_MAX_N, STATIC_QUADRATURE_MAX_STEPS = 32768, 1024       # include/bse.h
DIRECT_MAX_N = 24576                                                         # bse_solve_direct: 2N at most


class BseError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {STATUS.get(status, status)}")


class _Info(ctypes.Structure):
    _fields_ = [("n_apply", ctypes.c_int32), ("n_restart", ctypes.c_int32), ("nconv", ctypes.c_int32),
                ("ncv", ctypes.c_int32), ("seconds_apply", ctypes.c_double), ("seconds_orth", ctypes.c_double),
                ("seconds_project", ctypes.c_double), ("seconds_restart", ctypes.c_double),
                ("seconds_total", ctypes.c_double), ("norm_est", ctypes.c_double), ("basis_orth_err", ctypes.c_double)]


_vp, _i64, _i32, _u64, _dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_uint64, ctypes.c_double

_SIGNATURES = {
    "bse_layout": [_i64, _i32, ctypes.POINTER(_i32), ctypes.POINTER(_i64), ctypes.POINTER(_i64)],
    "bse_pack_from_dense": [_vp, _i64, _i64, _i32, _vp, _i32, _vp],
    "bse_unpack_to_dense": [_vp, _i32, _i64, _i32, _vp, _i64, _vp],
    "bse_fill_synthetic": [_vp, _i32, _i64, _i32, _u64, _dbl, _i32, _vp],
    "bse_fill_closed_form_tda": [_vp, _i32, _i64, _vp, _vp, _dbl, _vp],
    "bse_fill_closed_form_full": [_vp, _vp, _i32, _i64, _vp, _vp, _vp, _vp, _dbl, _dbl, _vp],
    "bse_create": [ctypes.POINTER(_vp), _i32, _i32, _i64, _vp, _vp, _vp],
    "bse_destroy": [_vp],
    "bse_to_real_form": [_vp, _vp, _i32, _i64, _vp],
    "bse_shard_layout": [_i64, _i32, _i32, _i32, ctypes.POINTER(_i32), ctypes.POINTER(_i32), ctypes.POINTER(_i64),
                         ctypes.POINTER(_i64), ctypes.POINTER(_i64)],
    "bse_fill_synthetic_shard": [_vp, _i32, _i64, _i32, _u64, _dbl, _i32, _i32, _i32, _vp],
    "bse_create_shard": [ctypes.POINTER(_vp), _i32, _i32, _i64, _i32, _i32, _vp, _vp, _vp],
    "bse_set_comm": [_vp, _vp, _vp],
    "bse_apply": [_vp, _vp, _i64, _vp, _i64, _i32],
    "bse_apply_half": [_vp, _i32, _vp, _i64, _vp, _i64, _i32],
    "bse_apply_host": [_vp, _vp, _i64, _vp, _i64, _i32],
    "bse_orth": [_vp, _vp, _i64, _i32, _vp, _i64, _vp, _i64, _i32, _vp, _i64, _vp, _vp, ctypes.POINTER(_i32)],
    "bse_lanczos_quadrature": [_vp, _vp, _i32, ctypes.POINTER(_dbl), ctypes.POINTER(_dbl), ctypes.POINTER(_i32)],
    "bse_lanczos_quadrature_static": [_vp, _vp, _i32, ctypes.POINTER(_dbl), ctypes.POINTER(_dbl), ctypes.POINTER(_i32)],
    "bse_quadrature_resolvent": [_i32, ctypes.POINTER(_dbl), ctypes.POINTER(_dbl), _i32, ctypes.POINTER(_dbl), _dbl, _vp],
    "bse_quadrature_resolvent_full": [_i32, ctypes.POINTER(_dbl), ctypes.POINTER(_dbl), _i32, ctypes.POINTER(_dbl), _dbl, _vp],
    "bse_host_heev": [_i32, _vp, _i32, _vp, _vp, _i32, _i32],
    "bse_host_syev": [_i32, _vp, _i32, _vp, _vp, _i32, _i32],
    "bse_solve": [_vp, _i32, _i32, _i32, _dbl, _i32, _u64, ctypes.POINTER(_dbl), _vp, _i64, ctypes.POINTER(_dbl),
                  ctypes.POINTER(_Info)],
    "bse_partner_vectors": [_vp, _vp, _i64, _i32, _i32, _vp, _i64],
    "bse_gram": [_vp, _vp, _i64, _i32, _vp, _i64, _i32, _i32, _vp],
    "bse_update": [_vp, _vp, _i64, _i32, _vp, _i32, _i32, _vp, _i64, _dbl, _dbl],
    "bse_solve_variant": [_vp, _i32, _i32, _i32, _i32, _dbl, _i32, _u64, ctypes.POINTER(_dbl), _vp, _i64, ctypes.POINTER(_dbl),
                          ctypes.POINTER(_Info)],
    "bse_selftest_peak": [_i32, _i32, _i32, _vp, _i64, _vp, ctypes.POINTER(_dbl), ctypes.POINTER(_dbl)],
    "bse_solve_direct": [_vp, _i32, ctypes.POINTER(_dbl), _vp, _i64, ctypes.POINTER(_dbl)],
    "bse_set_row_partition": [_vp, _i64, _i64],
    "bse_host_stev": [_i32, _vp, _vp, _vp, _vp, _i32, _i32],
    "bse_host_stev_lowest": [_i32, _vp, _vp, _i32, _vp, _vp, _i32],
}
EXPORTS = sorted(list(_SIGNATURES) + ["bse_status_string", "bse_launch_count"])


def lib():
    """Loads the C-ABI library.  Raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            raise ImportError(f"{_LIBPATH} is missing: run `python -m paper_2504_10096_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = ctypes.CDLL(_LIBPATH)
        for name, args in _SIGNATURES.items():
            fn = getattr(L, name)
            fn.argtypes = args
            fn.restype = ctypes.c_int
        L.bse_status_string.argtypes = [ctypes.c_int]
        L.bse_status_string.restype = ctypes.c_char_p
        L.bse_launch_count.argtypes = []
        L.bse_launch_count.restype = ctypes.c_int64
        _lib = L
    return _lib


def _check(st: int, where: str):
    if st != 0:
        raise BseError(st, where)


def _stream_ptr():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def bse_layout(N: int, storage: int = STORE_C128):
    t, n, b = _i32(), _i64(), _i64()
    _check(lib().bse_layout(N, storage, ctypes.byref(t), ctypes.byref(n), ctypes.byref(b)), "bse_layout")
    return t.value, n.value, b.value


def alloc_tiles(N: int, storage: int = STORE_C128):
    """Uninitialised device buffer for one packed matrix (torch uint8 tensor)."""
    import torch
    _, _, nbytes = bse_layout(N, storage)
    return torch.empty(nbytes, dtype=torch.uint8, device="cuda")


def _ld(t):
    """Leading dimension (complex elements) of a column-major block held as a torch tensor.

    Blocks are passed as torch complex128 tensors of shape (k, n) that are C-contiguous, i.e. the
    memory is column-major n x k with ld = n (or 1-D tensors of n elements for k = 1)."""
    assert t.is_cuda and t.dtype.is_complex and t.element_size() == 16 and t.is_contiguous()
    return t.shape[-1]


def bse_pack_from_dense(dense_cm, N: int, which: int, tiles=None, storage: int = STORE_C128):
    """dense_cm: torch complex128 CUDA tensor of shape (N, N) holding the matrix COLUMN-major
    (dense_cm[j, i] = A_ij), e.g. torch.from_numpy(A.T.copy()).cuda()."""
    tiles = alloc_tiles(N, storage) if tiles is None else tiles
    _check(lib().bse_pack_from_dense(dense_cm.data_ptr(), N, N, which, tiles.data_ptr(), storage, _stream_ptr()),
           "bse_pack_from_dense")
    return tiles


def bse_unpack_to_dense(tiles, N: int, which: int, storage: int = STORE_C128):
    import torch
    out = torch.zeros((N, N), dtype=torch.complex128, device="cuda")
    _check(lib().bse_unpack_to_dense(tiles.data_ptr(), storage, N, which, out.data_ptr(), N, _stream_ptr()),
           "bse_unpack_to_dense")
    return out      # out[j, i] = A_ij


def bse_fill_synthetic(N: int, which: int, seed: int, sigma: float = 0.0, group: int = 16, tiles=None,
                       storage: int = STORE_C128):
    tiles = alloc_tiles(N, storage) if tiles is None else tiles
    _check(lib().bse_fill_synthetic(tiles.data_ptr(), storage, N, which, seed, sigma, group, _stream_ptr()),
           "bse_fill_synthetic")
    return tiles


def bse_fill_closed_form_tda(N: int, lam, u, s: float, tiles=None, storage: int = STORE_C128):
    tiles = alloc_tiles(N, storage) if tiles is None else tiles
    _check(lib().bse_fill_closed_form_tda(tiles.data_ptr(), storage, N, lam.data_ptr(), u.data_ptr(), s,
                                          _stream_ptr()),
           "bse_fill_closed_form_tda")
    return tiles


def bse_fill_closed_form_full(N: int, d1, d2, ur, phi, s1: float, s2: float, storage: int = STORE_C128):
    rt, ct = alloc_tiles(N, storage), alloc_tiles(N, storage)
    _check(lib().bse_fill_closed_form_full(rt.data_ptr(), ct.data_ptr(), storage, N, d1.data_ptr(), d2.data_ptr(),
                                           ur.data_ptr(), phi.data_ptr(), s1, s2, _stream_ptr()),
           "bse_fill_closed_form_full")
    return rt, ct


@dataclass
class SolveResult:
    omega: "object"
    vectors: "object"
    resid: "object"
    info: dict
    status: int


def bse_shard_layout(N: int, n_shards: int, shard: int, storage: int = STORE_C128):
    """(tile_row_begin, tile_row_end, first_tile, n_tiles, bytes) of one of n_shards slices of the packed store with
    (nearly) equal tile counts.  Host-only: needs no device."""
    rb, re, ft, nt, by = _i32(), _i32(), _i64(), _i64(), _i64()
    _check(lib().bse_shard_layout(N, storage, n_shards, shard, ctypes.byref(rb), ctypes.byref(re), ctypes.byref(ft),
                                  ctypes.byref(nt), ctypes.byref(by)), "bse_shard_layout")
    return rb.value, re.value, ft.value, nt.value, by.value


def bse_fill_synthetic_shard(N: int, which: int, seed: int, sigma: float, group: int, rows, storage: int = STORE_C128):
    """The slice of bse_fill_synthetic's store holding tile rows rows = (begin, end) (torch uint8 tensor)."""
    import torch
    by = bse_layout(N, storage)[2] // bse_layout(N, storage)[1]
    n_tiles = rows[1] * (rows[1] + 1) // 2 - rows[0] * (rows[0] + 1) // 2
    tiles = torch.empty(max(n_tiles, 1) * by, dtype=torch.uint8, device="cuda")
    _check(lib().bse_fill_synthetic_shard(tiles.data_ptr(), storage, N, which, seed, sigma, group, rows[0], rows[1],
                                          _stream_ptr()), "bse_fill_synthetic_shard")
    return tiles


def bse_to_real_form(r_tiles, c_tiles, N: int, storage: int = STORE_C128):
    """In place: (R, C) stores -> (S = R + C, D = R - C); use with Bse(..., storage=STORE_REAL_FORM[_C64])."""
    _check(lib().bse_to_real_form(r_tiles.data_ptr(), c_tiles.data_ptr(), storage, bse_layout(N, storage)[1], _stream_ptr()),
           "bse_to_real_form")
    return r_tiles, c_tiles


class Bse:
    """Handle wrapper (bse_create / bse_destroy).  Keeps the borrowed tile buffers alive."""

    def __init__(self, mode: int, N: int, r_tiles, c_tiles=None, storage: int = STORE_C128, rows=None):
        """rows = (tile_row_begin, tile_row_end): r_tiles / c_tiles hold only that slice of the packed store
        (bse_create_shard); apply / apply_half then return this slice's contribution to Y."""
        self.mode, self.N, self.storage, self.rows = mode, N, storage, rows
        self._keep = (r_tiles, c_tiles)
        self.n_op = 2 * N if mode == MODE_FULL else N
        import torch
        self._stream = torch.cuda.current_stream()           # every call of this handle enqueues on this stream
        h = _vp()
        cp = c_tiles.data_ptr() if c_tiles is not None else None
        if rows is None:
            _check(lib().bse_create(ctypes.byref(h), mode, storage, N, r_tiles.data_ptr(), cp, _stream_ptr()), "bse_create")
        else:
            _check(lib().bse_create_shard(ctypes.byref(h), mode, storage, N, rows[0], rows[1], r_tiles.data_ptr(), cp,
                                          _stream_ptr()), "bse_create_shard")
        self._h = h

    # Every call of this handle enqueues on the stream captured at creation.  If the caller's current stream is another
    # one, order the two: the handle's stream first waits for the work already queued on the caller's stream (the producer
    # of X, the allocation of Y), and afterwards the caller's stream waits for the handle's.
    def _enter(self, *tensors):
        import torch
        cur = torch.cuda.current_stream()
        if cur != self._stream:
            self._stream.wait_stream(cur)
            for t in tensors:
                if t is not None:
                    t.record_stream(self._stream)        # the caching allocator must not recycle it while the handle's stream uses it
        return cur

    def _exit(self, cur):
        if cur != self._stream:
            cur.wait_stream(self._stream)

    def close(self):
        if getattr(self, "_h", None):
            lib().bse_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def apply(self, X, Y=None):
        """Y = H X.  X: torch complex128 CUDA tensor of shape (k, n_op) (column-major n_op x k)."""
        import torch
        k = X.shape[0] if X.dim() == 2 else 1
        Y = torch.empty_like(X) if Y is None else Y
        cur = self._enter(X, Y)
        _check(lib().bse_apply(self._h, X.data_ptr(), _ld(X), Y.data_ptr(), _ld(Y), k), "bse_apply")
        self._exit(cur)
        return Y

    def apply_half(self, X, sign: int, Y=None):
        import torch
        k = X.shape[0] if X.dim() == 2 else 1
        Y = torch.empty_like(X) if Y is None else Y
        cur = self._enter(X, Y)
        _check(lib().bse_apply_half(self._h, sign, X.data_ptr(), _ld(X), Y.data_ptr(), _ld(Y), k), "bse_apply_half")
        self._exit(cur)
        return Y

    def apply_host(self, X_np, Y_np=None):
        """Host entry point: X_np numpy complex128 of shape (k, n_op), C-contiguous."""
        import numpy as np
        assert X_np.dtype == np.complex128 and X_np.flags.c_contiguous
        Y_np = np.empty_like(X_np) if Y_np is None else Y_np
        k, n = X_np.shape
        _check(lib().bse_apply_host(self._h, X_np.ctypes.data, n, Y_np.ctypes.data, n, k), "bse_apply_host")
        return Y_np

    def orth(self, V, W, BV=None, BW=None):
        """Block CGS2 of W (k, n) against V (m, n) [+ P-images].  Returns (hcoef (k, m), Bfac (k, k), rank).
        W (and BW) are overwritten.  hcoef/Bfac are column-major m x k / k x k viewed as torch (k, m)/(k, k)."""
        import torch
        m = 0 if V is None else V.shape[0]
        k = W.shape[0]
        hcoef = torch.zeros((k, max(m, 1)), dtype=torch.complex128, device="cuda")
        bfac = torch.zeros((k, k), dtype=torch.complex128, device="cuda")
        rank = _i32(0)
        _check(lib().bse_orth(self._h, V.data_ptr() if m else None, _ld(V) if m else self.N, m,
                              BV.data_ptr() if BV is not None else None, _ld(BV) if BV is not None else self.N,
                              W.data_ptr(), _ld(W), k, BW.data_ptr() if BW is not None else None,
                              _ld(BW) if BW is not None else self.N, hcoef.data_ptr(), bfac.data_ptr(),
                              ctypes.byref(rank)), "bse_orth")
        return hcoef[:, :m], bfac, rank.value

    def partner_vectors(self, vectors, which: int = 0):
        """-omega right eigenvectors (which = 0), left eigenvectors of +omega (1) / -omega (2) from solve()'s vectors (nev, 2N)."""
        import torch
        out = torch.empty_like(vectors)
        _check(lib().bse_partner_vectors(self._h, vectors.data_ptr(), _ld(vectors), vectors.shape[0], which, out.data_ptr(),
                                         _ld(out)), "bse_partner_vectors")
        return out

    def gram(self, A, B, real_ip: bool = False):
        """A^H B (bse_gram): A (m, n), B (k, n) torch blocks -> torch (k, m) = column-major m x k."""
        import torch
        m, k = A.shape[0], B.shape[0]
        G = torch.empty((k, m), dtype=torch.complex128, device="cuda")
        _check(lib().bse_gram(self._h, A.data_ptr(), _ld(A), m, B.data_ptr(), _ld(B), k, 1 if real_ip else 0, G.data_ptr()),
               "bse_gram")
        return G

    def update(self, A, S, C, alpha: float = 1.0, beta: float = 0.0, real_ip: bool = False):
        """C = alpha A S + beta C (bse_update): A (m, n), S (l, m) = column-major m x l, C (l, n)."""
        m, l = A.shape[0], S.shape[0]
        _check(lib().bse_update(self._h, A.data_ptr(), _ld(A), m, S.data_ptr(), l, 1 if real_ip else 0, C.data_ptr(), _ld(C),
                                alpha, beta), "bse_update")
        return C

    def lanczos_quadrature(self, d, steps: int):
        """(alpha[steps'], beta[steps'+1]) of PAPER.md:65's Lanczos-with-quadrature solver; d: torch complex128 (N,)."""
        import numpy as np
        alpha = np.zeros(steps); beta = np.zeros(steps + 1)
        done = _i32(0)
        _check(lib().bse_lanczos_quadrature(self._h, d.data_ptr(), steps, alpha.ctypes.data_as(ctypes.POINTER(_dbl)),
                                            beta.ctypes.data_as(ctypes.POINTER(_dbl)), ctypes.byref(done)),
               "bse_lanczos_quadrature")
        return alpha[:done.value], beta[:done.value + 1]

    def lanczos_quadrature_static(self, d, steps: int, alpha=None, beta=None):
        """lanczos_quadrature through bse_lanczos_quadrature_static: no allocation inside the call (scratch in a fixed device
        array of the library; N <= STATIC_QUADRATURE_MAX_N, steps <= STATIC_QUADRATURE_MAX_STEPS).  alpha / beta: optional
        preallocated numpy arrays of steps / steps + 1 doubles."""
        import numpy as np
        alpha = np.zeros(steps) if alpha is None else alpha
        beta = np.zeros(steps + 1) if beta is None else beta
        done = _i32(0)
        _check(lib().bse_lanczos_quadrature_static(self._h, d.data_ptr(), steps, alpha.ctypes.data_as(ctypes.POINTER(_dbl)),
                                                   beta.ctypes.data_as(ctypes.POINTER(_dbl)), ctypes.byref(done)),
               "bse_lanczos_quadrature_static")
        return alpha[:done.value], beta[:done.value + 1]

    def solve(self, nev: int, k: int, ncv: int = 0, tol: float = 1e-8, max_restarts: int = 1000, seed: int = 1,
              raise_on_error: bool = True, variant: int = 0):
        import numpy as np
        import torch
        omega = np.zeros(nev)
        resid = np.zeros(nev)
        vec = torch.zeros((nev, self.n_op), dtype=torch.complex128, device="cuda")
        cur = self._enter(vec)
        info = _Info()
        st = lib().bse_solve_variant(self._h, variant, nev, k, ncv, tol, max_restarts, seed,
                             omega.ctypes.data_as(ctypes.POINTER(_dbl)), vec.data_ptr(), self.n_op,
                             resid.ctypes.data_as(ctypes.POINTER(_dbl)), ctypes.byref(info))
        self._exit(cur)
        if st != 0 and raise_on_error:
            raise BseError(st, "bse_solve")
        return SolveResult(omega, vec, resid, {f: getattr(info, f) for f, _ in _Info._fields_}, st)


    def solve_direct(self, nev: int, vectors: bool = True):
        """The diagonalisation scheme of PAPER.md section 2.1 on the device (full mode): (omega, vec or None, seconds) with
        seconds = dict(cholesky, w, tridiag, host_eig, back, total)."""
        import numpy as np
        import torch
        omega = np.zeros(nev)
        sec = np.zeros(6)
        vec = torch.zeros((nev, self.n_op), dtype=torch.complex128, device="cuda") if vectors else None
        cur = self._enter(vec) if vectors else self._enter()
        st = lib().bse_solve_direct(self._h, nev, omega.ctypes.data_as(ctypes.POINTER(_dbl)),
                                    vec.data_ptr() if vectors else None, self.n_op, sec.ctypes.data_as(ctypes.POINTER(_dbl)))
        self._exit(cur)
        _check(st, "bse_solve_direct")
        return omega, vec, dict(zip(("cholesky", "w", "tridiag", "host_eig", "back", "total"), sec.tolist()))


def sum_partials(Y, group=None):
    """Sum the shards' partial products in place over the process group (one all-reduce of 16 N k bytes; NCCL over
    NVLink on GPUs).  A no-op without an initialised process group or with a single rank."""
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(torch.view_as_real(Y), op=dist.ReduceOp.SUM, group=group)
    return Y


class ShardedBse:
    """The operator's tile stream sharded over the ranks of a torch.distributed process group, one process per GPU
    (the paper partitions the matrix by rows over MPI ranks).  Rank r holds the slice of
    the packed store that bse_shard_layout assigns to it (contiguous tile rows, equal tile counts); X is replicated;
    apply / apply_half run the local kernels on the slice and sum the partial Y with ONE all-reduce of 16 N k bytes.
    After install_comm() the library itself completes every product through the process group, and solve() /
    lanczos_quadrature() run on the sharded operator with replicated vectors, all ranks in bitwise lock step."""

    def __init__(self, mode: int, N: int, r_slice, c_slice=None, rows=None, storage: int = STORE_C128, group=None):
        self.local = Bse(mode, N, r_slice, c_slice, storage=storage, rows=rows)
        self.group, self.N, self.mode = group, N, mode
        self._cb = None
        self.comm_calls = [0, 0]                                 # sums, broadcasts issued through the hook

    def install_comm(self, row_partition: bool = False):
        """Give the library the process group (bse_set_comm): its products become complete (local + one all-reduce) and
        bse_solve / bse_lanczos_quadrature run on the sharded operator with replicated vectors (include/bse.h).
        row_partition=True also divides the VECTORS by rows over the ranks (bse_set_row_partition): bases,
        orthogonalisation and restart then work on N / world rows per rank; solve() still returns full-length vectors."""
        import torch
        import torch.distributed as dist
        group = self.group
        if row_partition:
            on = dist.is_available() and dist.is_initialized()
            world, rank = (dist.get_world_size(group), dist.get_rank(group)) if on else (1, 0)
            self.vec_rows = (self.N * rank // world, self.N * (rank + 1) // world)
            _check(lib().bse_set_row_partition(self.local._h, *self.vec_rows), "bse_set_row_partition")
        src = dist.get_global_rank(group, 0) if group is not None else 0
        calls = self.comm_calls

        class _Dev:                                              # zero-copy view of the library's device buffer
            def __init__(self, ptr, n):
                self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (ptr, False), "version": 2}

        stream = self.local._stream                          # the stream the library's kernels are ordered on

        def hook(user, op, ptr, n):
            try:
                t = torch.as_tensor(_Dev(ptr, n), device="cuda")
                with torch.cuda.stream(stream):                  # order the collective after the kernels that wrote the buffer
                    if op == 0:
                        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
                    else:
                        dist.broadcast(t, src=src, group=group)
                calls[op] += 1
                return 0
            except Exception as e:                               # never let an exception cross the C frame
                import sys
                print(f"[ShardedBse] communication hook failed: {e!r}", file=sys.stderr)
                return 1

        self._cb = ctypes.CFUNCTYPE(_i32, _vp, _i32, _vp, _i64)(hook)
        _check(lib().bse_set_comm(self.local._h, ctypes.cast(self._cb, _vp), None), "bse_set_comm")
        return self

    def solve(self, *args, **kw):
        assert self._cb is not None, "install_comm() first"
        return self.local.solve(*args, **kw)

    def lanczos_quadrature(self, d, steps: int):
        assert self._cb is not None, "install_comm() first"
        return self.local.lanczos_quadrature(d, steps)

    @classmethod
    def synthetic(cls, mode: int, N: int, seed: int, sigma: float, group_size: int, storage: int = STORE_C128, group=None,
                  real_form: bool = False):
        """Each rank generates its own slice of BASELINE.json's synthetic operator on its GPU (nothing crosses PCIe)."""
        import torch.distributed as dist
        on = dist.is_available() and dist.is_initialized()
        world, rank = (dist.get_world_size(group), dist.get_rank(group)) if on else (1, 0)
        rb, re, _, _, _ = bse_shard_layout(N, world, rank, storage)
        r = bse_fill_synthetic_shard(N, MATRIX_R, seed, sigma, group_size, (rb, re), storage)
        c = bse_fill_synthetic_shard(N, MATRIX_C, seed, 0.0, group_size, (rb, re), storage) if mode == MODE_FULL else None
        if real_form:
            _check(lib().bse_to_real_form(r.data_ptr(), c.data_ptr(), storage, re * (re + 1) // 2 - rb * (rb + 1) // 2,
                                          _stream_ptr()), "bse_to_real_form")
            storage = STORE_REAL_FORM if storage == STORE_C128 else STORE_REAL_FORM_C64
        return cls(mode, N, r, c, (rb, re), storage, group)

    def _sum(self, Y):
        import torch
        if self._cb is not None:                                 # with the hook the library has summed already
            return Y
        with torch.cuda.stream(self.local._stream):              # after the kernels that wrote Y
            return sum_partials(Y, self.group)

    def apply(self, X, Y=None):
        return self._sum(self.local.apply(X, Y))

    def apply_half(self, X, sign: int, Y=None):
        return self._sum(self.local.apply_half(X, sign, Y))


def host_heev(A, nz=None):
    """Host utility: eigenvalues (ascending) and first nz eigenvectors of a Hermitian numpy matrix."""
    import numpy as np
    m = A.shape[0]
    nz = m if nz is None else nz
    a = np.asfortranarray(A, dtype=np.complex128).copy(order="F")
    w = np.zeros(m)
    Z = np.zeros((m, max(nz, 1)), dtype=np.complex128, order="F")
    _check(lib().bse_host_heev(m, a.ctypes.data, m, w.ctypes.data, Z.ctypes.data, m, nz), "bse_host_heev")
    return w, Z[:, :nz]


def host_syev(A, nz=None):
    """Host utility: eigenvalues (ascending) and first nz eigenvectors of a REAL symmetric numpy matrix."""
    import numpy as np
    m = A.shape[0]
    nz = m if nz is None else nz
    a = np.asfortranarray(A, dtype=np.float64).copy(order="F")
    w = np.zeros(m)
    Z = np.zeros((m, max(nz, 1)), dtype=np.float64, order="F")
    _check(lib().bse_host_syev(m, a.ctypes.data, m, w.ctypes.data, Z.ctypes.data, m, nz), "bse_host_syev")
    return w, Z[:, :nz]


def host_stev(d, e, nz=None):
    """Host utility: eigenvalues (ascending) and first nz eigenvectors of the real symmetric tridiagonal (d, e)."""
    import numpy as np
    m = len(d)
    nz = m if nz is None else nz
    d = np.ascontiguousarray(d, dtype=np.float64); e = np.ascontiguousarray(e, dtype=np.float64)
    w = np.zeros(m)
    Z = np.zeros((m, max(nz, 1)), dtype=np.float64, order="F")
    _check(lib().bse_host_stev(m, d.ctypes.data, e.ctypes.data if m > 1 else None, w.ctypes.data, Z.ctypes.data, m, nz),
           "bse_host_stev")
    return w, Z[:, :nz]


def host_stev_lowest(d, e, nz, vectors: bool = True):
    """Host utility: the nz lowest eigenvalues (and eigenvectors) of the real symmetric tridiagonal (d, e)."""
    import numpy as np
    m = len(d)
    d = np.ascontiguousarray(d, dtype=np.float64); e = np.ascontiguousarray(e, dtype=np.float64)
    w = np.zeros(nz)
    Z = np.zeros((m, nz), dtype=np.float64, order="F") if vectors else None
    _check(lib().bse_host_stev_lowest(m, d.ctypes.data, e.ctypes.data if m > 1 else None, nz, w.ctypes.data,
                                      Z.ctypes.data if vectors else None, m), "bse_host_stev_lowest")
    return w, Z


def quadrature_resolvent(alpha, beta, omega, eta: float):
    """Host utility: d^H (omega + i eta - R)^-1 d from the continued fraction (numpy complex128 array)."""
    import numpy as np
    alpha = np.ascontiguousarray(alpha, dtype=np.float64); beta = np.ascontiguousarray(beta, dtype=np.float64)
    omega = np.ascontiguousarray(omega, dtype=np.float64)
    out = np.zeros(len(omega), dtype=np.complex128)
    P = ctypes.POINTER(_dbl)
    _check(lib().bse_quadrature_resolvent(len(alpha), alpha.ctypes.data_as(P), beta.ctypes.data_as(P), len(omega),
                                          omega.ctypes.data_as(P), eta, out.ctypes.data), "bse_quadrature_resolvent")
    return out


def quadrature_resolvent_full(alpha, beta, omega, eta: float):
    """Host utility, full mode: u^H Sigma (omega + i eta - H)^-1 u, u = [d; conj d] (numpy complex128 array)."""
    import numpy as np
    alpha = np.ascontiguousarray(alpha, dtype=np.float64); beta = np.ascontiguousarray(beta, dtype=np.float64)
    omega = np.ascontiguousarray(omega, dtype=np.float64)
    out = np.zeros(len(omega), dtype=np.complex128)
    P = ctypes.POINTER(_dbl)
    _check(lib().bse_quadrature_resolvent_full(len(alpha), alpha.ctypes.data_as(P), beta.ctypes.data_as(P), len(omega),
                                               omega.ctypes.data_as(P), eta, out.ctypes.data),
           "bse_quadrature_resolvent_full")
    return out


PEAK_DMMA, PEAK_DFMA, PEAK_BULK_READ, PEAK_BULK_READ_SMEM, PEAK_RED = 0, 1, 2, 3, 4


def selftest_peak(what: int, p1: int = 0, p2: int = 0, buf=None):
    """One of the library's microbenchmarks (include/bse.h): (rate, ms).  TFLOP/s, GB/s or G atomics/s."""
    r, ms = _dbl(), _dbl()
    _check(lib().bse_selftest_peak(what, p1, p2, buf.data_ptr() if buf is not None else None,
                                   buf.numel() * buf.element_size() if buf is not None else 0, _stream_ptr(),
                                   ctypes.byref(r), ctypes.byref(ms)), "bse_selftest_peak")
    return r.value, ms.value


def launch_count() -> int:
    return lib().bse_launch_count()
