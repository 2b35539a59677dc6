"""CPU oracle for the BSE hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper around oracle/bse_oracle.c (plain C, written from PAPER.md; see the header of
that file for what each routine follows and how it is pinned).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It imports nothing from the CUDA package and the CUDA package imports nothing from here.

All arrays handed to C are dense, row-major (C order) complex128; blocks are n_rows x k.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bse_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

_c128 = np.ctypeslib.ndpointer(dtype=np.complex128, flags="C_CONTIGUOUS")
_f64 = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_i64 = ctypes.c_int64


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.orc_apply_tda_rows.argtypes = [_i64, _i64, _c128, _c128, _c128, _i64, _i64]
        lib.orc_apply_full_rows.argtypes = [_i64, _i64, _c128, _c128, _c128, _c128, _i64, _i64]
        lib.orc_apply_half.argtypes = [_i64, _i64, ctypes.c_int, _c128, _c128, _c128, _c128]
        lib.orc_rows_times_block.argtypes = [_i64, _i64, _i64, _c128, _c128, _c128]
        lib.orc_jacobi_herm.argtypes = [_i64, _c128, _f64, _c128]
        lib.orc_jacobi_herm.restype = ctypes.c_int
        lib.orc_build_Mr.argtypes = [_i64, _c128, _c128, _f64]
        lib.orc_cholesky_real.argtypes = [_i64, _f64, _f64]
        lib.orc_cholesky_real.restype = ctypes.c_int
        lib.orc_bse_direct.argtypes = [_i64, _c128, _c128, ctypes.c_void_p, _f64, ctypes.c_void_p]
        lib.orc_bse_direct.restype = ctypes.c_int
        lib.orc_block_cgs2.argtypes = [_i64, _i64, _i64, _c128, _c128, _c128, _c128, _c128]
        lib.orc_block_cgs2.restype = ctypes.c_int
        lib.orc_lanczos_tda.argtypes = [_i64, _c128, ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.c_int,
                                        _c128, _f64, _c128, _f64]
        lib.orc_lanczos_tda.restype = ctypes.c_int
        lib.orc_lanczos_full.argtypes = [_i64, _c128, _c128, ctypes.c_int, ctypes.c_double, ctypes.c_int,
                                         ctypes.c_int, ctypes.c_int, _c128, _f64, _c128, _f64]
        lib.orc_lanczos_full.restype = ctypes.c_int
        lib.orc_lanczos_full_gruning.argtypes = [_i64, _c128, _c128, ctypes.c_int, ctypes.c_double, ctypes.c_int,
                                                 ctypes.c_int, ctypes.c_int, _c128, _f64, _c128, _f64, ctypes.c_void_p,
                                                 ctypes.c_int]
        lib.orc_lanczos_full_gruning.restype = ctypes.c_int
        lib.orc_tridiag_ql.argtypes = [_i64, _f64, _f64, _f64, ctypes.c_void_p]
        lib.orc_tridiag_ql.restype = ctypes.c_int
        lib.orc_round_c64.argtypes = [_i64, _c128, _c128]
        lib.orc_lanczos_quadrature.argtypes = [_i64, _c128, _c128, ctypes.c_int, _f64, _f64]
        lib.orc_lanczos_quadrature.restype = ctypes.c_int
        lib.orc_lanczos_quadrature_full.argtypes = [_i64, _c128, _c128, _c128, ctypes.c_int, _f64, _f64]
        lib.orc_lanczos_quadrature_full.restype = ctypes.c_int
        lib.orc_quadrature_resolvent_at.argtypes = [ctypes.c_int, _f64, _f64, ctypes.c_int, _c128, _c128]
        lib.orc_quadrature_resolvent.argtypes = [ctypes.c_int, _f64, _f64, ctypes.c_int, _f64, ctypes.c_double, _c128]
        _lib = lib
    return _lib


def _c(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def num_threads() -> int:
    """Threads the OpenMP loops of the oracle use (OMP_NUM_THREADS or all cores)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


def apply_tda(R, X, rows=None):
    """Y = R X (TDA).  R dense N x N (lower triangle read), X N x k."""
    R = _c(R); X = _c(X)
    N, k = X.shape
    Y = np.zeros((N, k), dtype=np.complex128)
    r0, r1 = (0, N) if rows is None else rows
    _load().orc_apply_tda_rows(N, k, R, X, Y, r0, r1)
    return Y if rows is None else Y[r0:r1]


def apply_full(R, C, X, rows=None):
    """[Y1;Y2] = [[R, C], [-C^H, -R^*]] [X1;X2] (Eq. 1 with PAPER.md:26)."""
    R = _c(R); C = _c(C); X = _c(X)
    N = R.shape[0]
    k = X.shape[1]
    assert X.shape[0] == 2 * N
    Y = np.zeros((2 * N, k), dtype=np.complex128)
    r0, r1 = (0, 2 * N) if rows is None else rows
    _load().orc_apply_full_rows(N, k, R, C, X, Y, r0, r1)
    return Y if rows is None else Y[r0:r1]


def apply_half(R, C, X, sign):
    """P(X) (sign=+1) or M(X) (sign=-1): R X + sign C conj(X) on N-row half vectors."""
    R = _c(R); C = _c(C); X = _c(X)
    N, k = X.shape
    Y = np.zeros((N, k), dtype=np.complex128)
    _load().orc_apply_half(N, k, int(sign), R, C, X, Y)
    return Y


def rows_times_block(Hrows, X):
    Hrows = _c(Hrows); X = _c(X)
    nr, n = Hrows.shape
    k = X.shape[1]
    Y = np.zeros((nr, k), dtype=np.complex128)
    _load().orc_rows_times_block(nr, n, k, Hrows, X, Y)
    return Y


def jacobi_herm(A):
    """Cyclic Jacobi eigen-decomposition of a Hermitian matrix: (w ascending, V columns)."""
    A = _c(A).copy()
    n = A.shape[0]
    w = np.zeros(n)
    V = np.zeros((n, n), dtype=np.complex128)
    sweeps = _load().orc_jacobi_herm(n, A, w, V)
    if sweeps < 0:
        raise RuntimeError("oracle Jacobi did not converge")
    return w, V


def build_Mr(R, C):
    R = _c(R); C = _c(C)
    N = R.shape[0]
    Mr = np.zeros((2 * N, 2 * N))
    _load().orc_build_Mr(N, R, C, Mr)
    return Mr


def bse_direct(R, C, want_vectors=True):
    """The paper's section-2.1 route (Eq. 2-4): all 2N eigenvalues (ascending) and right eigenvectors."""
    R = _c(R); C = _c(C)
    N = R.shape[0]
    om = np.zeros(2 * N)
    V = np.zeros((2 * N, 2 * N), dtype=np.complex128) if want_vectors else None
    rc = _load().orc_bse_direct(N, R, C, None, om, V.ctypes.data if want_vectors else None)
    if rc == 1:
        raise np.linalg.LinAlgError("M_r is not positive definite (PAPER.md:49 precondition)")
    if rc:
        raise RuntimeError("oracle direct route failed")
    return om, V


def block_cgs2(V, W):
    """W = V h + Q B with V^H Q = 0, Q^H Q = I, B upper triangular, positive diagonal."""
    V = _c(V); W = _c(W)
    N, m = V.shape
    k = W.shape[1]
    Q = np.zeros((N, k), dtype=np.complex128)
    h = np.zeros((m, k), dtype=np.complex128)
    B = np.zeros((k, k), dtype=np.complex128)
    rank = _load().orc_block_cgs2(N, m, k, V, W, Q, h, B)
    return Q, h, B, rank


def lanczos_tda(R, nev, tol, v0, maxit=None, check=10):
    R = _c(R)
    N = R.shape[0]
    maxit = N if maxit is None else maxit
    w = np.zeros(nev); Vec = np.zeros((N, nev), dtype=np.complex128); res = np.zeros(nev)
    steps = _load().orc_lanczos_tda(N, R, nev, tol, maxit, check, _c(v0).reshape(N), w, Vec, res)
    return w, Vec, res, steps


def tridiag_ql(d, e, want_vectors=True):
    """Eigenvalues (ascending) and eigenvectors (columns) of the real symmetric tridiagonal matrix tridiag(e, d, e)."""
    d = np.ascontiguousarray(d, dtype=np.float64); e = np.ascontiguousarray(e, dtype=np.float64)
    m = len(d)
    assert len(e) >= m - 1
    e = np.ascontiguousarray(np.concatenate([e, [0.0]])[:max(m, 1)])
    w = np.zeros(m)
    Z = np.zeros((m, m)) if want_vectors else None
    if _load().orc_tridiag_ql(m, d, e, w, Z.ctypes.data if want_vectors else None):
        raise RuntimeError("oracle tridiagonal QL did not converge")
    return w, Z


def lanczos_full(R, C, nev, tol, x0, maxit=None, check=10, minit=0):
    """nev lowest positive omega of Eq. (1) with Sigma-orthonormal eigenvectors (counted as eigenvectors of H: the
    second copy of every omega^2 that G = M o P has on R^2N is recognised by its vector and dropped, reading R1).
    minit: do not stop before this many steps (tests run far past first convergence)."""
    R = _c(R); C = _c(C)
    N = R.shape[0]
    maxit = 2 * N if maxit is None else maxit
    om = np.zeros(nev); Vec = np.zeros((2 * N, nev), dtype=np.complex128); res = np.zeros(nev)
    steps = _load().orc_lanczos_full(N, R, C, nev, tol, maxit, check, minit, _c(x0).reshape(N), om, Vec, res)
    if steps == -1000000:
        raise np.linalg.LinAlgError("Omega is not positive definite")
    return om, Vec, res, steps


def lanczos_full_gruning(R, C, nev, tol, x0, maxit=None, check=10, minit=0, n_ritz=0):
    """The "Gruning" variant (reading R9): Lanczos on H itself in the Omega inner product, T = tridiag(beta, 0, beta).
    Same outputs as lanczos_full; steps counts Lanczos vectors (one half apply each).  n_ritz > 0: also returns the n_ritz lowest
    positive Ritz values of the last projected matrix."""
    R = _c(R); C = _c(C)
    N = R.shape[0]
    maxit = 4 * N if maxit is None else maxit
    om = np.zeros(nev); Vec = np.zeros((2 * N, nev), dtype=np.complex128); res = np.zeros(nev)
    ritz = np.zeros(max(n_ritz, 1))
    steps = _load().orc_lanczos_full_gruning(N, R, C, nev, tol, maxit, check, minit, _c(x0).reshape(N), om, Vec, res,
                                             ritz.ctypes.data if n_ritz > 0 else None, n_ritz)
    if steps == -1000000:
        raise np.linalg.LinAlgError("Omega is not positive definite")
    return (om, Vec, res, steps, ritz[:n_ritz]) if n_ritz > 0 else (om, Vec, res, steps)


def lanczos_quadrature(R, d, steps):
    """Lanczos coefficients (alpha[steps], beta[steps+1], beta[0] = |d|) of the quadrature of PAPER.md:65 (TDA)."""
    R = _c(R)
    N = R.shape[0]
    alpha = np.zeros(steps); beta = np.zeros(steps + 1)
    done = _load().orc_lanczos_quadrature(N, R, _c(d).reshape(N), steps, alpha, beta)
    return alpha[:done], beta[:done + 1]


def quadrature_resolvent(alpha, beta, omega, eta):
    """d^H (omega + i eta - R)^{-1} d from the continued fraction of the Jacobi matrix."""
    alpha = np.ascontiguousarray(alpha, dtype=np.float64); beta = np.ascontiguousarray(beta, dtype=np.float64)
    omega = np.ascontiguousarray(omega, dtype=np.float64)
    out = np.zeros(len(omega), dtype=np.complex128)
    _load().orc_quadrature_resolvent(len(alpha), alpha, beta, len(omega), omega, float(eta), out)
    return out


def lanczos_quadrature_full(R, C, d, steps):
    """Full-mode Lanczos-with-quadrature coefficients (PAPER.md:65 on the operator of Eq. 1): the recurrence of G = M o P
    in the inner product Re(a^H P(b)) started at d; beta[0] = sqrt(Re(d^H P(d)))."""
    R, C = _c(R), _c(C)
    N = R.shape[0]
    alpha = np.zeros(steps); beta = np.zeros(steps + 1)
    done = _load().orc_lanczos_quadrature_full(N, R, C, _c(d).reshape(N), steps, alpha, beta)
    if done == -1000000:
        raise np.linalg.LinAlgError("Omega is not positive definite")
    return alpha[:done], beta[:done + 1]


def quadrature_resolvent_full(alpha, beta, omega, eta):
    """u^H Sigma (omega + i eta - H)^{-1} u, u = [d; conj d]:  2 beta_0^2 [(z^2 - T)^{-1}]_00."""
    alpha = np.ascontiguousarray(alpha, dtype=np.float64); beta = np.ascontiguousarray(beta, dtype=np.float64)
    s = np.ascontiguousarray((np.asarray(omega, dtype=np.float64) + 1j * float(eta)) ** 2, dtype=np.complex128)
    out = np.zeros(len(s), dtype=np.complex128)
    _load().orc_quadrature_resolvent_at(len(alpha), alpha, beta, len(s), s, out)
    return 2.0 * out


def round_c64(A):
    """The complex64-stored operand: every real and imaginary part rounded to
    the nearest IEEE binary32 value, ties to even; returned as complex128."""
    A = _c(A)
    out = np.empty_like(A)
    _load().orc_round_c64(A.size, A.reshape(-1), out.reshape(-1))
    return out
