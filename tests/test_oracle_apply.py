"""Pins for the oracle's operator apply (not the CUDA path).  Each test is chosen so that a plausible
mistake (dropped term, wrong sign or conjugate, transposed operand, wrong block) fails it."""
import numpy as np
import pytest

import bse_inputs as gen


def _rand_herm(n, seed):
    A = gen.block_X(n, n, seed)
    return (A + A.conj().T) / 2


def _rand_sym(n, seed):
    A = gen.block_X(n, n, seed)
    return (A + A.T) / 2


def test_identity_and_diagonal_are_exact(orc):
    N, k = 37, 3
    X = gen.block_X(N, k, 5)
    assert np.array_equal(orc.apply_tda(np.eye(N), X), X)
    d = np.linspace(-2, 3, N)
    # products are formed in long double then rounded once more: allow 1 ulp
    assert np.allclose(orc.apply_tda(np.diag(d), X), d[:, None] * X, rtol=3e-16, atol=0)


def test_unit_impulses_tda(orc):
    # PAPER.md:20 R = R^dagger: a single stored lower entry (i, j) acts as R_ij on row i and conj(R_ij) on row j
    N, k = 9, 2
    X = gen.block_X(N, k, 7)
    for (i, j) in [(5, 2), (8, 0), (3, 3), (1, 0)]:
        R = np.zeros((N, N), dtype=complex)
        R[i, j] = 0.7 - 1.3j
        Y = orc.apply_tda(R, X)
        exp = np.zeros_like(X)
        if i == j:
            exp[i] = 0.7 * X[i]            # diagonal of a Hermitian matrix is real
        else:
            exp[i] = (0.7 - 1.3j) * X[j]
            exp[j] = (0.7 + 1.3j) * X[i]
        assert np.allclose(Y, exp, rtol=0, atol=1e-15)


def test_upper_triangle_is_ignored(orc):
    N, k = 20, 2
    R = _rand_herm(N, 1)
    X = gen.block_X(N, k, 2)
    garbage = R.copy()
    garbage[np.triu_indices(N, 1)] = 99.0
    assert np.array_equal(orc.apply_tda(R, X), orc.apply_tda(garbage, X))


def test_tda_matches_numpy_matmul(orc):
    N, k = 150, 5
    R = _rand_herm(N, 11)
    X = gen.block_X(N, k, 12)
    Y = orc.apply_tda(R, X)
    ref = R @ X
    assert np.linalg.norm(Y - ref) / np.linalg.norm(ref) < 1e-14
    # Hermitian adjoint identity X^H (R Z) = (R X)^H Z
    Z = gen.block_X(N, k, 13)
    assert np.allclose(X.conj().T @ orc.apply_tda(R, Z), orc.apply_tda(R, X).conj().T @ Z, atol=1e-11)


def test_full_unit_impulses(orc):
    # Eq. (1) with A = R^*, C = C^T: check every block's sign and conjugation separately
    N, k = 6, 2
    X = gen.block_X(2 * N, k, 3)
    X1, X2 = X[:N], X[N:]
    a = 0.3 + 0.9j
    i, j = 4, 1
    R = np.zeros((N, N), dtype=complex); C = np.zeros((N, N), dtype=complex)
    R[i, j] = a
    Y = orc.apply_full(R, C, X)
    exp = np.zeros_like(X)
    exp[i] += a * X1[j]; exp[j] += np.conj(a) * X1[i]                      # R block
    exp[N + i] += -np.conj(a) * X2[j]; exp[N + j] += -a * X2[i]            # -R^* block
    assert np.allclose(Y, exp, atol=1e-15)
    R[:] = 0; C[i, j] = a
    Y = orc.apply_full(R, C, X)
    exp = np.zeros_like(X)
    exp[i] += a * X2[j]; exp[j] += a * X2[i]                               # C block (symmetric)
    exp[N + i] += -np.conj(a) * X1[j]; exp[N + j] += -np.conj(a) * X1[i]   # -C^dagger = -C^*
    assert np.allclose(Y, exp, atol=1e-15)


def _H_dense(R, C):
    return np.block([[R, C], [-C.conj().T, -R.conj()]])


def test_full_matches_numpy_block_operator(orc):
    N, k = 60, 3
    R = _rand_herm(N, 21); C = _rand_sym(N, 22)
    X = gen.block_X(2 * N, k, 23)
    ref = _H_dense(R, C) @ X
    Y = orc.apply_full(R, C, X)
    assert np.linalg.norm(Y - ref) / np.linalg.norm(ref) < 1e-14


def test_paper_identity_QHQ_equals_minus_i_J_Mr(orc):
    # PAPER.md:40-47 (Eq. 2-3): Q^H H Q = -i J M_r with Q = (1/sqrt2)[[I, -iI], [I, iI]]
    N = 24
    R = _rand_herm(N, 31); C = _rand_sym(N, 32)
    Mr = orc.build_Mr(R, C)
    I_ = np.eye(N)
    Q = np.block([[I_, -1j * I_], [I_, 1j * I_]]) / np.sqrt(2)
    J = np.block([[0 * I_, I_], [-I_, 0 * I_]])
    # H assembled column by column through the ORACLE apply (not numpy)
    H = orc.apply_full(R, C, np.eye(2 * N, dtype=complex))
    assert np.allclose(Mr, Mr.T)
    lhs = Q.conj().T @ H @ Q
    assert np.linalg.norm(lhs + 1j * J @ Mr) < 1e-13 * np.linalg.norm(H)


def test_half_apply_is_upper_half_of_structured_vectors(orc):
    # reading S4: H [x; conj x] = [P(x); -conj P(x)],  H [y; -conj y] = [M(y); conj M(y)]
    N, k = 40, 2
    R = _rand_herm(N, 41); C = _rand_sym(N, 42)
    x = gen.block_X(N, k, 43)
    P = orc.apply_half(R, C, x, +1)
    M = orc.apply_half(R, C, x, -1)
    Hp = orc.apply_full(R, C, np.vstack([x, x.conj()]))
    Hm = orc.apply_full(R, C, np.vstack([x, -x.conj()]))
    assert np.allclose(Hp[:N], P, atol=1e-12) and np.allclose(Hp[N:], -P.conj(), atol=1e-12)
    assert np.allclose(Hm[:N], M, atol=1e-12) and np.allclose(Hm[N:], M.conj(), atol=1e-12)
    assert np.allclose(P, R @ x + C @ x.conj(), atol=1e-12)
    assert np.allclose(M, R @ x - C @ x.conj(), atol=1e-12)


def test_rows_subset_and_row_panel(orc):
    N, k = 64, 3
    R = _rand_herm(N, 51)
    X = gen.block_X(N, k, 52)
    full = orc.apply_tda(R, X)
    assert np.array_equal(orc.apply_tda(R, X, rows=(10, 17)), full[10:17])
    assert np.allclose(orc.rows_times_block(R[10:17], X), full[10:17], atol=1e-13)


def test_table2_byte_accounting():
    # the dense complex64 operator is N^2 * 8 B (x2 with coupling)
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_table2_memory.txt")
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        N, res, cpl = line.split()
        N = int(N)
        assert abs(N * N * 8 / 2**30 - float(res)) < 0.006
        assert abs(2 * N * N * 8 / 2**30 - float(cpl)) < 0.011
