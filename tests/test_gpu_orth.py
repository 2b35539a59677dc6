"""bse_orth (block CGS2 + intra-block orthonormalisation) against the oracle's factorisation and its defining
properties (north_star: ||V^H V - I|| <= 1e-12)."""
import numpy as np
import pytest

import bse_inputs as gen
from gpu_util import pack, to_dev, to_host

pytestmark = pytest.mark.gpu
TOL_ORTH = 1e-12


def _tda_handle(N):
    import paper_2504_10096_b200 as b
    return b.Bse(b.MODE_TDA, N, pack(np.eye(N, dtype=complex), 0))


def _check_factorisation(V, W_in, Q, h, B, k):
    assert np.linalg.norm(Q.conj().T @ Q - np.eye(k)) <= TOL_ORTH
    if V is not None:
        assert np.linalg.norm(V.conj().T @ Q) <= TOL_ORTH
        rec = V @ h + Q @ B
    else:
        rec = Q @ B
    assert np.linalg.norm(W_in - rec) / np.linalg.norm(W_in) <= 1e-13
    assert np.allclose(B, np.triu(B), atol=0) and np.all(np.diag(B).real > 0) and np.allclose(np.diag(B).imag, 0)


@pytest.mark.parametrize("N,m,k", [(500, 12, 4), (64, 3, 1), (1030, 70, 8), (333, 9, 5)])
def test_euclidean_orth_matches_oracle(orc, N, m, k):
    V, _ = np.linalg.qr(gen.block_X(N, m, 1))
    W = gen.block_X(N, k, 2)
    h_ = _tda_handle(N)
    Wd = to_dev(W)
    hc, bf, rank = h_.orth(to_dev(V), Wd)
    Q, h, B = to_host(Wd), to_host(hc), to_host(bf)
    assert rank == k
    _check_factorisation(V, W, Q, h, B, k)
    Qo, ho, Bo, ranko = orc.block_cgs2(V, W)
    assert ranko == k
    assert np.max(np.abs(Q - Qo)) < 1e-10 and np.max(np.abs(B - Bo)) < 1e-10 and np.max(np.abs(h - ho)) < 1e-12


def test_no_basis(orc):
    N, k = 300, 4
    W = gen.block_X(N, k, 3)
    Wd = to_dev(W)
    hc, bf, rank = _tda_handle(N).orth(None, Wd)
    Q, B = to_host(Wd), to_host(bf)
    assert rank == k
    _check_factorisation(None, W, Q, None, B, k)


def test_nearly_dependent_on_basis_needs_second_pass(orc):
    N, m, k = 600, 20, 4
    V, _ = np.linalg.qr(gen.block_X(N, m, 1))
    W = V @ gen.block_X(m, k, 3) + 1e-10 * gen.block_X(N, k, 2)
    Wd = to_dev(W)
    hc, bf, rank = _tda_handle(N).orth(to_dev(V), Wd)
    assert rank == k
    _check_factorisation(V, W, to_host(Wd), to_host(hc), to_host(bf), k)


def test_ill_conditioned_block_takes_the_columnwise_path(orc):
    N, m, k = 400, 6, 4
    V, _ = np.linalg.qr(gen.block_X(N, m, 1))
    W = gen.block_X(N, k, 5)
    W[:, 3] = W[:, 1] + 1e-9 * W[:, 3]            # kappa ~ 1e9: CholQR alone would fail
    Wd = to_dev(W)
    hc, bf, rank = _tda_handle(N).orth(to_dev(V), Wd)
    assert rank == k
    _check_factorisation(V, W, to_host(Wd), to_host(hc), to_host(bf), k)


def test_rank_deficient_block(orc):
    N, m, k = 256, 5, 3
    V, _ = np.linalg.qr(gen.block_X(N, m, 4))
    W = gen.block_X(N, k, 5)
    W[:, 2] = W[:, 0] * (1 + 2j) + V[:, 1]
    Wd = to_dev(W)
    hc, bf, rank = _tda_handle(N).orth(to_dev(V), Wd)
    Q, h, B = to_host(Wd), to_host(hc), to_host(bf)
    assert rank == 2
    # the replaced column is still orthonormal to everything, and the factorisation still reproduces W
    assert np.linalg.norm(Q.conj().T @ Q - np.eye(k)) <= TOL_ORTH
    assert np.linalg.norm(V.conj().T @ Q) <= TOL_ORTH
    assert abs(B[2, 2]) == 0
    assert np.linalg.norm(W - V @ h - Q @ B) / np.linalg.norm(W) <= 1e-13


def test_P_inner_product_orth(orc):
    # full mode, reading S4/S10: real inner product <x, y> = Re(x^H P(y)), real coefficients, PW kept consistent
    import paper_2504_10096_b200 as b
    N, m, k = 320, 10, 4
    R = gen.dense_R(N, 1, sigma=1.0); C = gen.dense_C(N, 1)
    h_ = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    X = gen.block_X(N, m, 6)
    PX = orc.apply_half(R, C, X, +1)
    L = np.linalg.cholesky((X.conj().T @ PX).real)
    Li = np.linalg.inv(L).T
    X, PX = X @ Li, PX @ Li                                     # P-orthonormal basis
    assert np.linalg.norm((X.conj().T @ PX).real - np.eye(m)) < 1e-12
    W = gen.block_X(N, k, 7)
    PW = orc.apply_half(R, C, W, +1)
    Wd, PWd = to_dev(W), to_dev(PW)
    hc, bf, rank = h_.orth(to_dev(X), Wd, to_dev(PX), PWd)
    Q, PQ, h, B = to_host(Wd), to_host(PWd), to_host(hc), to_host(bf)
    assert rank == k
    assert np.max(np.abs(h.imag)) == 0 and np.max(np.abs(B.imag)) == 0
    assert np.linalg.norm((PX.conj().T @ Q).real) <= TOL_ORTH
    assert np.linalg.norm((Q.conj().T @ PQ).real - np.eye(k)) <= TOL_ORTH
    assert np.linalg.norm(PQ - orc.apply_half(R, C, Q, +1)) / np.linalg.norm(PQ) <= 1e-12
    assert np.linalg.norm(W - X @ h.real - Q @ B.real) / np.linalg.norm(W) <= 1e-13


def test_P_inner_product_rank_deficient_and_ill_conditioned(orc):
    """Full-mode inner product, column-wise path: one column nearly dependent on another (kappa ~ 1e6), one exactly
    dependent on the basis and a previous column.  Coefficients stay real and the factorisation holds to rounding;
    PW is carried by linear combination (include/bse.h), so P-orthonormality and PW = P(W) hold to kappa * eps."""
    import paper_2504_10096_b200 as b
    N, m, k = 256, 6, 4
    R = gen.dense_R(N, 4, sigma=1.0); C = gen.dense_C(N, 4)
    h_ = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    X = gen.block_X(N, m, 6)
    PX = orc.apply_half(R, C, X, +1)
    Li = np.linalg.inv(np.linalg.cholesky((X.conj().T @ PX).real)).T
    X, PX = X @ Li, PX @ Li
    W = gen.block_X(N, k, 7)
    W[:, 2] = W[:, 0] + 1e-6 * W[:, 2]                 # ill-conditioned pair
    W[:, 3] = 2.0 * W[:, 1] - 0.5 * X[:, 2]            # exactly dependent (real combination)
    PW = orc.apply_half(R, C, W, +1)
    Wd, PWd = to_dev(W), to_dev(PW)
    hc, bf, rank = h_.orth(to_dev(X), Wd, to_dev(PX), PWd)
    Q, PQ, h, B = to_host(Wd), to_host(PWd), to_host(hc), to_host(bf)
    assert rank == 3 and B[3, 3] == 0
    assert np.max(np.abs(h.imag)) == 0 and np.max(np.abs(B.imag)) == 0
    PQ_true = orc.apply_half(R, C, Q, +1)
    assert np.linalg.norm((PX.conj().T @ Q).real) <= 1e-11
    assert np.linalg.norm(PQ - PQ_true) / np.linalg.norm(PQ) <= 1e-9                        # kappa * eps
    assert np.linalg.norm((Q.conj().T @ PQ).real - np.eye(k)) <= 1e-9
    assert np.linalg.norm((Q.conj().T @ PQ_true).real - np.eye(k)) <= 1e-9
    assert np.linalg.norm(W - X @ h.real - Q @ B.real) / np.linalg.norm(W) <= 1e-12
