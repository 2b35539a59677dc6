"""Real-form full-mode store (BSE_STORE_REAL_FORM: S = R + C, D = R - C, the blocks of M_r in Eq. 3):
the same operator as the complex store, so every result is compared with the oracle on (R, C) at the usual tolerances."""
import numpy as np
import pytest

import bse_inputs as gen
from gpu_util import pack, relerr, to_dev, to_host

pytestmark = pytest.mark.gpu
TOL_APPLY = 1e-12


def _handle(R, C):
    import paper_2504_10096_b200 as b
    N = R.shape[0]
    rt, ct = b.bse_to_real_form(pack(R, 0), pack(C, 1), N)
    return b.Bse(b.MODE_FULL, N, rt, ct, storage=b.STORE_REAL_FORM)


def _pair(N, seed):
    Np = N if N % 16 == 0 else N + 16 - N % 16
    return gen.dense_R(Np, seed, sigma=1.0)[:N, :N], gen.dense_C(N, seed)


@pytest.mark.parametrize("N", [64, 100, 200, 448, 1024])
@pytest.mark.parametrize("k", [1, 3, 4, 5, 8, 11])
def test_half_apply_matches_oracle(orc, N, k):
    R, C = _pair(N, 21)
    h = _handle(R, C)
    x = gen.block_X(N, k, 24)
    for sign in (+1, -1):
        Y, ref = to_host(h.apply_half(to_dev(x), sign)), orc.apply_half(R, C, x, sign)
        assert relerr(Y, ref) <= TOL_APPLY
        for c in range(k):
            assert relerr(Y[:, c], ref[:, c]) <= TOL_APPLY


@pytest.mark.parametrize("N,k", [(64, 1), (200, 4), (448, 6), (320, 9)])
def test_general_apply_matches_oracle(orc, N, k):
    R, C = _pair(N, 22)
    h = _handle(R, C)
    X = gen.block_X(2 * N, k, 23)
    assert relerr(to_host(h.apply(to_dev(X))), orc.apply_full(R, C, X)) <= TOL_APPLY


def test_unit_impulses_every_block_sign_and_conjugation(orc):
    """One non-zero entry of R or C at a time (diagonal tile, off-diagonal tile, tile border): a wrong sign or a swapped
    plane in the mode tables of apply_kernel_real.cuh is an O(1) error here."""
    N = 130
    x = gen.block_X(N, 2, 5)
    for (i, j) in [(0, 0), (5, 3), (63, 0), (64, 63), (100, 7), (129, 64), (129, 129)]:
        for which in ("R", "C"):
            R = np.zeros((N, N), dtype=complex); C = np.zeros((N, N), dtype=complex)
            val = 0.7 - 1.3j
            if which == "R":
                R[i, j] = val; R[j, i] = np.conj(val)
                if i == j: R[i, i] = 0.9
            else:
                C[i, j] = val; C[j, i] = val
            h = _handle(R, C)
            for sign in (+1, -1):
                Y, ref = to_host(h.apply_half(to_dev(x), sign)), orc.apply_half(R, C, x, sign)
                assert np.max(np.abs(Y - ref)) <= 1e-14 * np.max(np.abs(ref)), (i, j, which, sign)


@pytest.mark.parametrize("kind", ["real_x", "imag_x", "real_RC", "imag_C"])
def test_special_operands(orc, kind):
    N, k = 330, 8
    R, C = _pair(N, 61)
    x = gen.block_X(N, k, 63)
    if kind == "real_x":
        x = x.real + 0j
    elif kind == "imag_x":
        x = 1j * x.imag
    elif kind == "real_RC":
        R, C = R.real + 0j, C.real + 0j
    else:
        C = 1j * C.imag
    h = _handle(R, C)
    for sign in (+1, -1):
        assert relerr(to_host(h.apply_half(to_dev(x), sign)), orc.apply_half(R, C, x, sign)) <= TOL_APPLY


@pytest.mark.parametrize("N,k,reps", [(4096, 4, 10), (8192, 8, 4)])
def test_many_units_per_cta_sampled_rows(orc, N, k, reps):
    import paper_2504_10096_b200 as b
    rt, ct = b.bse_fill_synthetic(N, 0, 2, 1.0, 16), b.bse_fill_synthetic(N, 1, 2, 0.0, 16)
    b.bse_to_real_form(rt, ct, N)
    h = b.Bse(b.MODE_FULL, N, rt, ct, storage=b.STORE_REAL_FORM)
    X = gen.block_X(N, k, 5)
    rows = np.unique(np.concatenate([np.arange(0, N, 397), [63, 64, N - 65, N - 1]]))
    RX = orc.rows_times_block(gen.rows_R(N, 2, rows, 1.0, 16), X)
    CX = orc.rows_times_block(gen.rows_C(N, 2, rows), X.conj())
    for _ in range(reps):
        for sign in (+1, -1):
            Y = to_host(h.apply_half(to_dev(X), sign))
            assert relerr(Y[rows], RX + sign * CX) <= TOL_APPLY


@pytest.mark.parametrize("k", [4, 8])
def test_solve_vs_direct_route(orc, k):
    from test_gpu_solve import _check_full
    N, nev = 192, 8
    R = gen.dense_R(N, 2, sigma=1.0); C = gen.dense_C(N, 2)
    res = _handle(R, C).solve(nev, k, tol=1e-9, seed=1)
    omd, _ = orc.bse_direct(R, C, want_vectors=False)
    _check_full(orc, R, C, res, nev, omd[N:])


def test_quadrature_matches_oracle(orc):
    import torch
    N, steps = 192, 30
    R, C = _pair(N, 5)
    d = gen.block_X(N, 1, 6)[:, 0]
    alpha, beta = _handle(R, C).lanczos_quadrature(torch.from_numpy(d).cuda(), steps)
    ao, bo = orc.lanczos_quadrature_full(R, C, d, steps)
    sc = np.max(np.abs(ao))
    assert np.max(np.abs(alpha[:15] - ao[:15])) <= 1e-10 * sc and np.max(np.abs(beta[:16] - bo[:16])) <= 1e-10 * sc


def test_real_form_is_full_mode_only():
    import paper_2504_10096_b200 as b
    N = 64
    R, C = _pair(N, 3)
    with pytest.raises(b.BseError):
        b.Bse(b.MODE_TDA, N, pack(R, 0), storage=b.STORE_REAL_FORM)
    assert b.bse_layout(N, b.STORE_REAL_FORM) == b.bse_layout(N, b.STORE_C128)
