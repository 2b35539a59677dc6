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
    plane in the mode tables of RoleReal in apply_tiles.cuh is an O(1) error here."""
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
    assert b.bse_layout(N, b.STORE_REAL_FORM_C64) == b.bse_layout(N, b.STORE_C64)


# ---- binary32 planes (BSE_STORE_REAL_FORM_C64): the operator is R' = (S32 + D32)/2, C' = (S32 - D32)/2 with
# ---- S32 = fl32(fl32(R) + fl32(C)), D32 = fl32(fl32(R) - fl32(C))  (include/bse.h) -- built here from oracle.round_c64

def _handle64(R, C):
    import paper_2504_10096_b200 as b
    N = R.shape[0]
    rt = b.bse_pack_from_dense(to_dev(R), N, 0, storage=b.STORE_C64)
    ct = b.bse_pack_from_dense(to_dev(C), N, 1, storage=b.STORE_C64)
    b.bse_to_real_form(rt, ct, N, storage=b.STORE_C64)
    return b.Bse(b.MODE_FULL, N, rt, ct, storage=b.STORE_REAL_FORM_C64)


def _operator64(orc, R, C):
    R32, C32 = orc.round_c64(R), orc.round_c64(C)
    S32, D32 = orc.round_c64(R32 + C32), orc.round_c64(R32 - C32)      # the FP64 sum of two binary32 values is exact
    return (S32 + D32) / 2, (S32 - D32) / 2, R32, C32


@pytest.mark.parametrize("N", [64, 200, 448])
@pytest.mark.parametrize("k", [1, 4, 8, 11])
def test_c64_planes_half_apply_matches_oracle(orc, N, k):
    R, C = _pair(N, 31)
    Rp, Cp, R32, C32 = _operator64(orc, R, C)
    h = _handle64(R, C)
    x = gen.block_X(N, k, 24)
    for sign in (+1, -1):
        Y = to_host(h.apply_half(to_dev(x), sign))
        assert relerr(Y, orc.apply_half(Rp, Cp, x, sign)) <= TOL_APPLY
        e = relerr(Y, orc.apply_half(R32, C32, x, sign))
        assert 1e-11 < e < 1e-6            # one binary32 ulp per entry away from the rounded (R, C), not equal to it
    X = gen.block_X(2 * N, min(k, 5), 25)
    assert relerr(to_host(h.apply(to_dev(X))), orc.apply_full(Rp, Cp, X)) <= TOL_APPLY


def test_c64_planes_many_units_and_solve(orc):
    from test_gpu_solve import _check_full
    N, nev, k = 192, 8, 8
    R = gen.dense_R(N, 2, sigma=1.0); C = gen.dense_C(N, 2)
    Rp, Cp, _, _ = _operator64(orc, R, C)
    res = _handle64(R, C).solve(nev, k, tol=1e-9, seed=1)
    omd, _ = orc.bse_direct(Rp, Cp, want_vectors=False)
    _check_full(orc, Rp, Cp, res, nev, omd[N:])
    # many units per CTA: N = 4096, dense host matrices (134 MB each) packed through the binary32 store
    N = 4096
    R = gen.dense_R(N, 3, sigma=1.0); C = gen.dense_C(N, 3)
    Rp, Cp, _, _ = _operator64(orc, R, C)
    h = _handle64(R, C)
    X = gen.block_X(N, 8, 5)
    rows = np.unique(np.concatenate([np.arange(0, N, 397), [63, 64, N - 65, N - 1]]))
    for sign in (+1, -1):
        ref = orc.rows_times_block(Rp[rows], X) + sign * orc.rows_times_block(Cp[rows], X.conj())
        for _ in range(4):
            assert relerr(to_host(h.apply_half(to_dev(X), sign))[rows], ref) <= TOL_APPLY


def test_config1_vs_oracle_golden_with_the_real_form_store(orc):
    """BASELINE.json config 1 (full N = 2048, nev = 20, k = 4) through the real-form store: same stored oracle values,
    residuals and Sigma-orthonormality as test_gpu_solve.test_config1_full_vs_oracle_golden."""
    import os
    from test_gpu_solve import _check_full, _golden
    if not os.path.exists(os.path.join(os.path.dirname(__file__), "golden", "oracle_config1.txt")):
        pytest.skip("tests/golden/oracle_config1.txt not generated yet")
    cfg = gen.CONFIGS[1]
    N, nev, k = cfg["N"], cfg["nev"], cfg["k"]
    R = gen.dense_R(N, 1, sigma=cfg["sigma"]); C = gen.dense_C(N, 1)
    res = _handle(R, C).solve(nev, k, tol=1e-8, seed=1)
    gold = _golden("oracle_config1.txt")
    distinct = [gold[0]]
    for x in gold[1:]:
        if x - distinct[-1] > 1e-7 * x:
            distinct.append(x)
    _check_full(orc, R, C, res, nev, np.array(distinct))
