"""-m gpu parity tests for the complex64-stored operand (the paper's matrices
are single precision).  The operator IS the binary32-rounded matrix (oracle.round_c64); vectors, arithmetic and
results stay complex128, so the tolerances are the complex128 ones."""
import numpy as np
import pytest

import bse_inputs as gen
from gpu_util import relerr, to_dev, to_host


def _bits(a):
    return np.ascontiguousarray(a).view(np.float64)

pytestmark = pytest.mark.gpu

TOL_APPLY = 1e-12     # north_star: apply, normwise relative
TOL_EIG = 1e-10       # north_star: eigenvalues, relative
TOL_RES = 1e-8        # north_star: residuals, relative to ||H||


def _pack64(A, which):
    import paper_2504_10096_b200 as b
    return b.bse_pack_from_dense(to_dev(A), A.shape[0], which, storage=b.STORE_C64)


@pytest.mark.parametrize("N", [1, 8, 64, 100, 257])
@pytest.mark.parametrize("which", [0, 1])
def test_pack_rounds_to_nearest_even_bit_exact(orc, N, which):
    import paper_2504_10096_b200 as b
    A = gen.dense_R(N + (-N) % 16, 3, sigma=1.0)[:N, :N] if which == 0 else gen.dense_C(N, 3)
    A = A * (10.0 ** np.linspace(-3, 3, N))[:, None] * (10.0 ** np.linspace(-3, 3, N))[None, :]   # spread exponents
    A = A + A.conj().T if which == 0 else A + A.T
    t = _pack64(A, which)
    assert t.numel() == b.bse_layout(N, b.STORE_C64)[2] == b.bse_layout(N)[2] // 2
    back = b.bse_unpack_to_dense(t, N, which, storage=b.STORE_C64).cpu().numpy().T
    want = orc.round_c64(A)
    if which == 0:
        want[np.diag_indices(N)] = want.diagonal().real
    assert np.array_equal(_bits(back), _bits(want))


def test_pack_ties_and_signed_zero(orc):
    import paper_2504_10096_b200 as b
    N = 8
    u = 2.0 ** -24
    vals = np.array([1 + u, 1 + 3 * u, 1 - u / 2, 16777217.0, 2.0 ** -150, 1.5 * 2.0 ** -149, 0.1, -(1 + 3 * u)])
    C = np.zeros((N, N), dtype=np.complex128)
    C[:, 0] = vals + 1j * vals[::-1]; C[0, :] = C[:, 0]
    back = b.bse_unpack_to_dense(_pack64(C, 1), N, 1, storage=b.STORE_C64).cpu().numpy().T
    assert np.array_equal(_bits(back), _bits(orc.round_c64(C)))
    assert back[1, 0].real == 1.0 + 4 * u and back[0, 0].real == 1.0 and back[4, 0].real == 0.0


@pytest.mark.parametrize("N", [64, 100, 320, 1024])
@pytest.mark.parametrize("k", [1, 2, 4, 5, 8])
def test_tda_apply_matches_oracle_on_rounded_operator(orc, N, k):
    import paper_2504_10096_b200 as b
    R = gen.dense_R(N if N % 16 == 0 else N + 16 - N % 16, 11, sigma=0.5)[:N, :N]
    X = gen.block_X(N, k, 12)
    h = b.Bse(b.MODE_TDA, N, _pack64(R, 0), storage=b.STORE_C64)
    Y = to_host(h.apply(to_dev(X)))
    R32 = orc.round_c64(R)
    assert relerr(Y, orc.apply_tda(R32, X)) <= TOL_APPLY
    assert relerr(Y, orc.apply_tda(R, X)) > 1e-10          # and it is NOT the unrounded operator


@pytest.mark.parametrize("N,k", [(64, 1), (200, 4), (448, 6), (448, 1)])
def test_full_apply_and_half_apply_match_oracle_on_rounded_operator(orc, N, k):
    import paper_2504_10096_b200 as b
    Np = N if N % 16 == 0 else N + 16 - N % 16
    R, C = gen.dense_R(Np, 21, sigma=1.0)[:N, :N], gen.dense_C(N, 22)
    h = b.Bse(b.MODE_FULL, N, _pack64(R, 0), _pack64(C, 1), storage=b.STORE_C64)
    R32, C32 = orc.round_c64(R), orc.round_c64(C)
    X = gen.block_X(2 * N, k, 23)
    assert relerr(to_host(h.apply(to_dev(X))), orc.apply_full(R32, C32, X)) <= TOL_APPLY
    x = gen.block_X(N, k, 24)
    for sign in (+1, -1):
        assert relerr(to_host(h.apply_half(to_dev(x), sign)), orc.apply_half(R32, C32, x, sign)) <= TOL_APPLY


@pytest.mark.parametrize("N", [1, 2, 63, 65, 127])
def test_tiny_and_ragged_sizes(orc, N):
    import paper_2504_10096_b200 as b
    R = gen.dense_R(128, 5, sigma=0.0)[:N, :N]
    X = gen.block_X(N, 3, 6)
    Y = to_host(b.Bse(b.MODE_TDA, N, _pack64(R, 0), storage=b.STORE_C64).apply(to_dev(X)))
    assert relerr(Y, orc.apply_tda(orc.round_c64(R), X)) <= TOL_APPLY


def test_device_generator_rounds_the_cpu_generator(orc):
    """bse_fill_synthetic with complex64 storage = the generator's complex128 entry, rounded.  The device generator
    matches the CPU one to a few ulp of FP64, so after rounding the two agree bit for bit except where an entry
    sits within those few ulp of a rounding boundary (probability ~1e-8 per entry)."""
    import paper_2504_10096_b200 as b
    N = 320
    for which, A in ((0, gen.dense_R(N, 7, sigma=1.0, group=64)), (1, gen.dense_C(N, 7))):
        t = b.bse_fill_synthetic(N, which, 7, 1.0 if which == 0 else 0.0, 64, storage=b.STORE_C64)
        back = b.bse_unpack_to_dense(t, N, which, storage=b.STORE_C64).cpu().numpy().T
        want = orc.round_c64(A)
        bad = back != want
        assert bad.sum() <= 2
        assert np.all(np.abs(back - want)[bad] <= 2.0 ** -23 * np.abs(want)[bad])


def _sampled_rows(N):
    base = (np.arange(N // 64)[:, None] * 64 + np.arange(8)[None, :]).reshape(-1)
    extra = (np.arange(97) * 2654435761 % N).astype(np.int64)
    return np.unique(np.concatenate([base, extra]))


@pytest.mark.parametrize("N,k,reps", [(4096, 4, 20), (8192, 1, 6), (16384, 8, 2)])
def test_many_units_per_cta_sampled_rows(orc, N, k, reps):
    """Six 32 KB stages and many units per CTA: the configuration in which a stage-release hazard would show
    (tests/test_gpu_apply.py has the complex128 twin).  The oracle gets the CPU generator's rows, rounded."""
    import paper_2504_10096_b200 as b
    h = b.Bse(b.MODE_TDA, N, b.bse_fill_synthetic(N, 0, 1, 0.0, 16, storage=b.STORE_C64), storage=b.STORE_C64)
    X = gen.block_X(N, k, 12)
    rows = _sampled_rows(N)
    ref = orc.rows_times_block(orc.round_c64(gen.rows_R(N, 1, rows, 0.0, 16)), X)
    Xd = to_dev(X)
    for _ in range(reps):
        Y = to_host(h.apply(Xd))
        assert relerr(Y[rows], ref) <= TOL_APPLY
    Z = gen.block_X(N, k, 13)
    RZ = to_host(h.apply(to_dev(Z)))
    lhs, rhs = X.conj().T @ RZ, Y.conj().T @ Z
    assert np.linalg.norm(lhs - rhs) <= 1e-12 * np.linalg.norm(lhs)


def test_full_many_units_sampled_rows(orc):
    import paper_2504_10096_b200 as b
    N, k = 4096, 4
    S = b.STORE_C64
    h = b.Bse(b.MODE_FULL, N, b.bse_fill_synthetic(N, 0, 2, 1.0, 16, storage=S), b.bse_fill_synthetic(N, 1, 2, storage=S),
              storage=S)
    X = gen.block_X(2 * N, k, 5)
    rows = _sampled_rows(N)[::4]
    Rr, Cr = orc.round_c64(gen.rows_R(N, 2, rows, 1.0, 16)), orc.round_c64(gen.rows_C(N, 2, rows))
    top = np.hstack([Rr, Cr]); bot = np.hstack([-Cr.conj(), -Rr.conj()])      # Eq. 1 with :26
    ref = orc.rows_times_block(np.vstack([top, bot]), X)
    for _ in range(5):
        Y = to_host(h.apply(to_dev(X)))
        assert relerr(np.vstack([Y[rows], Y[N + rows]]), ref) <= TOL_APPLY


def test_solve_tda_config0_on_rounded_operator(orc):
    """Eigenpairs of the rounded matrix to the complex128 tolerances; distance to the unrounded spectrum within
    Weyl's bound ||R32 - R||_2 ('accuracy limited by the data, not the solver')."""
    import paper_2504_10096_b200 as b
    cfg = gen.CONFIGS[0]
    N, nev = cfg["N"], cfg["nev"]
    R = gen.dense_R(N, 1, sigma=1.0, group=cfg["group"])
    R32 = orc.round_c64(R)
    res = b.Bse(b.MODE_TDA, N, _pack64(R, 0), storage=b.STORE_C64).solve(nev, cfg["k"], tol=1e-9, seed=1)
    assert res.status == 0
    w32 = np.linalg.eigvalsh(R32)
    assert np.max(np.abs(res.omega - w32[:nev]) / np.abs(w32[:nev])) <= TOL_EIG
    V = to_host(res.vectors)
    assert np.linalg.norm(V.conj().T @ V - np.eye(nev)) <= 1e-12
    resid = np.linalg.norm(orc.apply_tda(R32, V) - V * res.omega, axis=0)
    assert np.max(resid) <= TOL_RES * np.abs(w32).max()
    dR = np.linalg.norm(R32 - R, 2)
    dw = np.max(np.abs(res.omega - np.linalg.eigvalsh(R)[:nev]))
    assert 1e-12 < dw <= dR


def test_solve_full_on_rounded_operator(orc):
    import paper_2504_10096_b200 as b
    N, nev = 192, 6                      # the oracle's direct route (Jacobi on 2N x 2N) sets the size
    R, C = gen.dense_R(N, 4, sigma=1.0), gen.dense_C(N, 4)
    R32, C32 = orc.round_c64(R), orc.round_c64(C)
    h = b.Bse(b.MODE_FULL, N, _pack64(R, 0), _pack64(C, 1), storage=b.STORE_C64)
    res = h.solve(nev, 4, tol=1e-9, seed=2)
    assert res.status == 0
    w_direct = orc.bse_direct(R32, C32, want_vectors=False)[0][N:N + nev]        # the nev lowest positive omega
    assert np.max(np.abs(res.omega - w_direct) / w_direct) <= TOL_EIG
    V = to_host(res.vectors)
    HV = orc.apply_full(R32, C32, V)
    normH = np.linalg.norm(np.block([[R32, C32], [-C32.conj(), -R32.conj()]]), 2)
    assert np.max(np.linalg.norm(HV - V * res.omega, axis=0)) <= TOL_RES * normH


def test_full_mode_at_paper_largest_size_sampled_rows(orc):
    """Full BSE at N = 98304 (operator dimension 196608; R and C: 77 GB in complex64, too large for one GPU in
    complex128): the size class of the paper's largest system.  Rows of Y = H X sampled across both halves, against
    the oracle fed with the rounded rows of the CPU generator; plus the structure of Eq. 1 through the CUDA path:
    the lower half is minus the conjugate of the upper half applied to the swapped, conjugated input."""
    import torch
    import paper_2504_10096_b200 as b
    N, k, S = 98304, 2, b.STORE_C64
    if torch.cuda.mem_get_info()[0] < 95e9:
        pytest.skip("needs 95 GB of free device memory")
    h = b.Bse(b.MODE_FULL, N, b.bse_fill_synthetic(N, 0, 1, 1.0, 64, storage=S), b.bse_fill_synthetic(N, 1, 1, storage=S),
              storage=S)
    X = gen.block_X(2 * N, k, 12)
    rows = np.unique(np.concatenate([(np.arange(24) * 2654435761 % N), [0, 63, 64, N - 64, N - 1],
                                     np.arange(8) + 64 * 777]).astype(np.int64))
    Rr, Cr = orc.round_c64(gen.rows_R(N, 1, rows, 1.0, 64)), orc.round_c64(gen.rows_C(N, 1, rows))
    top = np.hstack([Rr, Cr]); bot = np.hstack([-Cr.conj(), -Rr.conj()])      # Eq. 1 with :26
    ref = orc.rows_times_block(np.vstack([top, bot]), X)
    Y = to_host(h.apply(to_dev(X)))
    assert relerr(np.vstack([Y[rows], Y[N + rows]]), ref) <= TOL_APPLY
    Xs = np.vstack([X[N:].conj(), X[:N].conj()])
    Ys = to_host(h.apply(to_dev(Xs)))
    assert relerr(Ys[N:], -Y[:N].conj()) <= TOL_APPLY and relerr(Ys[:N], -Y[N:].conj()) <= TOL_APPLY


def test_lanczos_quadrature_on_rounded_operator(orc):
    """bse_lanczos_quadrature over the complex64 store: the k = 1 kernel with widened fragments."""
    import torch
    import paper_2504_10096_b200 as b
    N, steps = 320, 60
    R = gen.dense_R(N, 3, sigma=0.0)
    R32 = orc.round_c64(R)
    d = gen.block_X(N, 1, 8)[:, 0]
    h = b.Bse(b.MODE_TDA, N, _pack64(R, 0), storage=b.STORE_C64)
    alpha, beta = h.lanczos_quadrature(torch.from_numpy(np.ascontiguousarray(d)).cuda(), steps)
    ao, bo = orc.lanczos_quadrature(R32, d, steps)
    assert np.max(np.abs(alpha - ao)) <= 1e-11 * 11 and np.max(np.abs(beta - bo)) <= 1e-11 * 11
    a_unrounded, _ = orc.lanczos_quadrature(R, d, steps)
    assert np.max(np.abs(alpha - a_unrounded)) > 1e-9            # it is the rounded operator that was applied
