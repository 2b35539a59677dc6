"""Pins for the oracle's eigen-routines: Jacobi, the paper's section-2.1 direct route, textbook Lanczos
(TDA and structure-preserving), block Gram-Schmidt.  Pinned to prescribed spectra, closed forms,
invariants of the pseudo-Hermitian spectrum and independent library routines."""
import numpy as np
import pytest

import bse_inputs as gen


def _H_dense(R, C):
    return np.block([[R, C], [-C.conj().T, -R.conj()]])


def test_jacobi_recovers_prescribed_spectrum(orc):
    # R = Q diag(lam) Q^H with a generic unitary Q (QR of a random matrix)
    n = 48
    lam = np.sort(np.linspace(-3.0, 7.0, n) + 0.01 * np.arange(n) ** 1.5)
    Q, _ = np.linalg.qr(gen.block_X(n, n, 3))
    A = (Q * lam) @ Q.conj().T
    A = (A + A.conj().T) / 2
    w, V = orc.jacobi_herm(A)
    assert np.max(np.abs(w - lam)) < 1e-13 * np.max(np.abs(lam))
    assert np.linalg.norm(V.conj().T @ V - np.eye(n)) < 1e-13
    assert np.linalg.norm(A @ V - V * w) < 1e-13 * np.linalg.norm(A)
    assert abs(np.sum(w) - np.trace(A).real) < 1e-12          # tr R = sum lambda


def test_jacobi_householder_closed_form(orc):
    n = 64
    lam = gen.prescribed_spectrum(n, 5, 1.0, 10.0)
    u = gen.householder_u(n, 5)
    R = gen.closed_form_tda_dense(lam, u)
    assert np.allclose(R, R.conj().T)
    w, _ = orc.jacobi_herm(R)
    assert np.max(np.abs(w - lam)) < 1e-13 * n   # ~ n eps |R|


def _bse_pair(N, seed, sigma=1.0):
    return gen.dense_R(N, seed, sigma=sigma), gen.dense_C(N, seed)


def test_direct_route_pairing_trace_and_library(orc):
    N = 48
    R, C = _bse_pair(N, 1)
    om, V = orc.bse_direct(R, C)
    # eigenvalues real, in (-w, +w) pairs
    assert np.allclose(om[:N][::-1], -om[N:], atol=1e-12)
    assert np.all(om[N:] > 0)
    assert abs(np.sum(om)) < 1e-11                                  # trace(H) = 0 = sum of all omega
    # sum omega^2 = |R|_F^2 - |C|_F^2 (tr H^2 = 2(|R|_F^2 - |C|_F^2))
    assert abs(np.sum(om[N:] ** 2) - (np.linalg.norm(R) ** 2 - np.linalg.norm(C) ** 2)) < 1e-10
    # independent library route
    ev = np.linalg.eigvals(_H_dense(R, C))
    assert np.max(np.abs(ev.imag)) < 1e-10
    assert np.max(np.abs(np.sort(ev.real) - om)) < 1e-11
    # right eigenvectors: residual, and the -w partner is [conj(Y); conj(X)]
    H = _H_dense(R, C)
    assert np.linalg.norm(H @ V - V * om) < 1e-11 * np.linalg.norm(H)
    v = V[:, N + 3]
    partner = np.concatenate([v[N:].conj(), v[:N].conj()])
    assert np.linalg.norm(H @ partner + om[N + 3] * partner) < 1e-11 * np.linalg.norm(H)


def test_direct_route_real_case_product_form(orc):
    # for real R and C: omega^2 = eig((R - C)(R + C))   (north_star pin)
    N = 48
    R, C = _bse_pair(N, 2)
    R = R.real.copy(); R = (R + R.T) / 2
    C = C.real.copy()
    om, _ = orc.bse_direct(R.astype(complex), C.astype(complex), want_vectors=False)
    ev = np.sort(np.linalg.eigvals((R - C) @ (R + C)).real)
    assert np.max(np.abs(np.sort(om[N:] ** 2) - ev)) < 1e-10


def test_direct_route_closed_form_pair(orc):
    # closed-form pair with omega_i = sqrt(d1_i d2_i) exactly
    N = 32
    d1 = gen.prescribed_spectrum(N, 7, 1.0, 9.0)
    d2 = gen.prescribed_spectrum(N, 8, 2.0, 5.0)
    u = gen.householder_u(N, 9, complex_u=False)
    R, C = gen.closed_form_full_dense(d1, d2, u, gen.phases(N, 9))
    assert np.allclose(R, R.conj().T) and np.allclose(C, C.T)
    om, _ = orc.bse_direct(R, C, want_vectors=False)
    assert np.max(np.abs(om[N:] - np.sort(np.sqrt(d1 * d2)))) < 1e-12


def test_direct_route_rejects_indefinite(orc):
    # literal generator (sigma = 0) at larger N is indefinite; here force it
    N = 16
    R, C = _bse_pair(N, 3)
    with pytest.raises(np.linalg.LinAlgError):
        orc.bse_direct(R - 20 * np.eye(N), C)


def test_lanczos_tda_vs_jacobi_and_residuals(orc):
    N, nev = 160, 6
    R = gen.dense_R(N, 4, sigma=0.0)
    v0 = gen.block_X(N, 1, 99)[:, 0]
    w, V, res, steps = orc.lanczos_tda(R, nev, 1e-10, v0, check=5)
    assert steps > 0
    wj, _ = orc.jacobi_herm(R)
    wl = np.linalg.eigvalsh(R)
    assert np.max(np.abs(wj - wl)) < 1e-12
    assert np.max(np.abs(w - wj[:nev])) < 1e-10 * np.max(np.abs(wj))
    nrmR = np.max(np.abs(wj))
    r = np.linalg.norm(R @ V - V * w, axis=0)
    assert np.all(r < 1e-8 * nrmR)
    assert np.linalg.norm(V.conj().T @ V - np.eye(nev)) < 1e-10


def test_lanczos_tda_prescribed_spectrum(orc):
    N, nev = 200, 5
    lam = gen.prescribed_spectrum(N, 11, 1.0, 10.0)
    R = gen.closed_form_tda_dense(lam, gen.householder_u(N, 11))
    v0 = gen.block_X(N, 1, 98)[:, 0]
    w, V, res, steps = orc.lanczos_tda(R, nev, 1e-10, v0, check=5)
    assert steps > 0
    assert np.max(np.abs(w - lam[:nev])) < 1e-10 * 10


def test_lanczos_full_vs_direct_route(orc):
    N, nev = 96, 5
    R, C = _bse_pair(N, 6)
    x0 = gen.block_X(N, 1, 97)[:, 0]
    om, V, res, steps = orc.lanczos_full(R, C, nev, 1e-10, x0, check=5)
    assert steps > 0
    omd, _ = orc.bse_direct(R, C, want_vectors=False)
    assert np.max(np.abs(om - omd[N:N + nev])) < 1e-10 * omd[-1]
    H = _H_dense(R, C)
    r = np.linalg.norm(H @ V - V * om, axis=0)
    assert np.all(r < 1e-8 * omd[-1])
    assert np.all(r < 5 * res + 1e-12)                      # the residual formula of reading S4
    # normalisation X^H X - Y^H Y = 1 (reading S9) and Sigma-orthogonality
    Sig = np.concatenate([np.ones(N), -np.ones(N)])
    G = V.conj().T @ (Sig[:, None] * V)
    assert np.linalg.norm(G - np.eye(nev)) < 1e-8


def test_lanczos_full_returns_distinct_omega_far_past_convergence(orc):
    # Reading R1: every omega^2 is a double eigenvalue of G = M o P on R^2N; the second copy grows out of rounding
    # noise once the first has converged.  Run 3 x past first convergence (copies present among the Ritz values)
    # and require the nev lowest DISTINCT omega of H -- a value-sorted list of Ritz values would return pairs.
    N, nev = 192, 12
    R, C = _bse_pair(N, 6)
    x0 = gen.block_X(N, 1, 97)[:, 0]
    om1, _, _, steps1 = orc.lanczos_full(R, C, nev, 1e-11, x0, check=4)
    assert 0 < steps1 < 2 * N - 4
    # ... and to (almost) the whole space R^2N, where EVERY omega^2 has both of its Ritz values: the 12 lowest Ritz
    # values are then 6 pairs
    minit = 2 * N - 4
    om, V, res, steps = orc.lanczos_full(R, C, nev, 1e-11, x0, check=4, minit=minit)
    assert steps >= minit
    omd, Vd = orc.bse_direct(R, C)
    assert np.max(np.abs(om - omd[N:N + nev])) < 1e-10 * omd[-1]
    assert np.max(np.abs(om1 - omd[N:N + nev])) < 1e-10 * omd[-1]
    assert np.min(np.diff(om)) > 1e-6                              # no value returned twice
    H = _H_dense(R, C)
    r = np.linalg.norm(H @ V - V * om, axis=0)
    assert np.all(r < 1e-8 * omd[-1])
    Sig = np.concatenate([np.ones(N), -np.ones(N)])
    assert np.linalg.norm(V.conj().T @ (Sig[:, None] * V) - np.eye(nev)) < 1e-8


def test_lanczos_full_copy_structure(orc):
    # the identities behind the multiplicity rule: K(x) = i P(x) satisfies K^2 = -G, and if P x = w y, M y = w x then
    # v(x) = [x + y; conj(x - y)] and v(K x / w) = i v(x)
    N = 48
    R, C = _bse_pair(N, 8)
    x = gen.block_X(N, 1, 5)
    P = lambda z: orc.apply_half(R, C, z, +1)
    M = lambda z: orc.apply_half(R, C, z, -1)
    K = lambda z: 1j * P(z)
    assert np.linalg.norm(K(K(x)) + M(P(x))) < 1e-12 * np.linalg.norm(M(P(x)))
    omd, Vd = orc.bse_direct(R, C)
    w, v = omd[N + 2], Vd[:, N + 2]
    xe, ye = (v[:N] + v[N:].conj()) / 2, (v[:N] - v[N:].conj()) / 2     # v = [x + y; conj(x - y)]
    xe, ye = xe[:, None], ye[:, None]
    assert np.linalg.norm(P(xe) - w * ye) < 1e-10 and np.linalg.norm(M(ye) - w * xe) < 1e-10
    x2 = K(xe) / w
    y2 = P(x2) / w
    v2 = np.concatenate([x2 + y2, (x2 - y2).conj()])[:, 0]
    assert np.linalg.norm(v2 - 1j * v) < 1e-10


def test_gruning_variant_vs_direct_route_and_shao_variant(orc):
    """The second structure-preserving variant (reading R9: Lanczos on H in the Omega inner product, T = tridiag(beta, 0, beta))
    against the paper's direct route, and against the first variant: 2 m of its vectors span what m steps of the H^2 recurrence
    span, so the Ritz values agree long before either has converged ("very similar in terms of operations")."""
    N, nev = 96, 5
    R, C = _bse_pair(N, 6)
    x0 = gen.block_X(N, 1, 97)[:, 0]
    om, V, res, steps = orc.lanczos_full_gruning(R, C, nev, 1e-10, x0, check=4)
    assert steps > 0
    omd, _ = orc.bse_direct(R, C, want_vectors=False)
    assert np.max(np.abs(om - omd[N:N + nev])) < 1e-10 * omd[-1]
    H = _H_dense(R, C)
    r = np.linalg.norm(H @ V - V * om, axis=0)
    assert np.all(r < 1e-8 * omd[-1]) and np.all(r < 5 * res + 1e-12)
    Sig = np.concatenate([np.ones(N), -np.ones(N)])
    assert np.linalg.norm(V.conj().T @ (Sig[:, None] * V) - np.eye(nev)) < 1e-8
    # one half apply per vector: exactly twice the step count of the H^2 recurrence for the same convergence
    om_s, _, _, steps_s = orc.lanczos_full(R, C, nev, 1e-10, x0, check=2)
    assert steps == 2 * steps_s
    # unconverged Ritz values after m = 30 steps (never-met tolerance, stop at maxit): same Krylov space, same values
    m = 30
    a, _, _, sa = orc.lanczos_full(R, C, 4, 1e-30, x0, maxit=m, check=m)
    b, _, _, sb = orc.lanczos_full_gruning(R, C, 4, 1e-30, x0, maxit=2 * m, check=2 * m)
    assert sa == -m and sb == -2 * m
    assert np.max(np.abs(a - b)) < 1e-9 * omd[-1] and np.max(np.abs(a - omd[N:N + 4])) > 1e-6    # equal, and not yet converged


def test_gruning_variant_returns_distinct_omega_on_the_whole_space(orc):
    N, nev = 96, 10
    R, C = _bse_pair(N, 9)
    x0 = gen.block_X(N, 1, 95)[:, 0]
    om, V, res, steps = orc.lanczos_full_gruning(R, C, nev, 1e-11, x0, check=4, minit=4 * N - 8)
    assert steps >= 4 * N - 8
    omd, _ = orc.bse_direct(R, C, want_vectors=False)
    assert np.max(np.abs(om - omd[N:N + nev])) < 1e-10 * omd[-1] and np.min(np.diff(om)) > 1e-6


def test_tridiag_ql_closed_form_and_jacobi(orc):
    # Toeplitz tridiag(b, a, b): eigenvalues a + 2 b cos(j pi / (m + 1)), eigenvectors sin(i j pi / (m + 1))
    m, a, b = 60, 1.5, -0.7
    w, Z = orc.tridiag_ql(np.full(m, a), np.full(m - 1, b))
    j = np.arange(1, m + 1)
    lam = a + 2 * b * np.cos(j * np.pi / (m + 1))
    order = np.argsort(lam)
    assert np.max(np.abs(w - lam[order])) < 1e-13
    U = np.sin(np.outer(j, j) * np.pi / (m + 1)) * np.sqrt(2.0 / (m + 1))
    assert np.max(np.abs(np.abs(np.sum(Z * U[:, order], axis=0)) - 1)) < 1e-12
    # random tridiagonal vs the (separately pinned) Jacobi routine, and the decomposition identities
    rng = np.random.default_rng(5)
    d, e = rng.standard_normal(40), rng.standard_normal(39)
    e[17] = 0.0                                                      # a reducible matrix splits cleanly
    T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
    w, Z = orc.tridiag_ql(d, e)
    wj, _ = orc.jacobi_herm(T.astype(complex))
    assert np.max(np.abs(w - wj)) < 1e-13 * np.max(np.abs(wj))
    assert np.linalg.norm(Z.T @ T @ Z - np.diag(w)) < 1e-13 * m and np.linalg.norm(Z.T @ Z - np.eye(40)) < 1e-13
    w1, _ = orc.tridiag_ql(np.array([3.0]), np.array([]))
    assert w1[0] == 3.0


def test_block_cgs2_factorisation(orc):
    N, m, k = 300, 12, 4
    V, _ = np.linalg.qr(gen.block_X(N, m, 1))
    W = gen.block_X(N, k, 2)
    # make W nearly dependent on V (kappa ~ 1e10): a single pass would lose orthogonality
    W = V @ gen.block_X(m, k, 3) + 1e-10 * W
    Q, h, B, rank = orc.block_cgs2(V, W)
    assert rank == k
    assert np.linalg.norm(V.conj().T @ Q) < 1e-13
    assert np.linalg.norm(Q.conj().T @ Q - np.eye(k)) < 1e-13
    assert np.linalg.norm(W - V @ h - Q @ B) / np.linalg.norm(W) < 1e-14
    assert np.allclose(B, np.triu(B)) and np.all(np.diag(B).real > 0) and np.allclose(np.diag(B).imag, 0)
    # library cross-check: Q B is the QR factorisation of (I - V V^H) W with positive diagonal
    Z = W - V @ (V.conj().T @ W); Z = Z - V @ (V.conj().T @ Z)
    Qn, Rn = np.linalg.qr(Z)
    ph = np.diag(Rn) / np.abs(np.diag(Rn))
    assert np.linalg.norm(Q - Qn * ph) < 1e-4     # kappa-limited agreement of the unique factor


def test_block_cgs2_rank_deficient(orc):
    N, m, k = 100, 5, 3
    V, _ = np.linalg.qr(gen.block_X(N, m, 4))
    W = gen.block_X(N, k, 5)
    W[:, 2] = W[:, 0] * (1 + 2j) + V[:, 1]
    Q, h, B, rank = orc.block_cgs2(V, W)
    assert rank == 2
    assert np.linalg.norm(W - V @ h - Q @ B) / np.linalg.norm(W) < 1e-13


def test_generator_statistics_and_structure():
    N = 512
    R = gen.dense_R(N, 1, sigma=0.0); C = gen.dense_C(N, 1)
    assert np.array_equal(R, R.conj().T) and np.array_equal(C, C.T)
    assert np.all(R.diagonal().imag == 0)
    d = gen.transition_energies(N, 1, 16)
    assert d.min() >= 1 and d.max() <= 10 and np.all(np.diff(d.reshape(-1, 16), axis=1) >= 0)
    i, j = np.tril_indices(N, -1)
    K = R[i, j] * (1 + np.abs(i - j) / 64.0) / 0.1
    assert abs(K.real.mean()) < 0.02 and abs(K.real.std() - 1) < 0.02 and abs(K.imag.std() - 1) < 0.02
    Cn = C[i, j] * (1 + np.abs(i - j) / 64.0) / 0.05
    assert abs(Cn.real.std() - 1) < 0.02
    # rows_R agrees with dense_R (same counter-based entries regardless of chunking)
    assert np.array_equal(gen.rows_R(N, 1, [5, 300]), R[[5, 300]])
