"""Pins for the oracle's Lanczos-with-quadrature routine (the spectrum-without-eigenpairs solver)."""
import numpy as np

import bse_inputs as gen


def _herm(n, seed):
    A = gen.block_X(n, n, seed)
    A = (A + A.conj().T) / 2
    A[np.diag_indices(n)] = A.diagonal().real
    return A


def test_gauss_quadrature_reproduces_moments(orc):
    # m Lanczos steps define a Gauss rule: d^H R^p d = beta_0^2 (T^p)_00 for p <= 2m - 1
    N, m = 60, 6
    R = _herm(N, 3) / 4
    d = gen.block_X(N, 1, 4)[:, 0]
    alpha, beta = orc.lanczos_quadrature(R, d, m)
    T = np.diag(alpha) + np.diag(beta[1:m], 1) + np.diag(beta[1:m], -1)
    v = d.copy(); Tp = np.eye(m)
    for p in range(2 * m):
        exact = np.vdot(d, v).real
        assert abs(beta[0] ** 2 * Tp[0, 0] - exact) <= 1e-10 * max(abs(exact), 1.0), p
        v = R @ v; Tp = Tp @ T
    assert abs(beta[0] - np.linalg.norm(d)) < 1e-14
    # one more power is NOT reproduced (the rule is exactly of degree 2m - 1): guards against an off-by-one
    assert abs(beta[0] ** 2 * Tp[0, 0] - np.vdot(d, v).real) > 1e-8


def test_resolvent_matches_exact_eigendecomposition(orc):
    # run to completion on a small matrix: the continued fraction is the exact resolvent sum_i |q_i^H d|^2 / (z - lam_i)
    N = 24
    lam = np.linspace(1.0, 4.0, N) + 0.05 * np.sin(np.arange(N))
    Q, _ = np.linalg.qr(gen.block_X(N, N, 5))
    R = (Q * lam) @ Q.conj().T; R = (R + R.conj().T) / 2
    d = gen.block_X(N, 1, 6)[:, 0]
    alpha, beta = orc.lanczos_quadrature(R, d, N)
    om = np.linspace(0.5, 4.5, 81); eta = 0.05
    G = orc.quadrature_resolvent(alpha, beta, om, eta)
    wts = np.abs(Q.conj().T @ d) ** 2
    exact = np.array([np.sum(wts / (w + 1j * eta - lam)) for w in om])
    assert np.max(np.abs(G - exact)) <= 1e-8 * np.max(np.abs(exact))
    # sum rule: -1/pi * integral Im G = |d|^2 (Lorentzians integrate to their weights)
    om2 = np.linspace(-60, 65, 500001)
    G2 = orc.quadrature_resolvent(alpha, beta, om2, eta)
    assert abs(-np.trapezoid(G2.imag, om2) / np.pi - np.vdot(d, d).real) < 2e-3 * np.vdot(d, d).real


def test_diagonal_operator_closed_form(orc):
    # R = diag(lam): alpha_0 = sum lam |d|^2 / |d|^2, beta_1^2 = variance of lam under the weights |d_i|^2
    N = 30
    lam = np.linspace(-1, 2, N)
    d = gen.block_X(N, 1, 7)[:, 0]
    alpha, beta = orc.lanczos_quadrature(np.diag(lam).astype(complex), d, 2)
    w = np.abs(d) ** 2 / np.sum(np.abs(d) ** 2)
    mean = np.sum(w * lam)
    assert abs(alpha[0] - mean) < 1e-14 and abs(beta[1] ** 2 - np.sum(w * (lam - mean) ** 2)) < 1e-14


# ---- full (pseudo-Hermitian) case: PAPER.md:65 on the operator of Eq. 1, reading R7 ----

def _full_pair(N, seed):
    return gen.dense_R(N, seed, sigma=1.0), gen.dense_C(N, seed)


def _block_H(R, C):
    # Eq. (1) with A = R^*, C = C^T, assembled by numpy from the definition (not through the oracle)
    return np.block([[R, C], [-C.conj(), -R.conj()]])


def test_full_quadrature_reproduces_odd_moments_and_even_vanish(orc):
    # u^H Sigma H^(2p+1) u = 2 beta_0^2 (T^p)_00 for p <= 2m - 1;  u^H Sigma H^(2p) u = 0;  u = [d; conj d]
    N, m = 48, 5
    R, C = _full_pair(N, 3)
    R, C = R / 8, C / 8
    d = gen.block_X(N, 1, 4)[:, 0]
    alpha, beta = orc.lanczos_quadrature_full(R, C, d, m)
    T = np.diag(alpha) + np.diag(beta[1:m], 1) + np.diag(beta[1:m], -1)
    u = np.concatenate([d, d.conj()])
    sig = np.concatenate([np.ones(N), -np.ones(N)])
    v = u.copy(); Tp = np.eye(m)
    for n in range(4 * m + 2):
        mom = np.vdot(u, sig * v)
        if n % 2 == 0:
            assert abs(mom) <= 1e-10 * np.vdot(u, u).real, n
        else:
            p = (n - 1) // 2
            quad = 2 * beta[0] ** 2 * Tp[0, 0]
            if p <= 2 * m - 1:
                assert abs(mom.imag) <= 1e-10 * abs(mom.real)
                assert abs(quad - mom.real) <= 1e-9 * abs(mom.real), p
            else:
                assert abs(quad - mom.real) > 1e-7 * abs(mom.real)      # degree exactly 2m - 1
            Tp = Tp @ T
        v = orc.apply_full(R, C, v.reshape(-1, 1))[:, 0]
    assert abs(beta[0] ** 2 - np.vdot(d, R @ d + C @ d.conj()).real) < 1e-13 * beta[0] ** 2


def test_full_resolvent_matches_dense_solve(orc):
    # run to completion at a tiny size: the continued fraction in z^2 is the exact u^H Sigma (z - H)^{-1} u
    N = 16
    R, C = _full_pair(N, 5)
    d = gen.block_X(N, 1, 6)[:, 0]
    alpha, beta = orc.lanczos_quadrature_full(R, C, d, N)
    H = _block_H(R, C)
    u = np.concatenate([d, d.conj()])
    sig = np.concatenate([np.ones(N), -np.ones(N)])
    om = np.linspace(-12.0, 12.0, 97); eta = 0.1
    exact = np.array([np.vdot(u, sig * np.linalg.solve((w + 1j * eta) * np.eye(2 * N) - H, u)) for w in om])
    G = orc.quadrature_resolvent_full(alpha, beta, om, eta)
    assert np.max(np.abs(G - exact)) <= 1e-7 * np.max(np.abs(exact))
    # the other start vector of the structure: [y; -conj y] = -i [iy; conj(iy)]  ->  same function with d = i y
    y = gen.block_X(N, 1, 7)[:, 0]
    um = np.concatenate([y, -y.conj()])
    exact_m = np.array([np.vdot(um, sig * np.linalg.solve((w + 1j * eta) * np.eye(2 * N) - H, um)) for w in om])
    a2, b2 = orc.lanczos_quadrature_full(R, C, 1j * y, N)
    assert np.max(np.abs(orc.quadrature_resolvent_full(a2, b2, om, eta) - exact_m)) <= 1e-7 * np.max(np.abs(exact_m))


def test_full_resolvent_against_direct_route_spectrum(orc):
    # spectral form with the paper's direct route (section 2.1): f(z) = sum_I s_I |v_I^H Sigma u|^2 / (z - w_I),
    # s_I = sign(w_I) = v_I^H Sigma v_I for Sigma-normalised right eigenvectors
    N = 16
    R, C = _full_pair(N, 8)
    d = gen.block_X(N, 1, 9)[:, 0]
    w, V = orc.bse_direct(R, C)
    u = np.concatenate([d, d.conj()])
    sig = np.concatenate([np.ones(N), -np.ones(N)])
    nrm = np.einsum("ij,i,ij->j", V.conj(), sig, V).real
    wt = np.abs(V.conj().T @ (sig * u)) ** 2 / np.abs(nrm)
    alpha, beta = orc.lanczos_quadrature_full(R, C, d, N)
    om = np.linspace(0.2, 11.0, 60); eta = 0.08
    exact = np.array([np.sum(np.sign(nrm) * wt / (x + 1j * eta - w)) for x in om])
    G = orc.quadrature_resolvent_full(alpha, beta, om, eta)
    assert np.max(np.abs(G - exact)) <= 1e-7 * np.max(np.abs(exact))


def test_full_quadrature_with_zero_coupling_is_tda_at_plus_and_minus_z(orc):
    # C = 0: H = diag(R, -conj R), so f(z) = g(z) + g(-z) with g the TDA resolvent d^H (z - R)^{-1} d
    N = 20
    lam = np.linspace(1.0, 3.0, N) + 0.03 * np.cos(np.arange(N))
    Q, _ = np.linalg.qr(gen.block_X(N, N, 10))
    R = (Q * lam) @ Q.conj().T; R = (R + R.conj().T) / 2
    d = gen.block_X(N, 1, 11)[:, 0]
    alpha, beta = orc.lanczos_quadrature_full(R, np.zeros((N, N), dtype=complex), d, N)
    at, bt = orc.lanczos_quadrature(R, d, N)
    om = np.linspace(0.5, 3.5, 41); eta = 0.05
    g_plus = orc.quadrature_resolvent(at, bt, om, eta)
    g_minus = np.conj(orc.quadrature_resolvent(at, bt, -om, eta))       # g(conj z) = conj g(z)
    G = orc.quadrature_resolvent_full(alpha, beta, om, eta)
    assert np.max(np.abs(G - (g_plus + g_minus))) <= 1e-8 * np.max(np.abs(G))
    # first coefficients in closed form: beta_0^2 = d^H R d, alpha_0 = d^H R^3 d / d^H R d
    wts = np.abs(Q.conj().T @ d) ** 2
    assert abs(beta[0] ** 2 - np.sum(wts * lam)) < 1e-12 * beta[0] ** 2
    assert abs(alpha[0] - np.sum(wts * lam ** 3) / np.sum(wts * lam)) < 1e-12 * alpha[0]


def test_full_quadrature_rejects_indefinite_omega(orc):
    N = 8
    with np.testing.assert_raises(np.linalg.LinAlgError):
        orc.lanczos_quadrature_full(-np.eye(N, dtype=complex), np.zeros((N, N), dtype=complex), np.ones(N, dtype=complex), 3)
