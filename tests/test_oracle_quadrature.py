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
