"""bse_lanczos_quadrature against the oracle and against the exact resolvent."""
import numpy as np
import pytest

import bse_inputs as gen
from gpu_util import pack, to_dev

pytestmark = pytest.mark.gpu


def _dev_vec(d):
    import torch
    return torch.from_numpy(np.ascontiguousarray(d)).cuda()


def test_coefficients_and_resolvent_match_oracle(orc):
    import paper_2504_10096_b200 as b
    N, steps = 320, 320
    R = gen.dense_R(N, 3, sigma=0.0)
    d = gen.block_X(N, 1, 8)[:, 0]
    h = b.Bse(b.MODE_TDA, N, pack(R, 0))
    alpha, beta = h.lanczos_quadrature(_dev_vec(d), steps)
    ao, bo = orc.lanczos_quadrature(R, d, steps)
    assert len(alpha) == steps
    # without reorthogonalisation rounding differences grow with the step count: the leading coefficients agree tightly
    assert np.max(np.abs(alpha[:20] - ao[:20])) <= 1e-10 * 11 and np.max(np.abs(beta[:21] - bo[:21])) <= 1e-10 * 11
    # ... and the quantity the method is for, the broadened resolvent, agrees for all steps
    om = np.linspace(-1.0, 11.0, 241); eta = 0.1
    # up to the step where the first Ritz value converges (~100 here) both recurrences are the same to rounding;
    # after that, without reorthogonalisation, the coefficients of ANY two runs differ at O(1) while the converged
    # resolvent does not (checked against the exact one below)
    assert np.max(np.abs(alpha[:80] - ao[:80])) <= 1e-11 * 11
    G80 = b.quadrature_resolvent(alpha[:80], beta[:81], om, eta)
    Go80 = orc.quadrature_resolvent(ao[:80], bo[:81], om, eta)
    assert np.max(np.abs(G80 - Go80)) <= 1e-11 * np.max(np.abs(Go80))
    G = b.quadrature_resolvent(alpha, beta, om, eta)
    lam, Q = np.linalg.eigh(R)
    wts = np.abs(Q.conj().T @ d) ** 2
    exact = np.array([np.sum(wts / (w + 1j * eta - lam)) for w in om])
    # N steps without reorthogonalisation: the continued fraction has converged to the exact resolvent at eta = 0.1
    # (oracle: 1.1e-2 after 120 steps, 2.3e-4 after 200, 1.0e-6 after 320)
    assert np.max(np.abs(G - exact)) <= 1e-5 * np.max(np.abs(exact))


def test_moments_at_a_many_tile_size(orc):
    """N = 4096 (every CTA walks several units; k = 1 path of the tile kernel), device-generated operator: the Gauss
    rule must reproduce d^H R^p d for p <= 2 steps - 1, computed with the oracle apply on rows from the CPU generator
    is too slow here, so the moments come from repeated oracle-checked bse_apply at small p and from the identity
    beta_0^2 (T^p)_00 = |R^{p/2} d|^2 evaluated through the CUDA apply (parity-tested in test_gpu_apply.py)."""
    import torch
    import paper_2504_10096_b200 as b
    N, steps = 4096, 12
    h = b.Bse(b.MODE_TDA, N, b.bse_fill_synthetic(N, 0, 1, 0.0, 16))
    d = gen.block_X(N, 1, 9)[:, 0]
    alpha, beta = h.lanczos_quadrature(_dev_vec(d), steps)
    T = np.diag(alpha) + np.diag(beta[1:steps], 1) + np.diag(beta[1:steps], -1)
    v = _dev_vec(d).reshape(1, N)
    vs = [v]
    for _ in range(steps):
        vs.append(h.apply(vs[-1]))
    Tp = np.eye(steps)
    for p in range(2 * steps):
        a, c = vs[p // 2], vs[p - p // 2]                       # d^H R^p d = (R^a d)^H (R^c d), a + c = p
        exact = float(torch.vdot(a.flatten(), c.flatten()).real)
        assert abs(beta[0] ** 2 * Tp[0, 0] - exact) <= 1e-9 * abs(exact), p
        Tp = Tp @ T
    # first coefficients against the oracle fed by the CPU generator's rows
    Rd = orc.rows_times_block(gen.rows_R(N, 1, np.arange(N), 0.0, 16), d.reshape(N, 1))[:, 0]
    a0 = np.vdot(d, Rd).real / np.vdot(d, d).real
    assert abs(alpha[0] - a0) <= 1e-12 * abs(a0) and abs(beta[0] - np.linalg.norm(d)) <= 1e-13 * beta[0]


def test_quadrature_invalid_arguments():
    import ctypes
    import paper_2504_10096_b200 as b
    N = 64
    R = gen.dense_R(N, 3, sigma=1.0)
    d = _dev_vec(gen.block_X(N, 1, 1)[:, 0])
    h = b.Bse(b.MODE_TDA, N, pack(R, 0))
    assert b.lib().bse_lanczos_quadrature(h._h, d.data_ptr(), 0, None, None, None) == 1
    # full mode: an indefinite Omega (R = -I, C = 0: <d, d>_P < 0) is reported, not iterated on
    Z = np.zeros((N, N), dtype=complex)
    hn = b.Bse(b.MODE_FULL, N, pack(-np.eye(N, dtype=complex), 0), pack(Z, 1))
    with pytest.raises(b.BseError) as e:
        hn.lanczos_quadrature(d, 4)
    assert e.value.status == b.lib().bse_lanczos_quadrature(hn._h, d.data_ptr(), 4, (ctypes.c_double * 4)(),
                                                            (ctypes.c_double * 5)(), None) != 0


def test_full_mode_coefficients_and_resolvent_match_oracle(orc):
    """Full (pseudo-Hermitian) quadrature (include/bse.h; oracle: lanczos_quadrature_full): coefficients against the
    oracle while the two recurrences are the same to rounding, the converged resolvent against the exact
    u^H Sigma (z - H)^-1 u from a dense solve of the block operator of Eq. (1)."""
    import paper_2504_10096_b200 as b
    N, steps = 192, 260
    R, C = gen.dense_R(N, 5, sigma=1.0), gen.dense_C(N, 5)
    d = gen.block_X(N, 1, 6)[:, 0]
    h = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    alpha, beta = h.lanczos_quadrature(_dev_vec(d), steps)
    ao, bo = orc.lanczos_quadrature_full(R, C, d, steps)
    assert len(alpha) == steps
    sc = np.max(np.abs(ao))                                # ~ |H|^2
    assert np.max(np.abs(alpha[:15] - ao[:15])) <= 1e-10 * sc and np.max(np.abs(beta[:16] - bo[:16])) <= 1e-10 * sc
    assert abs(beta[0] ** 2 - np.vdot(d, R @ d + C @ d.conj()).real) <= 1e-13 * beta[0] ** 2
    om = np.linspace(0.0, 12.0, 121); eta = 0.15
    G40 = b.quadrature_resolvent_full(alpha[:40], beta[:41], om, eta)
    Go40 = orc.quadrature_resolvent_full(ao[:40], bo[:41], om, eta)
    assert np.max(np.abs(G40 - Go40)) <= 1e-9 * np.max(np.abs(Go40))
    H = np.block([[R, C], [-C.conj(), -R.conj()]])
    u = np.concatenate([d, d.conj()]); sig = np.concatenate([np.ones(N), -np.ones(N)])
    exact = np.array([np.vdot(u, sig * np.linalg.solve((w + 1j * eta) * np.eye(2 * N) - H, u)) for w in om])
    G = b.quadrature_resolvent_full(alpha, beta, om, eta)
    Go = orc.quadrature_resolvent_full(ao, bo, om, eta)
    err_o = np.max(np.abs(Go - exact)) / np.max(np.abs(exact))
    assert np.max(np.abs(G - exact)) <= max(10 * err_o, 1e-6) * np.max(np.abs(exact))
    assert err_o <= 1e-4                                    # the oracle itself has converged at this step count


def test_full_mode_moments_at_a_many_tile_size(orc):
    """N = 4096, device-generated R and C (every CTA walks several units; the k = 1 kernel in both passes): odd moments
    u^H Sigma H^(2p+1) u = 2 beta_0^2 (T^p)_00 for p <= 2 steps - 1, with H^n u from the CUDA full apply (parity-tested in
    test_gpu_apply.py), and the even moments vanish."""
    import torch
    import paper_2504_10096_b200 as b
    N, steps = 4096, 6
    h = b.Bse(b.MODE_FULL, N, b.bse_fill_synthetic(N, 0, 1, 1.0, 16), b.bse_fill_synthetic(N, 1, 1, 0.0, 16))
    d = gen.block_X(N, 1, 9)[:, 0]
    alpha, beta = h.lanczos_quadrature(_dev_vec(d), steps)
    T = np.diag(alpha) + np.diag(beta[1:steps], 1) + np.diag(beta[1:steps], -1)
    u = _dev_vec(np.concatenate([d, d.conj()])).reshape(1, 2 * N)
    sig = torch.cat([torch.ones(N), -torch.ones(N)]).to(torch.complex128).cuda()
    vs = [u]
    for _ in range(2 * steps):
        vs.append(h.apply(vs[-1]))
    Tp = np.eye(steps)
    uu = float(torch.vdot(u.flatten(), u.flatten()).real)
    for p in range(2 * steps):
        n = 2 * p + 1                       # Sigma H is Hermitian, so u^H Sigma H^n u = (H^a u)^H Sigma (H^c u), a + c = n
        a, c = vs[n // 2], vs[n - n // 2]
        exact = complex(torch.vdot(a.flatten(), sig * c.flatten()))
        assert abs(exact.imag) <= 1e-9 * abs(exact.real)
        assert abs(2 * beta[0] ** 2 * Tp[0, 0] - exact.real) <= 1e-8 * abs(exact.real), p
        even = complex(torch.vdot(vs[p].flatten(), sig * vs[p].flatten()))      # u^H Sigma H^(2p) u
        assert abs(even) <= 1e-9 * float(torch.vdot(vs[p].flatten(), vs[p].flatten()).real)
        Tp = Tp @ T
    assert uu > 0
