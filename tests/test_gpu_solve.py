"""bse_solve against the oracle (north_star tolerances): eigenvalues rel. error <= 1e-10, residuals <= 1e-8 ||H||,
orthonormality <= 1e-12; closed-form prescribed spectra pin the eigenvalues independently of any solver."""
import numpy as np
import pytest

import bse_inputs as gen
from gpu_util import pack, to_dev, to_host

pytestmark = pytest.mark.gpu
TOL_EIG, TOL_RES, TOL_ORTH = 1e-10, 1e-8, 1e-12
# Reading R8: the eigenvalue error of a Ritz pair is ~ residual^2 / gap.  At the literal sigma = 0
# configs the wanted eigenvalues are ~1e-2 with gaps ~1e-2 and ||R|| ~ 11, so "1e-10 relative" asks for 1e-12 absolute
# and residuals of 1e-8 ||R|| (eigenvalue error ~1e-12) leave no margin: configs 0 and 1, whose tolerance BASELINE.json
# does not state, are solved with tol = 1e-10.  Configs 2 and 4 state tol 1e-8 and are certified through their residuals.
TOL_SMALL = 1e-10


def _check_tda(orc, R, res, nev, w_ref):
    """north_star: eigenvalues to 1e-10 RELATIVE (no absolute escape: DESIGN.md section 2, reading R8 says which tol the
    small-eigenvalue configs are solved with), residuals through the oracle apply, orthonormality of the vectors and of
    the final Krylov basis."""
    w, V = res.omega, to_host(res.vectors)
    nrm = np.max(np.abs(np.linalg.eigvalsh(R)[[0, -1]]))
    assert np.max(np.abs(w - w_ref[:nev]) / np.abs(w_ref[:nev])) <= TOL_EIG
    r = np.linalg.norm(orc.apply_tda(R, V) - V * w, axis=0)
    assert np.all(r <= TOL_RES * nrm)
    assert np.all(r <= 10 * res.resid + 1e-11 * nrm)            # the solver's own estimate is honest
    assert np.linalg.norm(V.conj().T @ V - np.eye(nev)) <= TOL_ORTH
    assert res.info["basis_orth_err"] <= TOL_ORTH                # ||V^H V - I||_F of the whole final basis


@pytest.mark.parametrize("sigma", [0.0, 1.0])
def test_config0_tda_vs_oracle_lanczos(orc, sigma):
    import paper_2504_10096_b200 as b
    cfg = gen.CONFIGS[0]
    N, nev, k = cfg["N"], cfg["nev"], cfg["k"]
    R = gen.dense_R(N, 1, sigma=sigma, group=cfg["group"])
    res = b.Bse(b.MODE_TDA, N, pack(R, 0)).solve(nev, k, tol=TOL_SMALL, seed=1)
    w_o, V_o, r_o, steps = orc.lanczos_tda(R, nev, 1e-10, gen.block_X(N, 1, 99)[:, 0], check=20)
    assert steps > 0
    # eigenvalues are unique: single-vector oracle and block GPU solver must agree
    _check_tda(orc, R, res, nev, w_o)
    assert np.max(np.abs(w_o - np.linalg.eigvalsh(R)[:nev])) < 1e-11
    # eigenvectors agree up to a phase for isolated eigenvalues
    ov = np.abs(np.sum(V_o.conj() * to_host(res.vectors), axis=0))
    assert np.all(ov > 1 - 1e-6)


@pytest.mark.parametrize("k", [1, 3, 8])
def test_tda_block_sizes_and_ragged_N(orc, k):
    import paper_2504_10096_b200 as b
    N, nev = 300, 6
    A = gen.block_X(N, N, 5); R = (A + A.conj().T) / 2 + np.diag(np.linspace(0, 30, N))
    res = b.Bse(b.MODE_TDA, N, pack(R, 0)).solve(nev, k, tol=1e-9, seed=3)
    _check_tda(orc, R, res, nev, np.linalg.eigvalsh(R))


def test_tda_closed_form_spectrum():
    import torch
    import paper_2504_10096_b200 as b
    N, nev, k = 4096, 12, 4
    lam = gen.prescribed_spectrum(N, 11, 1.0, 10.0, power=2 / 3)
    u = gen.householder_u(N, 11)
    t = b.bse_fill_closed_form_tda(N, torch.from_numpy(lam).cuda(), torch.from_numpy(u).cuda(),
                                   float(np.sum(lam * np.abs(u) ** 2)))
    res = b.Bse(b.MODE_TDA, N, t).solve(nev, k, tol=1e-9, seed=2)
    assert np.max(np.abs(res.omega - lam[:nev]) / lam[:nev]) <= TOL_EIG


def _H_dense(R, C):
    return np.block([[R, C], [-C.conj().T, -R.conj()]])


def _check_full(orc, R, C, res, nev, om_ref):
    N = R.shape[0]
    om, V = res.omega, to_host(res.vectors)
    assert len(om_ref) >= nev
    assert np.max(np.abs(om - om_ref[:nev]) / om_ref[:nev]) <= TOL_EIG
    HV = orc.apply_full(R, C, V)
    nrm = np.linalg.norm(_H_dense(R, C), 2) if N <= 600 else 12.0
    r = np.linalg.norm(HV - V * om, axis=0) / np.linalg.norm(V, axis=0)
    assert np.all(r <= TOL_RES * nrm)
    Sig = np.concatenate([np.ones(N), -np.ones(N)])
    G = V.conj().T @ (Sig[:, None] * V)
    # Reading S10: the 1e-12 figure is for the basis, orthonormal in <x, z>_P = Re(x^H P(z)); eigenvectors of distinct
    # omega are Sigma-orthogonal only to their own accuracy (residual / gap), their normalisation X^H X - Y^H Y = 1 is exact
    assert res.info["basis_orth_err"] <= TOL_ORTH
    assert np.linalg.norm(G - np.eye(nev)) <= 1e-7
    assert np.max(np.abs(np.diag(G) - 1)) <= 1e-10
    # -omega partner [conj(Y); conj(X)]
    Pn = np.vstack([V[N:].conj(), V[:N].conj()])
    rp = np.linalg.norm(orc.apply_full(R, C, Pn) + Pn * om, axis=0) / np.linalg.norm(Pn, axis=0)
    assert np.all(rp <= TOL_RES * nrm)


@pytest.mark.parametrize("k", [1, 4])
def test_full_small_vs_direct_route(orc, k):
    import paper_2504_10096_b200 as b
    N, nev = 192, 8
    R = gen.dense_R(N, 2, sigma=1.0); C = gen.dense_C(N, 2)
    res = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1)).solve(nev, k, tol=1e-9, seed=1)
    omd, _ = orc.bse_direct(R, C, want_vectors=False)           # the paper's section-2.1 route
    _check_full(orc, R, C, res, nev, omd[N:])


@pytest.mark.parametrize("k", [1, 4])
def test_gruning_variant_small_vs_direct_route(orc, k):
    """bse_solve_variant(BSE_VARIANT_GRUNING) (reading R9) against the paper's direct route, with the same
    checks as the default variant; both variants return the same omega."""
    import paper_2504_10096_b200 as b
    N, nev = 192, 8
    R = gen.dense_R(N, 2, sigma=1.0); C = gen.dense_C(N, 2)
    h = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    res = h.solve(nev, k, tol=1e-9, seed=1, variant=b.VARIANT_GRUNING)
    omd, _ = orc.bse_direct(R, C, want_vectors=False)
    _check_full(orc, R, C, res, nev, omd[N:])
    ref = h.solve(nev, k, tol=1e-9, seed=1)
    assert np.max(np.abs(res.omega - ref.omega) / ref.omega) <= TOL_EIG


def test_gruning_variant_config1_golden_and_oracle_variant(orc):
    """BASELINE.json config 1 with the second variant: the stored oracle values (20 distinct omega), live residuals through
    the oracle apply; and the oracle's own Gruning recurrence on a smaller instance of the same generator."""
    import paper_2504_10096_b200 as b
    cfg = gen.CONFIGS[1]
    N, nev, k = cfg["N"], cfg["nev"], cfg["k"]
    R = gen.dense_R(N, 1, sigma=cfg["sigma"]); C = gen.dense_C(N, 1)
    res = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1)).solve(nev, k, tol=TOL_SMALL, seed=1, variant=b.VARIANT_GRUNING)
    _check_full(orc, R, C, res, nev, _golden("oracle_config1.txt"))
    n = 256
    Rs = gen.dense_R(n, 4, sigma=1.0); Cs = gen.dense_C(n, 4)
    om_o, _, _, steps = orc.lanczos_full_gruning(Rs, Cs, 6, 1e-11, gen.block_X(n, 1, 96)[:, 0], check=4)
    assert steps > 0
    rs = b.Bse(b.MODE_FULL, n, pack(Rs, 0), pack(Cs, 1)).solve(6, 2, tol=1e-10, seed=2, variant=b.VARIANT_GRUNING)
    assert np.max(np.abs(rs.omega - om_o) / om_o) <= TOL_EIG


def test_gruning_variant_closed_form_degenerate_and_real_form():
    """Closed-form pair with a double omega (multiplicity decided from the vectors in both variants), complex stores and the
    real-form store."""
    import torch
    import paper_2504_10096_b200 as b
    N, nev, k = 2048, 10, 4
    d1 = gen.prescribed_spectrum(N, 7, 1.0, 9.0, power=2 / 3); d2 = gen.prescribed_spectrum(N, 8, 2.0, 5.0, power=2 / 3)
    d1[1], d2[1] = d1[0] * 1.2, d2[0] / 1.2
    ur = gen.householder_u(N, 9, complex_u=False).real.copy(); phi = gen.phases(N, 9)
    rt, ct = b.bse_fill_closed_form_full(N, *(torch.from_numpy(a).cuda() for a in (d1, d2, ur, phi)),
                                         float(np.sum(d1 * ur ** 2)), float(np.sum(d2 * ur ** 2)))
    exact = np.sort(np.sqrt(d1 * d2))[:nev]
    res = b.Bse(b.MODE_FULL, N, rt, ct).solve(nev, k, tol=1e-9, seed=4, variant=b.VARIANT_GRUNING)
    assert np.max(np.abs(res.omega - exact) / exact) <= TOL_EIG and res.info["basis_orth_err"] <= TOL_ORTH
    b.bse_to_real_form(rt, ct, N)
    res = b.Bse(b.MODE_FULL, N, rt, ct, storage=b.STORE_REAL_FORM).solve(nev, 8, tol=1e-9, seed=4, variant=b.VARIANT_GRUNING)
    assert np.max(np.abs(res.omega - exact) / exact) <= TOL_EIG


def test_partner_and_left_eigenvectors(orc):
    """eigenvectors of the negative eigenvalues and left eigenvectors "can be obtained trivially"."""
    import paper_2504_10096_b200 as b
    N, nev = 192, 6
    R = gen.dense_R(N, 2, sigma=1.0); C = gen.dense_C(N, 2)
    h = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    res = h.solve(nev, 4, tol=1e-10, seed=1)
    V, om = to_host(res.vectors), res.omega
    H = _H_dense(R, C)
    nrm = np.linalg.norm(H, 2)
    Vn = to_host(h.partner_vectors(res.vectors, 0))
    assert np.all(np.linalg.norm(orc.apply_full(R, C, Vn) + Vn * om, axis=0) <= TOL_RES * nrm)          # H v' = -omega v'
    Ul, Uln = to_host(h.partner_vectors(res.vectors, 1)), to_host(h.partner_vectors(res.vectors, 2))
    assert np.all(np.linalg.norm(Ul.conj().T @ H - om[:, None] * Ul.conj().T, axis=1) <= TOL_RES * nrm)   # u^H H = omega u^H
    assert np.all(np.linalg.norm(Uln.conj().T @ H + om[:, None] * Uln.conj().T, axis=1) <= TOL_RES * nrm)
    assert np.linalg.norm(Ul.conj().T @ V - np.eye(nev)) <= 1e-7 and np.linalg.norm(Uln.conj().T @ Vn + np.eye(nev)) <= 1e-7
    assert np.linalg.norm(Ul.conj().T @ Vn) <= 1e-7                                                      # bi-orthogonality across +-omega
    ht = b.Bse(b.MODE_TDA, N, pack(R, 0))
    assert b.lib().bse_partner_vectors(ht._h, res.vectors.data_ptr(), 2 * N, nev, 0, res.vectors.data_ptr(), 2 * N) == 1


def _golden(name):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", name)
    vals = [float(l.split()[0]) for l in open(path) if l.strip() and not l.startswith("#")]
    return np.array(vals)


def test_config1_full_vs_oracle_golden(orc):
    """BASELINE.json config 1.  The oracle's structure-preserving Lanczos needs many CPU-minutes at N = 2048, so its
    eigenvalues are stored (tests/golden/oracle_config1.txt, written by make_oracle_goldens.py from oracle/ only);
    residuals, Sigma-orthonormality and the -omega partner are checked live with the oracle apply."""
    import os
    import paper_2504_10096_b200 as b
    if not os.path.exists(os.path.join(os.path.dirname(__file__), "golden", "oracle_config1.txt")):
        pytest.skip("tests/golden/oracle_config1.txt not generated yet (python tests/golden/make_oracle_goldens.py)")
    cfg = gen.CONFIGS[1]
    N, nev, k = cfg["N"], cfg["nev"], cfg["k"]
    R = gen.dense_R(N, 1, sigma=cfg["sigma"]); C = gen.dense_C(N, 1)
    res = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1)).solve(nev, k, tol=TOL_SMALL, seed=1)
    # Reading R1: every omega^2 is a DOUBLE eigenvalue of G = M o P on C^N ~ R^2N; oracle and CUDA solver
    # both count eigenvectors of H (the copy is recognised by its vector), so the stored list is 20 distinct omega.
    gold = _golden("oracle_config1.txt")
    assert len(gold) == nev and np.all(np.diff(gold) > 1e-6 * gold[1:])
    _check_full(orc, R, C, res, nev, gold)


def test_config0_matches_stored_oracle_values(orc):
    import paper_2504_10096_b200 as b
    cfg = gen.CONFIGS[0]
    for sigma in (0.0, 1.0):
        R = gen.dense_R(cfg["N"], 1, sigma=sigma, group=cfg["group"])
        res = b.Bse(b.MODE_TDA, cfg["N"], pack(R, 0)).solve(cfg["nev"], cfg["k"], tol=TOL_SMALL, seed=5)
        ref = _golden(f"oracle_config0_sigma{int(sigma)}.txt")
        assert np.max(np.abs(res.omega - ref) / np.abs(ref)) <= TOL_EIG


def test_full_closed_form_pair():
    import torch
    import paper_2504_10096_b200 as b
    N, nev, k = 2048, 10, 4
    d1 = gen.prescribed_spectrum(N, 7, 1.0, 9.0, power=2 / 3); d2 = gen.prescribed_spectrum(N, 8, 2.0, 5.0, power=2 / 3)
    ur = gen.householder_u(N, 9, complex_u=False).real.copy(); phi = gen.phases(N, 9)
    rt, ct = b.bse_fill_closed_form_full(N, *(torch.from_numpy(a).cuda() for a in (d1, d2, ur, phi)),
                                         float(np.sum(d1 * ur ** 2)), float(np.sum(d2 * ur ** 2)))
    res = b.Bse(b.MODE_FULL, N, rt, ct).solve(nev, k, tol=1e-9, seed=4)
    exact = np.sort(np.sqrt(d1 * d2))[:nev]
    assert np.max(np.abs(res.omega - exact) / exact) <= TOL_EIG


def test_not_positive_definite_is_reported():
    import paper_2504_10096_b200 as b
    N = 256
    R = gen.dense_R(N, 3, sigma=0.0) - 20 * np.eye(N); C = gen.dense_C(N, 3)
    res = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1)).solve(4, 2, raise_on_error=False)
    assert res.status == 5


def test_solve_invalid_arguments_and_nonconvergence():
    import paper_2504_10096_b200 as b
    N = 128
    R = gen.dense_R(N, 3)
    h = b.Bse(b.MODE_TDA, N, pack(R, 0))
    assert h.solve(0, 4, raise_on_error=False).status == 1
    assert h.solve(126, 4, raise_on_error=False).status == 1       # nev + k > N
    r = h.solve(8, 2, ncv=12, tol=1e-14, max_restarts=1, raise_on_error=False)
    assert r.status == 4 and r.info["n_restart"] == 1               # best estimates are still returned
    assert np.all(np.isfinite(r.omega))


def _closed_tda(N, seed):
    import torch
    import paper_2504_10096_b200 as b
    lam = gen.prescribed_spectrum(N, seed, 1.0, 10.0, power=2 / 3)
    u = gen.householder_u(N, seed)
    t = b.bse_fill_closed_form_tda(N, torch.from_numpy(lam).cuda(), torch.from_numpy(u).cuda(),
                                   float(np.sum(lam * np.abs(u) ** 2)))
    return b.Bse(b.MODE_TDA, N, t), lam


def test_config2_size_closed_form_nev100():
    """Config 2's size and request (N = 16384, nev = 100, k = 4, tol 1e-8) on an instance whose spectrum is known
    exactly (R = Q diag(lam) Q^H): the CPU oracle cannot diagonalise N = 16384 in test time, the closed form can."""
    h, lam = _closed_tda(16384, 21)
    res = h.solve(100, 4, tol=1e-8, seed=1)
    assert np.max(np.abs(res.omega - lam[:100]) / lam[:100]) <= TOL_EIG
    V = res.vectors
    G = (V.conj() @ V.T).cpu().numpy()
    assert np.linalg.norm(G - np.eye(100)) <= 1e-11
    R = h.apply(V)                                     # residual through the CUDA apply (parity-tested separately)
    import torch
    r = (R - V * torch.from_numpy(res.omega).cuda()[:, None]).norm(dim=1).cpu().numpy()
    assert np.all(r <= TOL_RES * 10.0)


def test_config3_size_closed_form_pair():
    """Config 3's size (full mode, N = 32768, operator 65536) on the closed-form pair with omega = sqrt(d1 d2)."""
    import torch
    import paper_2504_10096_b200 as b
    N, nev, k = 32768, 100, 4
    if torch.cuda.mem_get_info()[0] < 30e9:
        pytest.skip("needs 30 GB of free device memory")
    d1 = gen.prescribed_spectrum(N, 7, 1.0, 9.0, power=2 / 3); d2 = gen.prescribed_spectrum(N, 8, 2.0, 5.0, power=2 / 3)
    ur = gen.householder_u(N, 9, complex_u=False).real.copy(); phi = gen.phases(N, 9)
    rt, ct = b.bse_fill_closed_form_full(N, *(torch.from_numpy(a).cuda() for a in (d1, d2, ur, phi)),
                                         float(np.sum(d1 * ur ** 2)), float(np.sum(d2 * ur ** 2)))
    res = b.Bse(b.MODE_FULL, N, rt, ct).solve(nev, k, tol=1e-8, seed=4)
    exact = np.sort(np.sqrt(d1 * d2))[:nev]
    assert np.max(np.abs(res.omega - exact) / exact) <= TOL_EIG
    # the same stores in the real form of Eq. (3) (S = R + C, D = R - C), block k = 8
    b.bse_to_real_form(rt, ct, N)
    res = b.Bse(b.MODE_FULL, N, rt, ct, storage=b.STORE_REAL_FORM).solve(nev, 8, tol=1e-8, seed=4)
    assert np.max(np.abs(res.omega - exact) / exact) <= TOL_EIG
    assert res.info["basis_orth_err"] <= TOL_ORTH


def test_config4_size_closed_form():
    """Config 4's size and request (N = 98304, 77 GB operand, nev = 500, k = 8, tol 1e-8) with a prescribed spectrum:
    the restart logic at a basis of 1000 columns with hundreds of locked pairs, against exactly known eigenvalues."""
    import torch
    if torch.cuda.mem_get_info()[0] < 100e9:
        pytest.skip("needs 100 GB of free device memory")
    h, lam = _closed_tda(98304, 23)
    res = h.solve(500, 8, tol=1e-8, seed=2)
    assert np.max(np.abs(res.omega - lam[:500]) / lam[:500]) <= TOL_EIG
    assert res.info["basis_orth_err"] <= TOL_ORTH


@pytest.mark.parametrize("seed", [2, 3])
def test_config0_other_matrix_seeds(orc, seed):
    """repeat config 0 with seeds 2 and 3 (new matrix, new start block)."""
    import paper_2504_10096_b200 as b
    cfg = gen.CONFIGS[0]
    R = gen.dense_R(cfg["N"], seed, sigma=1.0, group=cfg["group"])
    res = b.Bse(b.MODE_TDA, cfg["N"], pack(R, 0)).solve(cfg["nev"], cfg["k"], tol=TOL_SMALL, seed=seed)
    _check_tda(orc, R, res, cfg["nev"], np.linalg.eigvalsh(R))
    w_o, _, _, steps = orc.lanczos_tda(R, cfg["nev"], 1e-10, gen.block_X(cfg["N"], 1, 90 + seed)[:, 0], check=20)
    assert steps > 0 and np.max(np.abs(res.omega - w_o) / np.abs(w_o)) <= TOL_EIG


def test_tda_locking_returns_the_same_pairs(orc, monkeypatch):
    """Converged leading Ritz pairs are locked at restarts (Rayleigh-Ritz on the active columns only): same eigenpairs as
    without locking, ascending order, residuals through the oracle apply; many restarts (small basis) so that pairs are
    locked long before the end."""
    import paper_2504_10096_b200 as b
    N, nev, k = 1024, 40, 4
    R = gen.dense_R(N, 6, sigma=0.0)
    h = b.Bse(b.MODE_TDA, N, pack(R, 0))
    res = h.solve(nev, k, ncv=96, tol=1e-10, seed=5)
    monkeypatch.setenv("BSE_SOLVE_LOCK", "0")
    ref = h.solve(nev, k, ncv=96, tol=1e-10, seed=5)
    monkeypatch.delenv("BSE_SOLVE_LOCK")
    assert res.info["n_restart"] >= 5
    w = np.linalg.eigvalsh(R)[:nev]
    for r_ in (res, ref):
        assert np.all(np.diff(r_.omega) > 0)
        assert np.max(np.abs(r_.omega - w) / np.abs(w)) <= TOL_EIG
    _check_tda(orc, R, res, nev, w)
    assert abs(res.info["n_apply"] - ref.info["n_apply"]) <= max(8, ref.info["n_apply"] // 10)
    assert res.info["seconds_project"] <= ref.info["seconds_project"] * 1.5 + 0.05
