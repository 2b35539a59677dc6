"""bse_solve_direct (the diagonalisation scheme of PAPER.md section 2.1, Eq. 2-4, on the device) against the oracle's own
section-2.1 route, the closed-form pair omega = sqrt(d1 d2), the stored oracle values of config 1 and the iterative solver.
Eigenvalues rel. error <= 1e-10, residuals through the ORACLE apply <= 1e-8 ||H||, X^H X - Y^H Y = 1."""
import numpy as np
import pytest

import bse_inputs as gen
from gpu_util import pack, to_host

pytestmark = pytest.mark.gpu
TOL_EIG, TOL_RES = 1e-10, 1e-8


def _check_vectors(orc, R, C, om, V, nrm):
    N = R.shape[0]
    HV = orc.apply_full(R, C, V)
    r = np.linalg.norm(HV - V * om, axis=0) / np.linalg.norm(V, axis=0)
    assert np.all(r <= TOL_RES * nrm), r.max()
    Sig = np.concatenate([np.ones(N), -np.ones(N)])
    G = V.conj().T @ (Sig[:, None] * V)
    assert np.max(np.abs(np.diag(G) - 1)) <= 1e-10              # X^H X - Y^H Y = 1
    off = G - np.diag(np.diag(G))
    assert np.max(np.abs(off)) <= 1e-7                            # Sigma-orthogonal to their own accuracy (reading S10)


@pytest.mark.parametrize("N,seed", [(64, 3), (128, 5), (320, 7)])
def test_whole_spectrum_vs_oracle_direct_route(orc, N, seed):
    """Every positive omega and every eigenvector (nev = N: the direct route's use case)."""
    import paper_2504_10096_b200 as b
    R = gen.dense_R(N, seed, sigma=1.0); C = gen.dense_C(N, seed)
    om_o, _ = orc.bse_direct(R, C, want_vectors=False)
    h = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    om, vec, sec = h.solve_direct(N)
    assert np.all(np.diff(om) >= 0)
    assert np.max(np.abs(om - om_o[N:]) / om_o[N:]) <= TOL_EIG
    nrm = np.linalg.norm(np.block([[R, C], [-C.conj().T, -R.conj()]]), 2)
    _check_vectors(orc, R, C, om, to_host(vec), nrm)
    assert sec["total"] > 0
    # eigenvalues only: same values, no vectors
    om2, v2, _ = h.solve_direct(7, vectors=False)
    assert v2 is None and np.max(np.abs(om2 - om[:7])) <= 1e-13 * om[6]


def test_sum_rule_and_partner_vectors(orc):
    """Sum of omega^2 = ||R||_F^2 - ||C||_F^2 (fixed by tr H^2, independent of any solver) and the -omega partners."""
    import paper_2504_10096_b200 as b
    N = 256
    R = gen.dense_R(N, 11, sigma=1.0); C = gen.dense_C(N, 11)
    h = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    om, vec, _ = h.solve_direct(N)
    want = np.linalg.norm(R) ** 2 - np.linalg.norm(C) ** 2
    assert abs(np.sum(om ** 2) - want) <= 1e-11 * want
    Pn = to_host(h.partner_vectors(vec[:16], 0))
    rp = np.linalg.norm(orc.apply_full(R, C, Pn) + Pn * om[:16], axis=0) / np.linalg.norm(Pn, axis=0)
    assert np.all(rp <= TOL_RES * 13.0)


def test_not_positive_definite_is_reported():
    """the Cholesky factorisation exists only if M is positive definite; sigma = 0 gives an indefinite Omega."""
    import paper_2504_10096_b200 as b
    N = 256
    R = gen.dense_R(N, 1, sigma=0.0); C = gen.dense_C(N, 1)
    lam = np.linalg.eigvalsh(np.block([[R, C], [C.conj(), R.conj()]]))
    assert lam[0] < 0
    h = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    with pytest.raises(b.BseError) as e:
        h.solve_direct(4)
    assert e.value.status == 5                                  # BSE_ERR_NOT_POSITIVE_DEFINITE
    with pytest.raises(b.BseError):
        b.Bse(b.MODE_TDA, N, pack(R, 0)).solve_direct(4)       # full mode only


@pytest.mark.parametrize("store", ["c128", "real_form", "c64"])
def test_closed_form_pair_every_store(store):
    """omega_i = sqrt(d1_i d2_i) exactly: N = 1024, the lowest 40 and the whole list."""
    import torch
    import paper_2504_10096_b200 as b
    N = 1024
    d1 = gen.prescribed_spectrum(N, 21, 1.0, 9.0, power=0.8)
    d2 = gen.prescribed_spectrum(N, 22, 0.5, 7.0, power=0.9)
    ur = gen.householder_u(N, 23, complex_u=False).real.copy(); phi = gen.phases(N, 24)
    storage = b.STORE_C64 if store == "c64" else b.STORE_C128
    tr, tc = b.bse_fill_closed_form_full(N, *(torch.from_numpy(a).cuda() for a in (d1, d2, ur, phi)),
                                         float(np.sum(d1 * ur ** 2)), float(np.sum(d2 * ur ** 2)), storage=storage)
    if store == "real_form":
        b.bse_to_real_form(tr, tc, N)
        storage = b.STORE_REAL_FORM
    h = b.Bse(b.MODE_FULL, N, tr, tc, storage=storage)
    want = np.sort(np.sqrt(d1 * d2))
    om, vec, sec = h.solve_direct(N, vectors=False)
    tol = 2e-6 if store == "c64" else TOL_EIG                      # binary32 data: within its own precision
    assert np.max(np.abs(om - want) / want) <= tol
    om40, vec40, _ = h.solve_direct(40)
    assert np.max(np.abs(om40 - want[:40]) / want[:40]) <= tol
    # residuals through the library's own apply are a consistency check only; the eigenvalues above are the pin
    HV = h.apply(vec40)
    r = torch.linalg.vector_norm(HV - vec40 * torch.from_numpy(om40).cuda()[:, None], dim=1) / torch.linalg.vector_norm(vec40, dim=1)
    assert float(r.max()) <= 1e-8 * 10.0


def test_config1_stored_oracle_values_and_iterative_solver(orc):
    """BASELINE.json config 1 (N = 2048, operator 4096 x 4096): the 20 stored oracle values, live residuals through the oracle
    apply, and agreement with bse_solve on the same handle."""
    import os
    import paper_2504_10096_b200 as b
    cfg = gen.CONFIGS[1]
    N, nev = cfg["N"], cfg["nev"]
    R = gen.dense_R(N, 1, sigma=cfg["sigma"]); C = gen.dense_C(N, 1)
    h = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    om, vec, sec = h.solve_direct(nev)
    path = os.path.join(os.path.dirname(__file__), "golden", "oracle_config1.txt")
    ref = np.array([float(l.split()[0]) for l in open(path) if l.strip() and not l.startswith("#")])[:nev]
    assert len(ref) == nev
    assert np.max(np.abs(om - ref) / ref) <= TOL_EIG
    _check_vectors(orc, R, C, om, to_host(vec), 12.0)
    it = h.solve(nev, cfg["k"], tol=1e-10, seed=1)
    assert np.max(np.abs(it.omega - om) / om) <= TOL_EIG


@pytest.mark.parametrize("seed", range(14))
def test_random_sizes_and_stores_vs_oracle_direct_route(orc, seed):
    """Seeded sweep: N below one tile, ragged last tiles and last Cholesky blocks, every store; all eigenpairs against the
    oracle's section-2.1 route on the operator the store defines."""
    import paper_2504_10096_b200 as b
    from gpu_util import to_dev
    rng = np.random.default_rng(4000 + seed)
    N = int(rng.choice([1, 2, 7, 31, 33, 63, 65, 100, 129, 200, 257]))
    store = str(rng.choice(["c128", "c64", "real", "real64"]))
    Np = N if N % 16 == 0 else N + 16 - N % 16
    R = gen.dense_R(Np, 300 + seed, sigma=1.0)[:N, :N]
    C = gen.dense_C(Np, 300 + seed)[:N, :N]
    base = b.STORE_C64 if store in ("c64", "real64") else b.STORE_C128
    rt = b.bse_pack_from_dense(to_dev(R), N, 0, storage=base)
    ct = b.bse_pack_from_dense(to_dev(C), N, 1, storage=base)
    if base == b.STORE_C64:
        R, C = orc.round_c64(R), orc.round_c64(C)
    storage = base
    if store.startswith("real"):
        b.bse_to_real_form(rt, ct, N, storage=base)
        storage = b.STORE_REAL_FORM if base == b.STORE_C128 else b.STORE_REAL_FORM_C64
        if base == b.STORE_C64:                                # the operator the rounded planes define (include/bse.h)
            S32, D32 = orc.round_c64(R + C), orc.round_c64(R - C)
            R, C = (S32 + D32) / 2, (S32 - D32) / 2
    h = b.Bse(b.MODE_FULL, N, rt, ct, storage=storage)
    om_o, _ = orc.bse_direct(R, C, want_vectors=False)
    nev = N if seed % 3 else max(1, N // 5)
    om, vec, _ = h.solve_direct(nev)
    assert np.max(np.abs(om - om_o[N:N + nev]) / om_o[N:N + nev]) <= TOL_EIG, (N, store)
    nrm = np.linalg.norm(np.block([[R, C], [-C.conj().T, -R.conj()]]), 2)
    V = to_host(vec)
    r = np.linalg.norm(orc.apply_full(R, C, V) - V * om, axis=0) / np.linalg.norm(V, axis=0)
    assert np.all(r <= TOL_RES * nrm), (N, store, r.max())
    Sig = np.concatenate([np.ones(N), -np.ones(N)])
    assert np.max(np.abs(np.sum(Sig[:, None] * np.abs(V) ** 2, axis=0) - 1)) <= 1e-10
