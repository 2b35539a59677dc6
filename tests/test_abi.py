"""CPU-side checks of the boundary: the library loads, exports every symbol include/bse.h declares, and the host
logic (layout arithmetic, status strings, projected eigensolver) is right.  No compute calls need a GPU here."""
import ctypes
import os
import re

import numpy as np
import pytest

import bse_inputs as gen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def b():
    from paper_2504_10096_b200 import build
    build.build()
    import paper_2504_10096_b200 as pkg
    return pkg


def test_header_symbols_are_exported(b):
    hdr = open(os.path.join(ROOT, "include", "bse.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(bse_[a-z_0-9]+)\s*\(", hdr))
    assert {"bse_create", "bse_apply", "bse_orth", "bse_solve", "bse_destroy"} <= declared
    L = b.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(b.EXPORTS)


def test_layout_and_status(b):
    assert b.bse_layout(64) == (64, 1, 65536)
    assert b.bse_layout(65) == (64, 3, 3 * 65536)
    assert b.bse_layout(65, b.STORE_C64) == (64, 3, 3 * 32768)      # complex64 store: half the bytes, same tiles
    with pytest.raises(b.BseError):
        b.bse_layout(64, 7)
    for N, nbytes in [(1024, 8.40e6), (16384, 2.148e9), (98304, 77.31e9)]:
        t, nt, by = b.bse_layout(N)
        n = N // 64
        assert nt == n * (n + 1) // 2 and by == nt * 65536
        # B_mat = 16 N (N+1) / 2 plus the mirrored halves of the diagonal tiles
        assert abs(by - nbytes) / nbytes < 1.0 / n
    with pytest.raises(b.BseError):
        b.bse_layout(0)
    assert b.lib().bse_status_string(0) == b"ok"
    assert b"positive" in b.lib().bse_status_string(5)


def test_no_compute_without_arguments(b):
    # argument validation happens before any CUDA call
    h = ctypes.c_void_p()
    assert b.lib().bse_create(ctypes.byref(h), 7, 0, 64, None, None, None) == 1
    assert b.lib().bse_create(ctypes.byref(h), 0, 9, 64, ctypes.c_void_p(16), None, None) == 1     # unknown storage
    assert b.lib().bse_apply(None, None, 0, None, 0, 1) == 1
    assert b.lib().bse_solve(None, 1, 1, 0, 1e-8, 1, 0, None, None, 0, None, None) == 1


@pytest.mark.parametrize("m", [1, 2, 7, 40, 150])
def test_host_heev_matches_numpy(b, m):
    A = gen.block_X(m, m, m)
    A = (A + A.conj().T) / 2
    w, Z = b.host_heev(A)
    ref = np.linalg.eigvalsh(A)
    scale = max(np.max(np.abs(ref)), 1.0)
    assert np.max(np.abs(w - ref)) < 1e-13 * scale * max(m, 8)
    assert np.linalg.norm(Z.conj().T @ Z - np.eye(m)) < 1e-12
    assert np.linalg.norm(A @ Z - Z * w) < 1e-12 * scale * m


def test_host_heev_arrowhead_and_clusters(b):
    # the projected matrix after a thick restart: diag(theta) bordered by a block, plus repeated eigenvalues
    l, k = 30, 4
    T = np.zeros((l + k, l + k), dtype=complex)
    T[np.arange(l), np.arange(l)] = np.repeat(np.linspace(1, 3, l // 2), 2)      # pairs, as in full mode
    Bk = gen.block_X(k, l, 3) * 1e-3
    T[l:, :l] = Bk; T[:l, l:] = Bk.conj().T
    D = gen.block_X(k, k, 4); T[l:, l:] = (D + D.conj().T) / 2 + 5 * np.eye(k)
    w, Z = b.host_heev(T, nz=10)
    assert np.max(np.abs(w - np.linalg.eigvalsh(T))) < 1e-13 * 10
    assert np.linalg.norm(T @ Z - Z * w[:10]) < 1e-12
    # real symmetric input gives real eigenvectors up to a phase (full-mode T is real)
    Tr = T.real.copy()
    w2, Z2 = b.host_heev(Tr, nz=6)
    assert np.linalg.norm(Tr @ Z2 - Z2 * w2[:6]) < 1e-12 and np.max(np.abs(Z2.imag)) < 1e-13


@pytest.mark.parametrize("m", [1, 2, 7, 40, 150, 600])
def test_host_syev_matches_numpy(b, m):
    # the real symmetric driver used for the full-mode projected matrix (include/bse.h: bse_host_syev)
    A = gen.block_X(m, m, m + 1).real
    A = (A + A.T) / 2
    nz = m if m < 600 else 200
    w, Z = b.host_syev(A, nz=nz)
    ref = np.linalg.eigvalsh(A)
    scale = max(np.max(np.abs(ref)), 1.0)
    assert np.max(np.abs(w - ref)) < 1e-13 * scale * max(m, 8)
    assert np.linalg.norm(Z.T @ Z - np.eye(nz)) < 1e-12 * max(1, m / 50)
    assert np.linalg.norm(A @ Z - Z * w[:nz]) < 1e-12 * scale * m
    # the strictly upper triangle is never read
    A2 = np.tril(A) + np.triu(np.full((m, m), 7.0), 1)
    w2, _ = b.host_syev(A2, nz=0)
    assert np.array_equal(w2, w)


def test_host_syev_arrowhead_with_pairs_agrees_with_heev(b):
    # full-mode projected matrix after a thick restart: paired Ritz values on the diagonal, a real border block
    l, k = 40, 8
    T = np.zeros((l + k, l + k))
    T[np.arange(l), np.arange(l)] = np.repeat(np.linspace(0.3, 0.6, l // 2), 2)
    Bk = gen.block_X(k, l, 5).real * 1e-4
    T[l:, :l] = Bk; T[:l, l:] = Bk.T
    D = gen.block_X(k, k, 6).real; T[l:, l:] = (D + D.T) / 2 + 4 * np.eye(k)
    w, Z = b.host_syev(T, nz=l)
    wh, _ = b.host_heev(T.astype(complex), nz=0)
    assert np.max(np.abs(w - np.linalg.eigvalsh(T))) < 1e-13 * 10 and np.max(np.abs(w - wh)) < 1e-13 * 10
    assert np.linalg.norm(T @ Z - Z * w[:l]) < 1e-12 and np.linalg.norm(Z.T @ Z - np.eye(l)) < 1e-12


def test_quadrature_resolvent_host_utility_matches_oracle(b, orc):
    # host logic only: the continued fraction of a Jacobi matrix, against the oracle's and against (z - T)^-1 directly
    m = 17
    rng_a = np.linspace(1.0, 3.0, m) + 0.1 * np.cos(np.arange(m))
    beta = np.concatenate([[2.5], 0.3 + 0.05 * np.arange(m)])
    om = np.linspace(0.0, 4.0, 33)
    G = b.quadrature_resolvent(rng_a, beta, om, 0.07)
    assert np.max(np.abs(G - orc.quadrature_resolvent(rng_a, beta, om, 0.07))) < 1e-13 * np.max(np.abs(G))
    T = np.diag(rng_a) + np.diag(beta[1:m], 1) + np.diag(beta[1:m], -1)
    direct = np.array([beta[0] ** 2 * np.linalg.inv((w + 0.07j) * np.eye(m) - T)[0, 0] for w in om])
    assert np.max(np.abs(G - direct)) < 1e-11 * np.max(np.abs(direct))


def test_host_stev_vs_scipy():
    """bse_host_stev (last stage of bse_solve_direct): real symmetric tridiagonal, all eigenvalues + the lowest vectors."""
    import paper_2504_10096_b200 as b
    from scipy.linalg import eigh_tridiagonal
    rng = np.random.default_rng(5)
    for m, nz in [(1, 1), (2, 2), (37, 5), (300, 300), (513, 40), (2000, 150), (64, 16)]:     # nz <= m/4: inverse iteration
        d = rng.standard_normal(m) * 3
        e = rng.standard_normal(max(m - 1, 0))
        w, Z = b.host_stev(d, e, nz)
        T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
        wr = eigh_tridiagonal(d, e, eigvals_only=True) if m > 1 else d.copy()
        assert np.max(np.abs(w - wr)) <= 1e-13 * max(1.0, np.max(np.abs(wr)))
        assert np.linalg.norm(T @ Z - Z * w[:nz]) <= 1e-12 * np.linalg.norm(T) * np.sqrt(nz)
        assert np.linalg.norm(Z.T @ Z - np.eye(nz)) <= 1e-12 * np.sqrt(nz)
    # zero diagonal (the direct route's matrix): eigenvalues in +- pairs
    e = rng.standard_normal(63)
    w, _ = b.host_stev(np.zeros(64), e, 0)
    assert np.max(np.abs(w + w[::-1])) <= 1e-13 * np.max(np.abs(w))


def test_host_stev_clusters():
    """Inverse iteration inside clusters: Wilkinson's W21+ (pairs agreeing to 1e-14) glued three times (a cluster of close
    triples), and the direct route's own matrix B^T B of a bidiagonal with repeated singular values nearby."""
    import paper_2504_10096_b200 as b
    n1 = 21
    d1 = np.abs(np.arange(n1) - 10.0)
    d = np.concatenate([d1, d1, d1, d1]); e = np.ones(len(d) - 1); e[n1 - 1::n1] = 1e-9
    m = len(d)
    T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
    w_ref = np.linalg.eigvalsh(T)
    nz = m // 4
    w, Z = b.host_stev(d, e, nz)
    assert np.max(np.abs(w - w_ref)) <= 1e-13 * np.max(np.abs(w_ref))
    assert np.linalg.norm(T @ Z - Z * w[:nz]) <= 1e-11 * np.linalg.norm(T)
    assert np.linalg.norm(Z.T @ Z - np.eye(nz)) <= 1e-10


def test_host_stev_lowest_bisection_vs_scipy():
    """A few lowest eigenpairs by bisection + inverse iteration (8 nz <= m), and the fall-through to the full solver."""
    import paper_2504_10096_b200 as b
    from scipy.linalg import eigh_tridiagonal
    rng = np.random.default_rng(9)
    for m, nz in [(1000, 25), (1000, 125), (300, 100), (65, 8), (2048, 1)]:
        d = rng.uniform(0.3, 150.0, m)
        e = rng.standard_normal(m - 1) * 2
        wr = eigh_tridiagonal(d, e, eigvals_only=True)
        w, Z = b.host_stev_lowest(d, e, nz)
        assert np.max(np.abs(w - wr[:nz])) <= 2e-14 * np.max(np.abs(wr))
        T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
        assert np.linalg.norm(T @ Z - Z * w) <= 1e-11 * np.linalg.norm(T)
        assert np.linalg.norm(Z.T @ Z - np.eye(nz)) <= 1e-10
        w2, none = b.host_stev_lowest(d, e, nz, vectors=False)
        assert none is None and np.array_equal(w2, w) or np.max(np.abs(w2 - w)) <= 2e-14 * np.max(np.abs(wr))
    # a zero-diagonal matrix (pairs +-sigma): the lowest are the most negative
    e = rng.standard_normal(511)
    w, _ = b.host_stev_lowest(np.zeros(512), e, 10, vectors=False)
    wr = eigh_tridiagonal(np.zeros(512), e, eigvals_only=True)
    assert np.max(np.abs(w - wr[:10])) <= 2e-14 * np.max(np.abs(wr))
