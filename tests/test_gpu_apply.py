"""Parity of the CUDA apply path (through the C ABI) against the CPU oracle, element by element."""
import numpy as np
import pytest

import bse_inputs as gen
from gpu_util import pack, relerr, to_dev, to_host

pytestmark = pytest.mark.gpu

TOL_APPLY = 1e-12      # north_star: apply normwise relative error <= 1e-12


def _herm(n, seed):
    A = gen.block_X(n, n, seed)
    A = (A + A.conj().T) / 2
    A[np.diag_indices(n)] = A.diagonal().real
    return A


def _sym(n, seed):
    A = gen.block_X(n, n, seed)
    return (A + A.T) / 2


@pytest.mark.parametrize("N", [1, 8, 64, 100, 257])
@pytest.mark.parametrize("which", [0, 1])
def test_pack_unpack_roundtrip(N, which):
    import paper_2504_10096_b200 as b
    A = _herm(N, 3) if which == 0 else _sym(N, 4)
    junk = A.copy()
    junk[np.triu_indices(N, 1)] = 1e30          # the strictly upper triangle must never be read
    tiles = pack(junk, which)
    back = to_host(b.bse_unpack_to_dense(tiles, N, which))
    assert np.array_equal(back, A)


def test_pack_drops_imaginary_diagonal_of_R():
    import paper_2504_10096_b200 as b
    N = 70
    A = _herm(N, 5) + 1j * np.eye(N)
    back = to_host(b.bse_unpack_to_dense(pack(A, 0), N, 0))
    assert np.all(back.diagonal().imag == 0)


@pytest.mark.parametrize("N,group", [(256, 16), (320, 64)])
def test_device_generator_matches_cpu_generator(N, group):
    import paper_2504_10096_b200 as b
    R = gen.dense_R(N, 7, sigma=0.5, group=group)
    C = gen.dense_C(N, 7)
    Rd = to_host(b.bse_unpack_to_dense(b.bse_fill_synthetic(N, 0, 7, 0.5, group), N, 0))
    Cd = to_host(b.bse_unpack_to_dense(b.bse_fill_synthetic(N, 1, 7), N, 1))
    # same integer hash on both sides; log / sincos differ by a few ulp
    assert np.max(np.abs(Rd - R)) < 1e-14
    assert np.max(np.abs(Cd - C)) < 1e-14
    assert np.array_equal(Rd, Rd.conj().T) and np.array_equal(Cd, Cd.T)


def test_closed_form_fill_matches_cpu():
    import torch
    import paper_2504_10096_b200 as b
    N = 200
    lam = gen.prescribed_spectrum(N, 5); u = gen.householder_u(N, 5)
    s = float(np.sum(lam * np.abs(u) ** 2))
    t = b.bse_fill_closed_form_tda(N, torch.from_numpy(lam).cuda(), torch.from_numpy(u).cuda(), s)
    Rd = to_host(b.bse_unpack_to_dense(t, N, 0))
    assert np.max(np.abs(Rd - gen.closed_form_tda_dense(lam, u))) < 1e-13
    d1 = gen.prescribed_spectrum(N, 7, 1.0, 9.0); d2 = gen.prescribed_spectrum(N, 8, 2.0, 5.0)
    ur = gen.householder_u(N, 9, complex_u=False).real.copy(); phi = gen.phases(N, 9)
    rt, ct = b.bse_fill_closed_form_full(N, *(torch.from_numpy(a).cuda() for a in (d1, d2, ur, phi)),
                                         float(np.sum(d1 * ur ** 2)), float(np.sum(d2 * ur ** 2)))
    R, C = gen.closed_form_full_dense(d1, d2, ur, phi)
    assert np.max(np.abs(to_host(b.bse_unpack_to_dense(rt, N, 0)) - R)) < 1e-13
    assert np.max(np.abs(to_host(b.bse_unpack_to_dense(ct, N, 1)) - C)) < 1e-13


def test_identity_and_diagonal_exact():
    import paper_2504_10096_b200 as b
    N, k = 200, 3
    X = gen.block_X(N, k, 5)
    h = b.Bse(b.MODE_TDA, N, pack(np.eye(N, dtype=complex), 0))
    assert np.array_equal(to_host(h.apply(to_dev(X))), X)
    d = np.linspace(-2, 3, N)
    h = b.Bse(b.MODE_TDA, N, pack(np.diag(d).astype(complex), 0))
    assert np.array_equal(to_host(h.apply(to_dev(X))), d[:, None] * X)


def test_unit_impulses_cover_tile_borders(orc):
    # every stored entry class: inside a diagonal tile (both triangles), off-diagonal tile, tile borders
    import paper_2504_10096_b200 as b
    N, k = 136, 2
    X = gen.block_X(N, k, 7)
    Xd = to_dev(X)
    for (i, j) in [(5, 2), (63, 0), (64, 63), (65, 64), (127, 64), (128, 0), (135, 127), (135, 135), (100, 37)]:
        R = np.zeros((N, N), dtype=complex)
        R[i, j] = 0.7 - 1.3j
        Y = to_host(b.Bse(b.MODE_TDA, N, pack(R, 0)).apply(Xd))
        assert np.allclose(Y, orc.apply_tda(R, X), rtol=0, atol=1e-15), (i, j)


@pytest.mark.parametrize("N", [64, 100, 320, 1024])
@pytest.mark.parametrize("k", [1, 2, 3, 4, 5, 8])
def test_tda_apply_matches_oracle(orc, N, k):
    import paper_2504_10096_b200 as b
    R = _herm(N, 11) if N < 1024 else gen.dense_R(N, 1)
    X = gen.block_X(N, k, 12)
    Y = to_host(b.Bse(b.MODE_TDA, N, pack(R, 0)).apply(to_dev(X)))
    assert relerr(Y, orc.apply_tda(R, X)) <= TOL_APPLY


@pytest.mark.parametrize("N", [64, 200, 448])
@pytest.mark.parametrize("k", [1, 4, 6])
def test_full_apply_and_half_apply_match_oracle(orc, N, k):
    import paper_2504_10096_b200 as b
    R, C = _herm(N, 21), _sym(N, 22)
    h = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    X = gen.block_X(2 * N, k, 23)
    assert relerr(to_host(h.apply(to_dev(X))), orc.apply_full(R, C, X)) <= TOL_APPLY
    x = gen.block_X(N, k, 24)
    for sign in (+1, -1):
        assert relerr(to_host(h.apply_half(to_dev(x), sign)), orc.apply_half(R, C, x, sign)) <= TOL_APPLY


def test_apply_host_entry_point(orc):
    import paper_2504_10096_b200 as b
    N, k = 320, 4
    R = _herm(N, 31)
    X = gen.block_X(N, k, 32)
    h = b.Bse(b.MODE_TDA, N, pack(R, 0))
    Y = h.apply_host(np.ascontiguousarray(X.T)).T
    assert relerr(Y, orc.apply_tda(R, X)) <= TOL_APPLY


def test_invalid_arguments():
    import paper_2504_10096_b200 as b
    with pytest.raises(b.BseError):
        b.bse_layout(0)
    N = 64
    t = pack(np.eye(N, dtype=complex), 0)
    with pytest.raises(b.BseError):
        b.Bse(b.MODE_FULL, N, t, None)
    h = b.Bse(b.MODE_TDA, N, t)
    with pytest.raises(b.BseError):
        h.apply_half(to_dev(np.ones((N, 1))), +1)      # half apply is full-mode only


def _sampled_rows(N):
    # rows 0..7 of every tile (the slab of consumer warp 0, the first bytes a refill overwrites) plus a ragged mix
    base = (np.arange(N // 64)[:, None] * 64 + np.arange(8)[None, :]).reshape(-1)
    extra = (np.arange(97) * 2654435761 % N).astype(np.int64)
    return np.unique(np.concatenate([base, extra]))


@pytest.mark.parametrize("N,k,reps", [(4096, 4, 25), (8192, 4, 8), (16384, 8, 3), (16384, 1, 2)])
def test_tda_apply_many_units_per_cta_sampled_rows(orc, N, k, reps):
    """Sizes where every CTA walks many units (the launch configuration bench.py times at N = 16384).  The matrix
    is generated on the device; the oracle consumes the same rows from the CPU generator (bse_inputs.rows_R, equal
    to a few ulp).  Repeated to catch timing-dependent faults: round 1 had a shared-memory WAR hazard here that
    corrupted about one 8-row group per launch."""
    import paper_2504_10096_b200 as b
    h = b.Bse(b.MODE_TDA, N, b.bse_fill_synthetic(N, 0, 1, 0.0, 16))
    X = gen.block_X(N, k, 12)
    rows = _sampled_rows(N)
    ref = orc.rows_times_block(gen.rows_R(N, 1, rows, 0.0, 16), X)
    Xd = to_dev(X)
    for _ in range(reps):
        Y = to_host(h.apply(Xd))
        assert relerr(Y[rows], ref) <= TOL_APPLY
    # properties that hold at any size: Hermitian adjoint identity through the CUDA path
    Z = gen.block_X(N, k, 13)
    RZ = to_host(h.apply(to_dev(Z)))
    lhs, rhs = X.conj().T @ RZ, Y.conj().T @ Z
    assert np.linalg.norm(lhs - rhs) <= 1e-12 * np.linalg.norm(lhs)


def test_full_apply_many_units_sampled_rows(orc):
    import paper_2504_10096_b200 as b
    N, k = 4096, 4
    h = b.Bse(b.MODE_FULL, N, b.bse_fill_synthetic(N, 0, 2, 1.0, 16), b.bse_fill_synthetic(N, 1, 2))
    X = gen.block_X(2 * N, k, 5)
    rows = _sampled_rows(N)[::4]
    Rr, Cr = gen.rows_R(N, 2, rows, 1.0, 16), gen.rows_C(N, 2, rows)
    # rows of H = [[R, C], [-C^*, -R^*]] (Eq. 1, PAPER.md:18 with :26) assembled from generator rows
    top = np.hstack([Rr, Cr]); bot = np.hstack([-Cr.conj(), -Rr.conj()])
    ref = orc.rows_times_block(np.vstack([top, bot]), X)
    for _ in range(5):
        Y = to_host(h.apply(to_dev(X)))
        assert relerr(np.vstack([Y[rows], Y[N + rows]]), ref) <= TOL_APPLY


def test_config4_full_size_sampled_rows(orc):
    """BASELINE.json config 4 (N = 98304, 77 GB operand filled on the device): rows of Y sampled across the matrix,
    against the oracle fed with the same rows from the CPU generator, for every kernel bench.py times at this size
    (k = 1: plain-FMA kernel, k = 4: four-product DMMA kernel, k = 8: three-product DMMA kernel).  Needs ~80 GB of HBM."""
    import torch
    import paper_2504_10096_b200 as b
    cfg = gen.CONFIGS[4]
    N = cfg["N"]
    if torch.cuda.mem_get_info()[0] < 90e9:
        pytest.skip("needs 90 GB of free device memory")
    h = b.Bse(b.MODE_TDA, N, b.bse_fill_synthetic(N, 0, 1, 0.0, cfg["group"]))
    X = gen.block_X(N, 8, 12)
    rows = np.unique(np.concatenate([(np.arange(40) * 2654435761 % N), [0, 7, 63, 64, N - 65, N - 64, N - 1],
                                     np.arange(8) + 64 * 777]).astype(np.int64))
    ref = orc.rows_times_block(gen.rows_R(N, 1, rows, 0.0, cfg["group"]), X)
    for k in (4, 8, 1):
        Y = to_host(h.apply(to_dev(X[:, :k])))
        assert relerr(Y[rows], ref[:, :k]) <= TOL_APPLY, k
        Z = gen.block_X(N, k, 13)
        RZ = to_host(h.apply(to_dev(Z)))
        lhs, rhs = X[:, :k].conj().T @ RZ, Y.conj().T @ Z
        assert np.linalg.norm(lhs - rhs) <= 1e-12 * np.linalg.norm(lhs), k


def test_config3_full_size_half_apply_sampled_rows(orc):
    """BASELINE.json config 3 (full mode, N = 32768, R and C 8.6 GB each, filled on the device): sampled rows of
    P(X) = R X + C conj(X) and M(X) = R X - C conj(X) -- the two products bse_solve issues per block step -- for the
    four-product (k = 4) and three-product (k = 8) kernels and for the real-form kernel, against the oracle on rows from
    the CPU generator."""
    import torch
    import paper_2504_10096_b200 as b
    cfg = gen.CONFIGS[3]
    N = cfg["N"]
    if torch.cuda.mem_get_info()[0] < 30e9:
        pytest.skip("needs 30 GB of free device memory")
    rt, ct = b.bse_fill_synthetic(N, 0, 1, cfg["sigma"], cfg["group"]), b.bse_fill_synthetic(N, 1, 1, 0.0, cfg["group"])
    h = b.Bse(b.MODE_FULL, N, rt, ct)
    X = gen.block_X(N, 8, 14)
    rows = np.unique(np.concatenate([(np.arange(24) * 2654435761 % N), [0, 63, 64, N - 64, N - 1]]).astype(np.int64))
    RX = orc.rows_times_block(gen.rows_R(N, 1, rows, cfg["sigma"], cfg["group"]), X)
    CX = orc.rows_times_block(gen.rows_C(N, 1, rows), X.conj())
    for k in (4, 8):
        for sign in (+1, -1):
            Y = to_host(h.apply_half(to_dev(X[:, :k]), sign))
            assert relerr(Y[rows], (RX + sign * CX)[:, :k]) <= TOL_APPLY, (k, sign)
    # the general apply [Y1; Y2] = H [X1; X2] at the same size (two tile passes with 2k operand columns):
    # rows of the upper half  R X1 + C X2  and of the lower half  -conj(C) X1 - conj(R) X2  from the same generator rows
    X2 = gen.block_X(2 * N, 4, 15)
    Rrows, Crows = gen.rows_R(N, 1, rows, cfg["sigma"], cfg["group"]), gen.rows_C(N, 1, rows)
    up = orc.rows_times_block(np.hstack([Rrows, Crows]), X2)
    lo = orc.rows_times_block(np.hstack([-Crows.conj(), -Rrows.conj()]), X2)
    for k in (1, 3, 4):
        Y = to_host(h.apply(to_dev(X2[:, :k])))
        assert relerr(Y[rows], up[:, :k]) <= TOL_APPLY and relerr(Y[N + rows], lo[:, :k]) <= TOL_APPLY, ("general", k)
    # the same stores rewritten as S = R + C, D = R - C (real form of Eq. 3): same operator
    del h
    b.bse_to_real_form(rt, ct, N)
    hr = b.Bse(b.MODE_FULL, N, rt, ct, storage=b.STORE_REAL_FORM)
    for k in (4, 8):
        for sign in (+1, -1):
            Y = to_host(hr.apply_half(to_dev(X[:, :k]), sign))
            assert relerr(Y[rows], (RX + sign * CX)[:, :k]) <= TOL_APPLY, ("real form", k, sign)
    for k in (1, 4):
        Y = to_host(hr.apply(to_dev(X2[:, :k])))
        assert relerr(Y[rows], up[:, :k]) <= TOL_APPLY and relerr(Y[N + rows], lo[:, :k]) <= TOL_APPLY, ("general, real form", k)


@pytest.mark.parametrize("N", [1, 2, 63, 65, 127])
def test_tiny_and_ragged_sizes(orc, N):
    import paper_2504_10096_b200 as b
    R = _herm(N, 40 + N)
    for k in (1, 4, 7):
        X = gen.block_X(N, k, 41)
        Y = to_host(b.Bse(b.MODE_TDA, N, pack(R, 0)).apply(to_dev(X)))
        assert relerr(Y, orc.apply_tda(R, X)) <= TOL_APPLY


def test_leading_dimensions_and_side_stream(orc):
    """ldx, ldy > N through the raw C ABI, on a non-default stream."""
    import ctypes
    import torch
    import paper_2504_10096_b200 as b
    N, k, ldx, ldy = 200, 3, 256, 231
    R = _herm(N, 51)
    X = gen.block_X(N, k, 52)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        tiles = pack(R, 0)
        Xd = torch.full((k, ldx), 7.0 + 1j, dtype=torch.complex128, device="cuda")
        Xd[:, :N] = to_dev(X)
        Yd = torch.full((k, ldy), 3.0 - 2j, dtype=torch.complex128, device="cuda")
        h = b.Bse(b.MODE_TDA, N, tiles)                       # captures the current (side) stream
        st = b.lib().bse_apply(h._h, Xd.data_ptr(), ldx, Yd.data_ptr(), ldy, k)
        assert st == 0
    s.synchronize()
    Y = to_host(Yd)
    assert relerr(Y[:N], orc.apply_tda(R, X)) <= TOL_APPLY
    assert np.all(Y[N:] == 3.0 - 2j)                          # padding rows of Y are not touched
    assert b.lib().bse_apply(h._h, Xd.data_ptr(), N - 1, Yd.data_ptr(), ldy, k) == 1     # ld < N
    assert b.lib().bse_apply(h._h, Xd.data_ptr(), ldx, Yd.data_ptr(), ldy, 0) == 1       # k < 1
    assert b.lib().bse_apply(h._h, Xd.data_ptr(), ldx, Xd.data_ptr(), ldx, k) == 1       # aliasing


@pytest.mark.parametrize("k", [5, 7, 8, 9, 11, 16])
def test_column_groups_agree_with_oracle(orc, k):
    """k > 4: 5..8 columns per pass over the operand with three real products per complex product (Role3M), the rest with
    the four-product role (2..4 columns) or the single-column kernel.  Against the oracle, on a size with several units per
    CTA and a ragged last tile; the launch count is pre-pass + tile pass + post-pass per group (one kernel for k = 1)."""
    import paper_2504_10096_b200 as b
    N = 2000
    R = gen.dense_R(N, 31, sigma=0.5)
    X = gen.block_X(N, k, 32)
    ref = orc.apply_tda(R, X)
    h = b.Bse(b.MODE_TDA, N, pack(R, 0))
    n0 = b.launch_count()
    Y = to_host(h.apply(to_dev(X)))
    launches = b.launch_count() - n0
    assert relerr(Y, ref) <= TOL_APPLY
    left, expect = k, 0
    while left > 0:                            # the launcher's greedy rule (bse_apply.cu, group_width)
        w = min(left, 8) if left > 4 else left
        expect += 1 if w == 1 else 3
        left -= w
    assert launches == expect


@pytest.mark.parametrize("k", [2, 3, 4, 6, 8])
def test_tile_roles_every_store_agree_with_oracle(orc, k, monkeypatch):
    """The tile kernels' roles (four-product 2..4 columns, three-product 5..8) against the oracle: TDA (HERM pass), full mode
    (HERM + SYMC passes, both signs), complex128 and complex64 stores, a ragged size with several units per CTA; and single
    columns through the tensor-core kernels (BSE_APPLY_K1=0 at handle creation)."""
    import paper_2504_10096_b200 as b
    N = 2000
    R, C = gen.dense_R(N, 31, sigma=1.0), gen.dense_C(N, 31)
    X = gen.block_X(N, k, 33)
    refs = {b.STORE_C128: (R, C), b.STORE_C64: (orc.round_c64(R), orc.round_c64(C))}
    for storage, (Rs, Cs) in refs.items():
        rt = b.bse_pack_from_dense(to_dev(R), N, 0, storage=storage)
        ct = b.bse_pack_from_dense(to_dev(C), N, 1, storage=storage)
        ht, hf = b.Bse(b.MODE_TDA, N, rt, storage=storage), b.Bse(b.MODE_FULL, N, rt, ct, storage=storage)
        assert relerr(to_host(ht.apply(to_dev(X))), orc.apply_tda(Rs, X)) <= TOL_APPLY, storage
        for sign in (+1, -1):
            assert relerr(to_host(hf.apply_half(to_dev(X), sign)), orc.apply_half(Rs, Cs, X, sign)) <= TOL_APPLY
        if k == 2:
            monkeypatch.setenv("BSE_APPLY_K1", "0")
            h1, hf1 = b.Bse(b.MODE_TDA, N, rt, storage=storage), b.Bse(b.MODE_FULL, N, rt, ct, storage=storage)
            monkeypatch.delenv("BSE_APPLY_K1")
            assert relerr(to_host(h1.apply(to_dev(X[:, :1]))), orc.apply_tda(Rs, X[:, :1])) <= TOL_APPLY
            assert relerr(to_host(hf1.apply_half(to_dev(X[:, :1]), -1)), orc.apply_half(Rs, Cs, X[:, :1], -1)) <= TOL_APPLY


@pytest.mark.parametrize("kind", ["real_x", "imag_x", "real_T", "imag_T", "one_column_dominant"])
def test_three_product_form_special_operands(orc, kind):
    """The 5..8-column kernel forms re/im from Q1 = Tr xr, Q2 = Ti xi, Q3 = (Tr + Ti)(xr +- xi): operands for which one
    of the three products vanishes or dominates must still meet the normwise tolerance (a wrong sign in one row of the
    combination table shows up as an O(1) error here), for both passes (HERM through R, SYMC through C) and both
    half-apply signs."""
    import paper_2504_10096_b200 as b
    N, k = 330, 8
    R, C = _herm(N, 61), _sym(N, 62)
    x = gen.block_X(N, k, 63)
    if kind == "real_x":
        x = x.real + 0j
    elif kind == "imag_x":
        x = 1j * x.imag
    elif kind == "real_T":
        R, C = R.real + 0j, C.real + 0j
    elif kind == "imag_T":
        R = 1j * np.tril(R.imag, -1); R = R + R.conj().T + np.diag(np.arange(1.0, N + 1))
        C = 1j * C.imag
    else:
        x[:, 3] *= 1e8
    h = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
    for sign in (+1, -1):
        Y, ref = to_host(h.apply_half(to_dev(x), sign)), orc.apply_half(R, C, x, sign)
        assert relerr(Y, ref) <= TOL_APPLY
        for c in range(k):                     # column by column: a large column must not drown the others
            assert relerr(Y[:, c], ref[:, c]) <= TOL_APPLY
    ht = b.Bse(b.MODE_TDA, N, pack(R, 0))
    assert relerr(to_host(ht.apply(to_dev(x))), orc.apply_tda(R, x)) <= TOL_APPLY


@pytest.mark.parametrize("k", [4, 8])
def test_repeated_launches_stay_within_rounding_of_each_other(k):
    """Timing-dependent faults (the round-1 shared-memory WAR hazard corrupted about one 8-row group per launch) show up
    as an entry that differs from the other launches by far more than the summation-order noise of the RED flushes:
    200 launches of the role-split (k = 4) and three-product (k = 8) kernels and of the real-form kernel, many units per
    CTA, every entry compared with the first launch."""
    import torch
    import paper_2504_10096_b200 as b
    N = 8192
    rt, ct = b.bse_fill_synthetic(N, 0, 1, 1.0, 16), b.bse_fill_synthetic(N, 1, 1, 0.0, 16)
    X = torch.randn(k, N, dtype=torch.complex128, device="cuda", generator=torch.Generator("cuda").manual_seed(5))
    ht = b.Bse(b.MODE_TDA, N, rt)
    ref = ht.apply(X).clone()
    scale = float(ref.abs().max())
    worst = max(float((ht.apply(X) - ref).abs().max()) for _ in range(200))
    assert worst <= 1e-13 * scale
    del ht
    b.bse_to_real_form(rt, ct, N)
    hr = b.Bse(b.MODE_FULL, N, rt, ct, storage=b.STORE_REAL_FORM)
    ref = hr.apply_half(X, -1).clone()
    worst = max(float((hr.apply_half(X, -1) - ref).abs().max()) for _ in range(200))
    assert worst <= 1e-13 * float(ref.abs().max())


def test_apply_is_capturable_in_a_cuda_graph(orc):
    """bse_apply / bse_apply_half only enqueue work (a memset and kernel launches) on the handle's stream, so a
    launch-bound loop of small products can be captured once and replayed: the graph is captured on the stream the
    handle was created on, replayed with new contents of X, and must reproduce the oracle."""
    import torch
    import paper_2504_10096_b200 as b
    N, k = 1024, 4
    R, C = gen.dense_R(N, 1, sigma=1.0), gen.dense_C(N, 1)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        ht = b.Bse(b.MODE_TDA, N, pack(R, 0))
        hf = b.Bse(b.MODE_FULL, N, pack(R, 0), pack(C, 1))
        X = torch.zeros((k, N), dtype=torch.complex128, device="cuda")
        Y = torch.empty_like(X); Z = torch.empty_like(X); W = torch.empty_like(X)
        ht.apply(X, Y); hf.apply_half(X, -1, Z)             # warm-up outside the capture (one-time attribute setup)
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            ht.apply(X, Y)                                   # Y = R X
            hf.apply_half(Y, -1, Z)                          # Z = M(Y)
            ht.apply(Z, W)                                   # W = R Z
    for seed in (3, 4):
        x = gen.block_X(N, k, seed)
        X.copy_(to_dev(x))
        g.replay()
        torch.cuda.synchronize()
        y = orc.apply_tda(R, x); z = orc.apply_half(R, C, y, -1); w = orc.apply_tda(R, z)
        assert relerr(to_host(Y), y) <= TOL_APPLY and relerr(to_host(Z), z) <= 3 * TOL_APPLY
        assert relerr(to_host(W), w) <= 10 * TOL_APPLY       # three products deep: errors accumulate
