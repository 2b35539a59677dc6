"""bse_lanczos_quadrature_static -- the entry point that allocates nothing (scratch in a fixed device array of the library,
include/bse.h) -- against the existing bse_lanczos_quadrature, on two calls in a row.  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

import bse_inputs as gen
from gpu_util import pack

pytestmark = pytest.mark.gpu


def _dev_vec(d):
    import torch
    return torch.from_numpy(np.ascontiguousarray(d)).cuda()


def test_static_quadrature_matches_existing_path_twice_in_a_row():
    import paper_2504_10096_b200 as b
    N, steps = 2000, 40                                     # ragged last tile, several units per CTA
    R = gen.dense_R(N, 3, sigma=0.0)
    h = b.Bse(b.MODE_TDA, N, pack(R, 0))
    d1, d2 = gen.block_X(N, 2, 8).T.copy()
    ref1 = h.lanczos_quadrature(_dev_vec(d1), steps)
    ref2 = h.lanczos_quadrature(_dev_vec(d2), steps // 2)
    # two calls in a row share the scratch array: the second (another start vector, fewer steps) must not see the first's sums
    got1 = h.lanczos_quadrature_static(_dev_vec(d1), steps)
    got2 = h.lanczos_quadrature_static(_dev_vec(d2), steps // 2)
    tol = 1e-10 * 11                                        # tests/test_gpu_quadrature.py: 1e-10 ||R|| on the leading coefficients
    for (a, bt), (ar, br) in ((got1, ref1), (got2, ref2)):
        assert len(a) == len(ar) and len(bt) == len(br)
        assert np.max(np.abs(a - ar)) <= tol and np.max(np.abs(bt - br)) <= tol
    # and the quantity the coefficients are for
    om = np.linspace(-1.0, 11.0, 121)
    G, Gr = b.quadrature_resolvent(*got1, om, 0.1), b.quadrature_resolvent(*ref1, om, 0.1)
    assert np.max(np.abs(G - Gr)) <= 1e-10 * np.max(np.abs(Gr))


def test_static_quadrature_rejects_sizes_beyond_the_array():
    import ctypes
    import torch
    import paper_2504_10096_b200 as b
    small = b.Bse(b.MODE_TDA, 256, pack(gen.dense_R(256, 5), 0))
    d = _dev_vec(gen.block_X(256, 1, 9)[:, 0])
    with pytest.raises(b.BseError) as e:
        small.lanczos_quadrature_static(d, b.STATIC_QUADRATURE_MAX_STEPS + 1)
    assert e.value.status == 7 and b.lib().bse_status_string(7) == b"size exceeds the static scratch limit"
    Nbig = b.STATIC_QUADRATURE_MAX_N + 64
    big = b.Bse(b.MODE_TDA, Nbig, b.bse_fill_synthetic(Nbig, b.MATRIX_R, 1, 0.0, 16))
    dbig = torch.ones(Nbig, dtype=torch.complex128, device="cuda")
    with pytest.raises(b.BseError) as e:
        big.lanczos_quadrature_static(dbig, 4)
    assert e.value.status == 7
    a, bt = big.lanczos_quadrature(dbig, 4)                 # the allocating path takes any size
    assert len(a) == 4
    # the largest size the array takes
    Nmax = b.STATIC_QUADRATURE_MAX_N
    hm = b.Bse(b.MODE_TDA, Nmax, b.bse_fill_synthetic(Nmax, b.MATRIX_R, 1, 0.0, 16))
    dm = _dev_vec(gen.block_X(Nmax, 1, 10)[:, 0])
    a1, b1 = hm.lanczos_quadrature_static(dm, 6)
    a0, b0 = hm.lanczos_quadrature(dm, 6)
    assert np.max(np.abs(a1 - a0)) <= 1e-10 * 11 and np.max(np.abs(b1 - b0)) <= 1e-10 * 11 * np.max(b0)
