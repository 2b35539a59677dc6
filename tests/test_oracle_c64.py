"""Pins for the oracle's single-precision operand (oracle.round_c64).
Nothing here touches the CUDA library."""
import numpy as np

import bse_inputs as gen


def _r(orc, x):
    return orc.round_c64(np.array([complex(x, 0.0)]))[0].real


def test_hand_computed_neighbours_of_one(orc):
    # binary32 spacing above 1 is 2^-23, below 1 it is 2^-24
    u = 2.0 ** -24
    assert _r(orc, 1.0 + u) == 1.0                            # tie -> even significand
    assert _r(orc, 1.0 + 3 * u) == 1.0 + 4 * u                # tie between odd 1+2u and even 1+4u
    assert _r(orc, 1.0 + 1.01 * u) == 1.0 + 2 * u             # just above the tie
    assert _r(orc, 1.0 + 0.99 * u) == 1.0
    assert _r(orc, 1.0 - u) == 1.0 - u                        # representable below 1
    assert _r(orc, 1.0 - u / 2) == 1.0                        # tie between 1 - u (odd) and 1 (even)
    assert _r(orc, -(1.0 + 3 * u)) == -(1.0 + 4 * u)          # sign symmetric
    assert _r(orc, 0.1) == float.fromhex("0x1.99999ap-4")      # the textbook binary32 image of 0.1
    assert _r(orc, 16777217.0) == 16777216.0                  # 2^24 + 1 is a tie -> even


def test_range_edges(orc):
    big = (2.0 - 2.0 ** -23) * 2.0 ** 127                     # largest binary32
    assert _r(orc, big) == big
    assert _r(orc, big * (1 + 2.0 ** -26)) == big
    assert np.isinf(_r(orc, 2.0 ** 128)) and _r(orc, -2.0 ** 128) == -np.inf
    assert np.isinf(_r(orc, (2.0 - 2.0 ** -24) * 2.0 ** 127))     # halfway to 2^128 rounds to even = overflow
    assert _r(orc, (2.0 - 2.0 ** -24 - 2.0 ** -40) * 2.0 ** 127) == big   # just below halfway
    assert _r(orc, 2.0 ** -149) == 2.0 ** -149                # smallest subnormal
    assert _r(orc, 2.0 ** -150) == 0.0                        # tie -> even (0)
    assert _r(orc, 1.5 * 2.0 ** -149) == 2.0 ** -148          # tie between 1 and 2 quanta -> even
    assert _r(orc, 2.0 ** -126 * (1 + 2.0 ** -24)) == 2.0 ** -126
    assert _r(orc, 0.0) == 0.0 and np.signbit(_r(orc, -0.0))


def test_matches_hardware_conversion_and_bounds(orc):
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.standard_normal(20000) * 10.0 ** rng.integers(-42, 38, 20000),
                        np.float32(rng.standard_normal(1000)).astype(np.float64) * (1 + 2.0 ** -24),   # exact ties
                        [0.0, -0.0, 1.0, -1.0, 2.0 ** -130, 3.4e38, -3.5e38]])
    z = x + 1j * x[::-1]
    with np.errstate(over="ignore"):
        hw = z.astype(np.complex64).astype(np.complex128)
    got = orc.round_c64(z)
    assert np.array_equal(got.view(np.float64), hw.view(np.float64))
    assert np.array_equal(orc.round_c64(got).view(np.float64), got.view(np.float64))          # idempotent
    normal = (np.abs(x) > 2.0 ** -126) & (np.abs(x) < 3.0e38)
    assert np.all(np.abs(got.real[normal] - x[normal]) <= 2.0 ** -24 * np.abs(x[normal]))


def test_structure_and_weyl_bound(orc):
    N = 96
    R = gen.dense_R(N, 3, sigma=1.0); C = gen.dense_C(N, 3)
    R32, C32 = orc.round_c64(R), orc.round_c64(C)
    assert np.array_equal(R32, R32.conj().T) and np.array_equal(C32, C32.T)     # rounding keeps both structures
    assert np.all(R32.imag.diagonal() == 0)
    dR = np.linalg.norm(R32 - R, 2)
    assert 0 < dR <= 2.0 ** -24 * np.linalg.norm(np.abs(R), 2) * 1.0000001
    # Weyl: |lambda_i(R + E) - lambda_i(R)| <= ||E||_2 -- "accuracy limited by the data, not the solver"
    assert np.max(np.abs(np.linalg.eigvalsh(R32) - np.linalg.eigvalsh(R))) <= dR
    # the apply of the rounded operator is the oracle apply of the rounded matrix (definition), and differs from the
    # unrounded one by at most ||E||_2 ||x||
    X = gen.block_X(N, 3, 8)
    Y, Y32 = orc.apply_tda(R, X), orc.apply_tda(R32, X)
    assert 0 < np.linalg.norm(Y32 - Y, 2) <= dR * np.linalg.norm(X, 2)
