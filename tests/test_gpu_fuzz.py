"""Seeded random sweep over (N, k, mode, store, slices, leading dimensions): every apply entry point against the oracle.
Sizes are small (the oracle is a triple loop) but cover N < one tile, ragged last tiles, k across the kernel switch points
(1 | 2..4 | 5..8 | > 8) and the chunking of k > 8."""
import numpy as np
import pytest

import bse_inputs as gen
from gpu_util import relerr, to_dev, to_host

pytestmark = pytest.mark.gpu


def _case(rng):
    N = int(rng.choice([1, 2, 7, 63, 64, 65, 100, 129, 200, 257, 320]))
    k = int(rng.choice([1, 2, 3, 4, 5, 6, 7, 8, 9, 12, 13, 17]))
    mode = str(rng.choice(["tda", "full", "real"]))
    store = str(rng.choice(["c128", "c64"]))
    G = int(rng.choice([1, 1, 2, 3]))
    pad = int(rng.choice([0, 0, 5]))
    return N, k, mode, store, G, pad


@pytest.mark.parametrize("seed", range(48))
def test_random_configuration_matches_oracle(orc, seed):
    import torch
    import paper_2504_10096_b200 as b
    rng = np.random.default_rng(1000 + seed)
    N, k, mode, store, G, pad = _case(rng)
    Np = N if N % 16 == 0 else N + 16 - N % 16
    R = gen.dense_R(Np, 100 + seed, sigma=1.0)[:N, :N]
    C = gen.dense_C(N, 100 + seed)
    base = b.STORE_C128 if store == "c128" else b.STORE_C64
    rt = b.bse_pack_from_dense(to_dev(R), N, 0, storage=base)
    ct = b.bse_pack_from_dense(to_dev(C), N, 1, storage=base)
    if store == "c64":
        R, C = orc.round_c64(R), orc.round_c64(C)
    storage = base
    if mode == "real":
        b.bse_to_real_form(rt, ct, N, storage=base)
        storage = b.STORE_REAL_FORM if base == b.STORE_C128 else b.STORE_REAL_FORM_C64
        if store == "c64":                                   # the operator the rounded planes define (include/bse.h)
            S32, D32 = orc.round_c64(R + C), orc.round_c64(R - C)
            R, C = (S32 + D32) / 2, (S32 - D32) / 2
    nt = (N + 63) // 64
    G = min(G, nt)
    per = b.bse_layout(N, base)[2] // b.bse_layout(N, base)[1]
    handles = []
    for r in range(G):
        rb, re, ft, n, by = b.bse_shard_layout(N, G, r, base)
        if n == 0:
            continue
        sr, sc = rt[ft * per: ft * per + by], ct[ft * per: ft * per + by]
        rows = None if G == 1 else (rb, re)
        if mode == "tda":
            handles.append(b.Bse(b.MODE_TDA, N, sr, storage=storage, rows=rows))
        else:
            handles.append(b.Bse(b.MODE_FULL, N, sr, sc, storage=storage, rows=rows))
    n_op = N if mode == "tda" else 2 * N
    X = gen.block_X(n_op, k, 500 + seed)
    ld = n_op + pad

    def call(fn_name, Xb, rows_out, *extra):
        Xd = torch.full((k, Xb.shape[0] + pad), 9.0 - 3j, dtype=torch.complex128, device="cuda")
        Xd[:, :Xb.shape[0]] = to_dev(Xb)
        tot = None
        for h in handles:
            Yd = torch.full((k, rows_out + pad), -1.0 + 2j, dtype=torch.complex128, device="cuda")
            fn = getattr(b.lib(), fn_name)
            st = fn(h._h, *extra, Xd.data_ptr(), Xb.shape[0] + pad, Yd.data_ptr(), rows_out + pad, k)
            assert st == 0, (fn_name, st)
            assert bool(torch.all(Yd[:, rows_out:] == (-1.0 + 2j)))      # padding rows untouched
            tot = Yd[:, :rows_out].clone() if tot is None else tot + Yd[:, :rows_out]
        return to_host(tot)

    what = (N, k, mode, store, G, pad)
    if mode == "tda":
        assert relerr(call("bse_apply", X, N), orc.apply_tda(R, X)) <= 1e-12, what
    else:
        assert relerr(call("bse_apply", X, 2 * N), orc.apply_full(R, C, X)) <= 1e-12, what
        x = X[:N]
        for sign in (+1, -1):
            assert relerr(call("bse_apply_half", x, N, sign), orc.apply_half(R, C, x, sign)) <= 1e-12, (what, sign)
