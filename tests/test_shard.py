"""Sharding of the tile stream (include/bse.h): the partition helper (host only), the all-reduce plumbing
on two gloo ranks (CPU), and -- on the GPU -- the sum of the shards' partial products against the oracle."""
import os

import numpy as np
import pytest

import bse_inputs as gen


@pytest.mark.parametrize("N", [64, 1000, 16384, 98304])
@pytest.mark.parametrize("G", [1, 2, 3, 8, 128])
def test_shard_layout_partitions_the_store(N, G):
    import paper_2504_10096_b200 as b
    for storage in (b.STORE_C128, b.STORE_C64):
        _, total, total_bytes = b.bse_layout(N, storage)
        nt = (N + 63) // 64
        prev_end, prev_tile, sizes = 0, 0, []
        for r in range(G):
            rb, re, ft, n, by = b.bse_shard_layout(N, G, r, storage)
            assert rb == prev_end and ft == prev_tile == rb * (rb + 1) // 2           # contiguous, in order
            assert n == re * (re + 1) // 2 - rb * (rb + 1) // 2 and by == n * (total_bytes // total)
            prev_end, prev_tile = re, ft + n
            sizes.append(n)
        assert prev_end == nt and sum(sizes) == total                                # every tile exactly once
        # balanced to within one tile row of the ideal share
        assert max(sizes) - total / G <= nt + 1


def _gloo_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import paper_2504_10096_b200 as b
    Y = torch.full((3, 10), complex(rank + 1, -(rank + 1)), dtype=torch.complex128)
    b.sum_partials(Y)
    rows = b.bse_shard_layout(1000, world, rank)[:2]
    q.put((rank, Y[0, 0].item(), rows))
    dist.destroy_process_group()


def test_sum_partials_on_two_gloo_ranks():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps: p.start()
    out = sorted(q.get(timeout=120) for _ in ps)
    for p in ps: p.join(60)
    assert all(p.exitcode == 0 for p in ps)
    assert out[0][1] == out[1][1] == complex(3, -3)                 # both ranks hold the sum
    assert out[0][2][0] == 0 and out[0][2][1] == out[1][2][0] and out[1][2][1] == 16     # the two slices tile the rows


# ------------------------------------------------- GPU: shards run one after another on one device -----------------

def _slices(tiles, N, G, storage):
    import paper_2504_10096_b200 as b
    per_tile = b.bse_layout(N, storage)[2] // b.bse_layout(N, storage)[1]
    out = []
    for r in range(G):
        rb, re, ft, n, by = b.bse_shard_layout(N, G, r, storage)
        out.append(((rb, re), tiles[ft * per_tile: ft * per_tile + max(by, 1)]))
    return out


@pytest.mark.gpu
@pytest.mark.parametrize("G", [2, 3, 8])
@pytest.mark.parametrize("k", [1, 4, 8])
def test_tda_partial_products_sum_to_the_oracle(orc, G, k):
    import torch
    import paper_2504_10096_b200 as b
    from gpu_util import pack, relerr, to_dev, to_host
    N = 1000
    R = gen.dense_R(1008, 41, sigma=0.5)[:N, :N]
    X = gen.block_X(N, k, 42)
    ref = orc.apply_tda(R, X)
    for storage in (b.STORE_C128, b.STORE_C64):
        tiles = b.bse_pack_from_dense(to_dev(R), N, 0, storage=storage)
        Y = torch.zeros((k, N), dtype=torch.complex128, device="cuda")
        for rows, sl in _slices(tiles, N, G, storage):
            Y += b.Bse(b.MODE_TDA, N, sl, storage=storage, rows=rows).apply(to_dev(X))
        want = ref if storage == b.STORE_C128 else orc.apply_tda(orc.round_c64(R), X)
        assert relerr(to_host(Y), want) <= 1e-12


@pytest.mark.gpu
@pytest.mark.parametrize("G", [2, 5])
def test_full_mode_partial_products_complex_and_real_form(orc, G):
    import torch
    import paper_2504_10096_b200 as b
    from gpu_util import pack, relerr, to_dev, to_host
    N, k = 520, 8
    R, C = gen.dense_R(528, 43, sigma=1.0)[:N, :N], gen.dense_C(N, 43)
    x = gen.block_X(N, k, 44)
    X2 = gen.block_X(2 * N, 3, 45)
    for real in (False, True):
        rt, ct = pack(R, 0), pack(C, 1)
        storage = b.STORE_C128
        if real:
            b.bse_to_real_form(rt, ct, N)
            storage = b.STORE_REAL_FORM
        hs = [b.Bse(b.MODE_FULL, N, sr, sc, storage=storage, rows=rows)
              for (rows, sr), (_, sc) in zip(_slices(rt, N, G, b.STORE_C128), _slices(ct, N, G, b.STORE_C128))]
        for sign in (+1, -1):
            Y = sum(h.apply_half(to_dev(x), sign) for h in hs)
            assert relerr(to_host(Y), orc.apply_half(R, C, x, sign)) <= 1e-12
        Y = sum(h.apply(to_dev(X2)) for h in hs)
        assert relerr(to_host(Y), orc.apply_full(R, C, X2)) <= 1e-12
        with pytest.raises(b.BseError):
            hs[0].solve(4, 4)                                  # a partial handle is apply-level only


@pytest.mark.gpu
def test_generated_slices_equal_slices_of_the_generated_store():
    import torch
    import paper_2504_10096_b200 as b
    N, G = 4096, 3
    for which, sigma in ((0, 0.5), (1, 0.0)):
        full = b.bse_fill_synthetic(N, which, 5, sigma, 16)
        for r in range(G):
            rb, re, ft, n, by = b.bse_shard_layout(N, G, r)
            sl = b.bse_fill_synthetic_shard(N, which, 5, sigma, 16, (rb, re))
            assert torch.equal(sl[:by], full[ft * 65536: ft * 65536 + by])


@pytest.mark.gpu
def test_sharded_bse_single_process_many_units(orc):
    """ShardedBse without a process group is the one-rank case (its slice is the whole store); sampled rows at a size
    where every CTA walks several units."""
    import paper_2504_10096_b200 as b
    from gpu_util import relerr, to_dev, to_host
    N, k = 8192, 8
    h = b.ShardedBse.synthetic(b.MODE_TDA, N, 1, 0.0, 16)
    X = gen.block_X(N, k, 12)
    rows = np.arange(0, N, 509)
    ref = orc.rows_times_block(gen.rows_R(N, 1, rows, 0.0, 16), X)
    assert relerr(to_host(h.apply(to_dev(X)))[rows], ref) <= 1e-12
    # three slices generated separately, many units each, summed
    import torch
    Y = torch.zeros((k, N), dtype=torch.complex128, device="cuda")
    for r in range(3):
        rb, re = b.bse_shard_layout(N, 3, r)[:2]
        sl = b.bse_fill_synthetic_shard(N, 0, 1, 0.0, 16, (rb, re))
        Y += b.Bse(b.MODE_TDA, N, sl, rows=(rb, re)).apply(to_dev(X))
    assert relerr(to_host(Y)[rows], ref) <= 1e-12


# ------------------------------------------------- GPU: the solver on a sharded operator, two host processes ----------
# Both ranks use cuda:0 and exchange through gloo (host-staged): their kernels are ordinary finite launches that never
# wait on one another -- only the HOSTS meet in collectives -- so sharing the device is safe; it is slow, not a hazard.

def _solver_worker(rank, world, port, q):
    try:
        import torch
        import torch.distributed as dist
        os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        torch.cuda.set_device(0)
        dist.init_process_group("gloo", rank=rank, world_size=world)
        import paper_2504_10096_b200 as b
        from gpu_util import pack, to_dev, to_host
        out = {}
        # TDA: apply, solve, quadrature on rank-local slices of the same packed store
        N, k, nev = 320, 4, 6
        R = gen.dense_R(N, 1, sigma=1.0)
        C = gen.dense_C(N, 1)
        X = gen.block_X(N, 8, 7)

        def sliced(tiles, storage=b.STORE_C128):
            rb, re, ft, n, by = b.bse_shard_layout(N, world, rank, storage)
            per = b.bse_layout(N, storage)[2] // b.bse_layout(N, storage)[1]
            return (rb, re), tiles[ft * per: ft * per + by]
        rows, sl = sliced(pack(R, 0))
        h = b.ShardedBse(b.MODE_TDA, N, sl, None, rows).install_comm()
        out["tda_apply"] = to_host(h.apply(to_dev(X)))
        res = h.solve(nev, k, tol=1e-9, seed=1)
        out["tda_omega"], out["tda_vec"], out["tda_info"] = res.omega, to_host(res.vectors), res.info
        a, bb = h.lanczos_quadrature(to_dev(X[:, 0]).reshape(-1), 10)
        out["tda_quad"] = (a, bb)
        out["tda_calls"] = list(h.comm_calls)
        # full mode, real-form slices
        rt, ct = pack(R, 0), pack(C, 1)
        b.bse_to_real_form(rt, ct, N)
        (rows, sr), (_, sc) = sliced(rt), sliced(ct)
        hf = b.ShardedBse(b.MODE_FULL, N, sr, sc, rows, storage=b.STORE_REAL_FORM).install_comm()
        out["full_half"] = to_host(hf.apply_half(to_dev(X), -1))
        resf = hf.solve(4, k, tol=1e-9, seed=1)
        out["full_omega"], out["full_vec"] = resf.omega, to_host(resf.vectors)
        af, bf = hf.lanczos_quadrature(to_dev(X[:, 1]).reshape(-1), 8)
        out["full_quad"] = (af, bf)
        dist.barrier()
        dist.destroy_process_group()
        q.put((rank, out))
    except Exception as e:                                      # report instead of hanging the parent
        import traceback
        q.put((rank, {"error": traceback.format_exc()}))


@pytest.mark.gpu
def test_solver_on_a_sharded_operator_two_ranks(orc):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29700 + os.getpid() % 2000
    ps = [ctx.Process(target=_solver_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps: p.start()
    got = dict(q.get(timeout=600) for _ in ps)
    for p in ps: p.join(120)
    for r in (0, 1):
        assert "error" not in got[r], got[r].get("error")
    N, nev = 320, 6
    R, C = gen.dense_R(N, 1, sigma=1.0), gen.dense_C(N, 1)
    X = gen.block_X(N, 8, 7)
    rel = lambda a, b_: np.linalg.norm(a - b_) / np.linalg.norm(b_)
    for r in (0, 1):
        o = got[r]
        assert rel(o["tda_apply"], orc.apply_tda(R, X)) <= 1e-12
        wj, _ = orc.jacobi_herm(R)
        assert np.max(np.abs(o["tda_omega"] - wj[:nev]) / np.abs(wj[:nev])) <= 1e-10
        V = o["tda_vec"]
        assert np.linalg.norm(V.conj().T @ V - np.eye(nev)) <= 1e-12
        assert np.max(np.linalg.norm(orc.apply_tda(R, V) - V * o["tda_omega"], axis=0)) <= 1e-8 * 12
        ao, bo = orc.lanczos_quadrature(R, X[:, 0], 10)
        assert np.max(np.abs(o["tda_quad"][0] - ao)) <= 1e-10 * 12 and np.max(np.abs(o["tda_quad"][1] - bo)) <= 1e-10 * 30
        assert rel(o["full_half"], orc.apply_half(R, C, X, -1)) <= 1e-12
        omd, _ = orc.bse_direct(R, C, want_vectors=False)
        assert np.max(np.abs(o["full_omega"] - omd[N:N + 4]) / omd[N:N + 4]) <= 1e-10
        Vf = o["full_vec"]
        rr = np.linalg.norm(orc.apply_full(R, C, Vf) - Vf * o["full_omega"], axis=0) / np.linalg.norm(Vf, axis=0)
        assert np.all(rr <= 1e-8 * 12)
        af, bf = orc.lanczos_quadrature_full(R, C, X[:, 1], 8)
        assert np.max(np.abs(o["full_quad"][0] - af)) <= 1e-10 * np.max(np.abs(af))
        assert o["tda_calls"][0] > 0 and o["tda_calls"][1] > 0
    # lock step: both ranks took the same path and hold bitwise identical results
    assert got[0]["tda_info"]["n_apply"] == got[1]["tda_info"]["n_apply"]
    assert got[0]["tda_info"]["n_restart"] == got[1]["tda_info"]["n_restart"]
    assert np.array_equal(got[0]["tda_omega"], got[1]["tda_omega"]) and np.array_equal(got[0]["tda_vec"], got[1]["tda_vec"])
    assert np.array_equal(got[0]["full_omega"], got[1]["full_omega"]) and np.array_equal(got[0]["full_vec"], got[1]["full_vec"])


@pytest.mark.gpu
def test_comm_hook_single_rank_counts_and_leaves_results_unchanged(orc):
    """One rank, no process group needed for the arithmetic: the hook is called after every product and every
    atomically accumulated quantity, and a one-rank sum / broadcast changes nothing."""
    import ctypes
    import paper_2504_10096_b200 as b
    from gpu_util import pack, to_dev, to_host
    N, k, nev = 320, 4, 6
    R = gen.dense_R(N, 1, sigma=1.0)
    h = b.Bse(b.MODE_TDA, N, pack(R, 0))
    ref = h.solve(nev, k, tol=1e-9, seed=1)
    calls = [0, 0]
    cb = ctypes.CFUNCTYPE(ctypes.c_int32, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_int64)(
        lambda user, op, ptr, n: (calls.__setitem__(op, calls[op] + 1), 0)[1])
    assert b.lib().bse_set_comm(h._h, ctypes.cast(cb, ctypes.c_void_p), None) == 0
    res = h.solve(nev, k, tol=1e-9, seed=1)
    assert np.max(np.abs(res.omega - ref.omega)) <= 1e-12 and res.info["n_apply"] == ref.info["n_apply"]
    assert calls[0] == res.info["n_apply"] and calls[1] >= 2 * res.info["n_apply"]
    # a failing hook aborts the call with an error status instead of continuing on partial data
    bad = ctypes.CFUNCTYPE(ctypes.c_int32, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_int64)(
        lambda user, op, ptr, n: 1)
    b.lib().bse_set_comm(h._h, ctypes.cast(bad, ctypes.c_void_p), None)
    with pytest.raises(b.BseError):
        h.apply(to_dev(gen.block_X(N, 2, 3)))
    b.lib().bse_set_comm(h._h, None, None)
    assert np.max(np.abs(h.solve(nev, k, tol=1e-9, seed=1).omega - ref.omega)) <= 1e-12


@pytest.mark.gpu
@pytest.mark.parametrize("L", [1, 2, 3, 5, 32])
def test_unit_length_and_slices_every_kernel(orc, L, monkeypatch):
    """The unit length L (tiles of one tile row a CTA accumulates before flushing Y_I) is chosen from the operand size;
    BSE_APPLY_UNIT forces it here so that small matrices exercise multi-tile units, partial last units and slice
    boundaries that are not multiples of L, for every apply kernel (k = 1 plain FMA, k = 4 four-product, k = 8
    three-product, real form) and for 1 and 3 slices."""
    import torch
    import paper_2504_10096_b200 as b
    from gpu_util import pack, relerr, to_dev, to_host
    monkeypatch.setenv("BSE_APPLY_UNIT", str(L))
    N = 1000
    R, C = gen.dense_R(1008, 51, sigma=1.0)[:N, :N], gen.dense_C(N, 51)
    rt, ct = pack(R, 0), pack(C, 1)
    X = gen.block_X(N, 8, 52)
    for G in (1, 3):
        for k in (1, 4, 8):
            Y = sum(b.Bse(b.MODE_TDA, N, sl, rows=rows).apply(to_dev(X[:, :k])) for rows, sl in _slices(rt, N, G, b.STORE_C128))
            assert relerr(to_host(Y), orc.apply_tda(R, X[:, :k])) <= 1e-12, (G, k)
    rs, cs = rt.clone(), ct.clone()
    b.bse_to_real_form(rs, cs, N)
    for G in (1, 3):
        hs = [b.Bse(b.MODE_FULL, N, sr, sc, storage=b.STORE_REAL_FORM, rows=rows)
              for (rows, sr), (_, sc) in zip(_slices(rs, N, G, b.STORE_C128), _slices(cs, N, G, b.STORE_C128))]
        for sign in (+1, -1):
            Y = sum(h.apply_half(to_dev(X), sign) for h in hs)
            assert relerr(to_host(Y), orc.apply_half(R, C, X, sign)) <= 1e-12, (G, sign)


# ------------------------------------------------- GPU: vectors partitioned by rows as well, two host processes
def _rowpart_worker(rank, world, port, q):
    try:
        import torch
        import torch.distributed as dist
        os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        torch.cuda.set_device(0)
        dist.init_process_group("gloo", rank=rank, world_size=world)
        import paper_2504_10096_b200 as b
        from gpu_util import pack, to_host
        out = {}
        N, k, nev = 448, 4, 6                                  # 7 tile rows: unequal tile slices; 224 vector rows per rank
        R = gen.dense_R(N, 3, sigma=1.0)
        C = gen.dense_C(N, 3)

        def sliced(tiles):
            rb, re, ft, n, by = b.bse_shard_layout(N, world, rank)
            return (rb, re), tiles[ft * 65536: ft * 65536 + by]
        rows, sl = sliced(pack(R, 0))
        h = b.ShardedBse(b.MODE_TDA, N, sl, None, rows).install_comm(row_partition=True)
        out["vec_rows"] = h.vec_rows
        res = h.solve(nev, k, tol=1e-9, seed=1)
        out["tda_omega"], out["tda_vec"], out["tda_info"] = res.omega, to_host(res.vectors), res.info
        out["tda_calls"] = list(h.comm_calls)
        (rows, sr), (_, sc) = sliced(pack(R, 0)), sliced(pack(C, 1))
        hf = b.ShardedBse(b.MODE_FULL, N, sr, sc, rows).install_comm(row_partition=True)
        resf = hf.solve(5, k, tol=1e-9, seed=2)
        out["full_omega"], out["full_vec"], out["full_info"] = resf.omega, to_host(resf.vectors), resf.info
        # what a row-partitioned handle does not take
        try:
            hf.solve(5, k, variant=b.VARIANT_GRUNING)
            out["gruning_refused"] = False
        except b.BseError as e:
            out["gruning_refused"] = e.status == 1
        dist.barrier()
        dist.destroy_process_group()
        q.put((rank, out))
    except Exception:
        import traceback
        q.put((rank, {"error": traceback.format_exc()}))


@pytest.mark.gpu
def test_solver_with_row_partitioned_vectors_two_ranks(orc):
    """bse_set_row_partition: each rank holds half of the rows of every basis vector and its own slice of the tile store; the
    eigenpairs (gathered to full length) are certified by the oracle on both ranks, and agree with the replicated-vector
    solve of one process to the solver's accuracy (the Gram sums are split differently, so not bitwise)."""
    import torch.multiprocessing as mp
    import paper_2504_10096_b200 as b
    from gpu_util import pack
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31700 + os.getpid() % 2000
    ps = [ctx.Process(target=_rowpart_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps: p.start()
    got = dict(q.get(timeout=600) for _ in ps)
    for p in ps: p.join(120)
    for r in (0, 1):
        assert "error" not in got[r], got[r].get("error")
    N, nev = 448, 6
    R, C = gen.dense_R(N, 3, sigma=1.0), gen.dense_C(N, 3)
    assert got[0]["vec_rows"] == (0, 224) and got[1]["vec_rows"] == (224, 448)
    wj, _ = orc.jacobi_herm(R)
    omd, _ = orc.bse_direct(R, C, want_vectors=False)
    for r in (0, 1):
        o = got[r]
        assert np.max(np.abs(o["tda_omega"] - wj[:nev]) / np.abs(wj[:nev])) <= 1e-10
        V = o["tda_vec"]
        assert V.shape == (N, nev)
        assert np.linalg.norm(V.conj().T @ V - np.eye(nev)) <= 1e-12
        assert np.max(np.linalg.norm(orc.apply_tda(R, V) - V * o["tda_omega"], axis=0)) <= 1e-8 * 12
        assert o["tda_info"]["basis_orth_err"] <= 1e-12
        assert np.max(np.abs(o["full_omega"] - omd[N:N + 5]) / omd[N:N + 5]) <= 1e-10
        Vf = o["full_vec"]
        assert Vf.shape == (2 * N, 5)
        rr = np.linalg.norm(orc.apply_full(R, C, Vf) - Vf * o["full_omega"], axis=0) / np.linalg.norm(Vf, axis=0)
        assert np.all(rr <= 1e-8 * 12)
        Sig = np.concatenate([np.ones(N), -np.ones(N)])
        assert np.max(np.abs(np.sum(Sig[:, None] * np.abs(Vf) ** 2, axis=0) - 1)) <= 1e-10
        assert o["full_info"]["basis_orth_err"] <= 1e-12
        assert o["gruning_refused"]
    # both ranks hold the same gathered result and took the same path
    assert np.array_equal(got[0]["tda_omega"], got[1]["tda_omega"]) and np.array_equal(got[0]["tda_vec"], got[1]["tda_vec"])
    assert np.array_equal(got[0]["full_vec"], got[1]["full_vec"])
    assert got[0]["tda_info"]["n_apply"] == got[1]["tda_info"]["n_apply"]
    # and agree with the replicated-vector solve of a single handle
    ref = b.Bse(b.MODE_TDA, N, pack(R, 0)).solve(nev, 4, tol=1e-9, seed=1)
    assert np.max(np.abs(ref.omega - got[0]["tda_omega"]) / np.abs(ref.omega)) <= 1e-10
