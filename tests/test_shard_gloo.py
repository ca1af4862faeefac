"""N > 1 host logic on CPU: world_size-2 (and 3) `gloo` process groups.

The CUDA kernels cannot run here, so every rank stands in for its GPU with the ORACLE restricted to its own
row shard (tests may use the oracle); what is under test is the product's host side of the sharded path
(paper_2509_21754_b200/shard.py): the row split, the ONE all-gather of 2 + 2U doubles (plus the 3-double one of the
frequency branch), the candidate gather and the (unit, tile row, tile col) merge -- and that the exchange protocol of include/fitrig.h
(fitrig_shard_export / fitrig_shard_import) reproduces the whole-image result.  The merge arithmetic of
fitrig_shard_import is restated below in numpy from its header comment.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import synth
from paper_2509_21754_b200 import shard
from paper_2509_21754_b200.binding import CANDIDATE_DTYPE


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _export_vector(stack_rows, tile):
    """What fitrig_shard_export returns for a shard, from the oracle: M = 1 makes q the M-free product p.
    v = [largest pixel, tiles per unit, mean_p[U], M2_p[U]] (M2 = sum of squared deviations from the shard's mean)."""
    r = oracle.tlisi(stack_rows, tile=tile, M=1.0)
    U = r.U
    mx = max(float(s.max()) for s in stack_rows)
    p = r.q.reshape(U, -1)
    v = np.zeros(2 + 2 * U)
    v[0], v[1] = mx, r.Ty * r.Tx
    v[2:2 + U] = p.mean(axis=1)
    v[2 + U:] = ((p - p.mean(axis=1, keepdims=True)) ** 2).sum(axis=1)
    return v, r


def _chan(n, mean, m2, nb, mb, m2b):
    """Chan's merge of two (count, mean, M2) triples, as include/fitrig.h states it for fitrig_shard_import."""
    if nb <= 0:
        return n, mean, m2
    tot = n + nb
    d = mb - mean
    return tot, mean + d * (nb / tot), m2 + m2b + d * d * (n * nb / tot)


def _import(allv, U, C=1e-6):
    """fitrig_shard_import's merge, restated from include/fitrig.h: M = max over shards (floored at C), and per unit the
    shards' (n, mean, M2) merged in shard order; mu = mean / M^2, sigma = sqrt(M2 / n) / M^2."""
    M = max(float(np.float32(allv[:, 0].max())), C)
    mu, sd = np.zeros(U), np.zeros(U)
    for u in range(U):
        n, mean, m2 = 0.0, 0.0, 0.0
        for r in range(allv.shape[0]):
            n, mean, m2 = _chan(n, mean, m2, allv[r, 1], allv[r, 2 + u], allv[r, 2 + U + u])
        mu[u], sd[u] = mean / M ** 2, np.sqrt(m2 / n) / M ** 2
    return M, mu, sd


def _import_eta(allw):
    """fitrig_shard_import_eta's merge: the shards' (tiles, mean eta, M2 of eta) in shard order."""
    n, mean, m2 = 0.0, 0.0, 0.0
    for r in range(allw.shape[0]):
        n, mean, m2 = _chan(n, mean, m2, allw[r, 0], allw[r, 1], allw[r, 2])
    return mean, np.sqrt(m2 / n)


def _worker(rank, world, port, H, W, L, tile, tau, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        oracle.set_threads(1)
        cfg = synth.scaled(synth.CONFIGS["tiny"], H, W, L=L)
        st, _ = synth.make_stack(cfg, device="cpu")  # same seed on every rank: the same image
        full = [st[s].numpy() for s in range(L)]
        r0, r1 = shard.row_shards(H, tile, world)[rank]
        # what ShardedContext.stream hands to fitrig_stream: this rank's rows of the WHOLE host snapshots, as views
        # (one contiguous block per snapshot, r0 * W floats into it) -- no copy, and 1 / world of the bytes per rank
        rows = shard.shard_host_rows(full, r0, r1)
        assert all(v_.ctypes.data == x.ctypes.data + 4 * r0 * W and v_.flags["C_CONTIGUOUS"] and v_.shape == (r1 - r0, W)
                   for v_, x in zip(rows, full))
        nbytes = shard.all_gather_vectors(torch.tensor([sum(v_.nbytes for v_ in rows)], dtype=torch.int64)).reshape(-1)
        assert int(nbytes.sum()) == 4 * L * H * W and int(nbytes[rank]) == 4 * L * (r1 - r0) * W
        v, res = _export_vector(rows, tile)
        allv = shard.all_gather_vectors(torch.from_numpy(v)).numpy()  # the ONE exchange
        assert allv.shape == (world, 2 + 2 * (L - 2)) and np.array_equal(allv[rank], v)
        M, mu, sd = _import(allv, L - 2)
        q = res.q / M ** 2
        z = (q - mu[:, None, None]) / sd[:, None, None]
        sel = oracle.select(z, res.argmax, W, tau)
        local = np.zeros(len(sel.x), dtype=CANDIDATE_DTYPE)
        local["x"], local["y"], local["snapshot"], local["score"] = sel.x, sel.y + r0, sel.snapshot, sel.score
        merged = shard.merge_candidates(shard.gather_candidates(local))
        t_max = shard.max_over_ranks(10.0 + rank)
        assert t_max == 10.0 + world - 1
        # whole-image oracle, on every rank
        ref = oracle.run(full, tile=tile, tau=tau)
        assert abs(M - ref.res.M) <= 1e-12 * ref.res.M
        np.testing.assert_allclose(mu, ref.mu, rtol=1e-10)
        np.testing.assert_allclose(sd, ref.sigma, rtol=1e-8)
        ty0 = r0 // tile
        np.testing.assert_allclose(q, ref.res.q[:, ty0:ty0 + res.Ty], rtol=1e-12)
        assert len(merged) == ref.cands.n_found > 0
        assert np.array_equal(merged["x"], ref.cands.x) and np.array_equal(merged["y"], ref.cands.y)
        assert np.array_equal(merged["snapshot"], ref.cands.snapshot)
        np.testing.assert_allclose(merged["score"], ref.cands.score, rtol=1e-5)
        ret[rank] = len(merged)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,H,W,tile", [(2, 256, 256, 32), (2, 250, 252, 32), (3, 200, 96, 8)])
def test_row_sharded_image_over_gloo(world, H, W, tile):
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), H, W, 8, tile, 3.0, ret), nprocs=world, join=True)
    assert len(ret) == world and len(set(ret.values())) == 1


def _worker_frequency(rank, world, port, H, W, L, tile, tau, ret):
    """Frequency branch under row shards: the SECOND exchange (3 doubles: tiles, mean eta, M2 of eta), which can only
    follow the first because eta scales with 1 / M^2 (include/fitrig.h, fitrig_shard_export_eta / _import_eta)."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        oracle.set_threads(1)
        cfg = synth.scaled(synth.CONFIGS["imgfreq"], H, W, L=L)
        st, _ = synth.make_stack(cfg, device="cpu")
        full = [st[s].numpy() for s in range(L)]
        r0, r1 = shard.row_shards(H, tile, world)[rank]
        rows = [np.ascontiguousarray(x[r0:r1]) for x in full]
        v, res = _export_vector(rows, tile)
        allv = shard.all_gather_vectors(torch.from_numpy(v)).numpy()          # first exchange: M (and mu, sigma of q)
        M, _, _ = _import(allv, L - 2)
        eta, ks = oracle.spectrum(res.q / M ** 2)                              # this shard's tiles, global M
        w = np.array([eta.size, eta.mean(), ((eta - eta.mean()) ** 2).sum()])
        allw = shard.all_gather_vectors(torch.from_numpy(w)).numpy()          # second exchange: statistics of eta
        assert allw.shape == (world, 3) and np.array_equal(allw[rank], w)
        mean_eta, sd_eta = _import_eta(allw)
        z = (eta - mean_eta) / sd_eta
        sel = oracle.select_spectrum(z, ks, r1 - r0, W, tile, tau)
        local = np.zeros(len(sel.x), dtype=CANDIDATE_DTYPE)
        local["x"], local["y"], local["snapshot"], local["score"] = sel.x, sel.y + r0, sel.snapshot, sel.score
        # (one unit-free list: the frequency branch sorts by tile row, tile col; shards are in row order already)
        merged = np.concatenate(shard.gather_candidates(local))
        ref = oracle.run(full, tile=tile, tau=tau, branch=1)
        assert abs(mean_eta - ref.mu[0]) <= 1e-10 * abs(ref.mu[0]) and abs(sd_eta - ref.sigma[0]) <= 1e-8 * ref.sigma[0]
        ty0 = r0 // tile
        np.testing.assert_allclose(eta, ref.eta[ty0:ty0 + res.Ty], rtol=1e-9, atol=1e-12 * float(ref.eta.max()))
        assert len(merged) == ref.cands.n_found > 0
        assert np.array_equal(merged["x"], ref.cands.x) and np.array_equal(merged["y"], ref.cands.y)
        assert np.array_equal(merged["snapshot"], ref.cands.snapshot)
        np.testing.assert_allclose(merged["score"], ref.cands.score, rtol=1e-5)
        ret[rank] = len(merged)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,H,W,tile", [(2, 256, 256, 16), (3, 200, 96, 8)])
def test_row_sharded_frequency_branch_over_gloo(world, H, W, tile):
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker_frequency, args=(world, _free_port(), H, W, 12, tile, 2.0, ret), nprocs=world, join=True)
    assert len(ret) == world and len(set(ret.values())) == 1


def test_split_range_and_row_shards():
    for n in (0, 1, 7, 16, 1563):
        for world in (1, 2, 3, 8):
            parts = [shard.split_range(n, world, r) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
            assert max(hi - lo for lo, hi in parts) - min(hi - lo for lo, hi in parts) <= 1
    rows = shard.row_shards(50000, 32, 8)  # config 4 over 8 GPUs: 1563 tile rows, the last one 16 px
    assert rows[0][0] == 0 and rows[-1][1] == 50000
    assert all(a[1] == b[0] and a[0] % 32 == 0 for a, b in zip(rows, rows[1:]))
    assert {(r1 - r0 + 31) // 32 for r0, r1 in rows} <= {195, 196}
    assert shard.row_shards(40, 32, 4) == [(0, 0), (0, 32), (32, 32), (32, 40)]  # more ranks than tile rows
    with pytest.raises(ValueError):
        shard.split_range(4, 2, 2)


def test_shard_host_rows_are_views_that_tile_the_image():
    H, W, L, tile = 200, 96, 3, 8
    snaps = [np.arange(H * W, dtype=np.float32).reshape(H, W) + s for s in range(L)]
    tsnaps = [torch.from_numpy(x) for x in snaps]
    for world in (1, 2, 3, 7):
        seen = np.zeros(H, dtype=np.int64)
        for (r0, r1) in shard.row_shards(H, tile, world):
            views = shard.shard_host_rows(snaps, r0, r1)
            tviews = shard.shard_host_rows(tsnaps, r0, r1)
            for x, v_, t_ in zip(snaps, views, tviews):
                assert np.shares_memory(x, v_) and v_.ctypes.data == x.ctypes.data + 4 * r0 * W == t_.data_ptr()
                assert np.array_equal(v_, x[r0:r1]) and r0 % tile == 0
            seen[r0:r1] += 1
        assert np.all(seen == 1)  # every image row is streamed by exactly one rank
    with pytest.raises(ValueError):
        shard.shard_host_rows(snaps, 10, 10)
    with pytest.raises(ValueError):
        shard.shard_host_rows(snaps, 0, H + 1)
    with pytest.raises(ValueError):
        shard.shard_host_rows([x.T for x in snaps], 0, 8)  # column-major: rows are not contiguous blocks


def test_merge_candidates_orders_by_unit_then_shard():
    a = np.array([(5, 3, 0, 7.0), (9, 40, 2, 6.5)], dtype=CANDIDATE_DTYPE)      # shard 0: rows 0..63
    b = np.array([(1, 70, 0, 8.0), (2, 100, 1, 9.0), (3, 65, 2, 6.1)], dtype=CANDIDATE_DTYPE)  # shard 1
    m = shard.merge_candidates([a, b])
    assert [(int(r["snapshot"]), int(r["y"])) for r in m] == [(0, 3), (0, 70), (1, 100), (2, 40), (2, 65)]
    assert len(shard.merge_candidates([])) == 0
    assert len(shard.merge_candidates([a[:0], b[:0]])) == 0


def test_single_process_fallbacks_need_no_process_group():
    v = torch.arange(6, dtype=torch.float64)
    assert shard.all_gather_vectors(v).shape == (1, 6)
    assert shard.max_over_ranks(3.5) == 3.5
    c = np.array([(1, 2, 3, 4.0)], dtype=CANDIDATE_DTYPE)
    assert np.array_equal(shard.gather_candidates(c)[0], c)
