"""GPU tier, second batch of round 2: the code paths added after the first batch -- 8-byte records of one-pixel
tiles through every entry point, tiles of 4 / 2 pixels held whole by one lane, the staged / re-walked compaction,
the degenerate sigma == 0 rows with a negative threshold, batches whose tLISI kernels are chained by programmatic
dependent launches.  Same rules as test_parity_gpu.py: through the C ABI, against the CPU fp64 oracle on the same
seeded buffers, tolerances of DESIGN.md section 3.
"""
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2509_21754_b200 as fitrig
import synth
from tests import util
from tests.test_parity_gpu import check_against_oracle, gpu_run, oracle_delta_at, oracle_run

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _stack(H, W, L=8, seed_cfg="tiny"):
    cfg = synth.scaled(synth.CONFIGS[seed_cfg], H, W, L=L)
    return synth.make_stack(cfg, device=DEV)[0]


# ------------------------------------------------------------------------------------------
# tiles of ONE pixel keep {Delta, r} records of 8 bytes: every reader of the map records must agree
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("H,W,use_stream", [(96, 128, False), (70, 100, False), (96, 128, True), (65, 36, True)])
def test_pixel_tiles_whole_path(H, W, use_stream):
    st = _stack(H, W)
    taus = (4.0, 6.0)
    g = gpu_run(st, taus=taus, tile=1, capacity=1 << 18, use_stream=use_stream)
    ref = oracle_run(st, tile=1, tau=5.0)
    check_against_oracle(st, g, ref, taus, 1, small_tiles=True)
    sd, md, sr, ax, ay = g["raw"]
    assert np.array_equal(sd, md)  # one pixel: sum Delta == max Delta, and the position is the pixel itself
    U, Ty, Tx = g["dims"]
    assert np.array_equal(ax, np.broadcast_to(np.arange(Tx), (U, Ty, Tx))) and np.array_equal(ay, np.broadcast_to(np.arange(Ty)[:, None], (U, Ty, Tx)))


def test_pixel_tiles_unaligned_base_take_the_generic_kernel_with_the_same_records():
    H, W = 64, 96
    big = _stack(H, W + 4)
    flat = torch.empty(big.shape[0] * H * W + 1, dtype=torch.float32, device=DEV)
    view = flat[1:].view(big.shape[0], H, W)  # base pointer 4 bytes off a 16-byte boundary
    view.copy_(big[:, :, :W])
    a = gpu_run(view, taus=(5.0,), tile=1, capacity=1 << 18)
    b = gpu_run(view.clone(), taus=(5.0,), tile=1, capacity=1 << 18)  # aligned copy: the fused kernel
    np.testing.assert_allclose(a["q"], b["q"], rtol=2e-6, atol=1e-30)
    assert a["cands"][5.0][1] == b["cands"][5.0][1]
    ref = oracle_run(view, tile=1, tau=5.0)
    check_against_oracle(view, a, ref, (5.0,), 1, small_tiles=True)


def test_pixel_tiles_push_and_row_shards():
    H, W, L, tau = 64, 96, 7, 5.0
    st = _stack(H, W, L)
    ref = oracle.run_realtime(st.cpu().numpy(), tile=1, tau=tau)
    with fitrig.Context(H, W, 3, tile=1) as ctx:
        units = {}
        for s in list(st) + [None]:
            u, c, n = ctx.push(s, tau, None, 1 << 18)
            if u >= 0:
                units[u] = (c.copy(), n, ctx.get_map(0)[0])
    assert sorted(units) == list(range(L - 2))
    for n_, (c, cnt, q) in units.items():
        eS, eM, eR = util.fp32_slack(st[n_:n_ + 3].cpu().numpy(), 1)
        r = ref[n_]
        slack = (eS * r.res.maxD * r.res.sumR + r.res.sumD * eM * r.res.sumR + r.res.sumD * r.res.maxD * eR)[0] / r.res.M ** 2
        util.assert_map_close(q, r.res.q[0], slack=slack)
    # two row shards of the same image against the whole-image context (bit-identical rows)
    whole = gpu_run(st, taus=(tau,), tile=1, capacity=1 << 18)
    from paper_2509_21754_b200 import shard
    rows = shard.row_shards(H, 1, 2)
    ctxs, vecs = [], []
    try:
        for (r0, r1) in rows:
            ctx = fitrig.Context(r1 - r0, W, L, tile=1, row_offset=r0)
            ctxs.append(ctx)
            ctx.tlisi(st[:, r0:r1].contiguous())
            v = torch.empty(2 + 2 * (L - 2), dtype=torch.float64, device=DEV)
            ctx.shard_export(v)
            vecs.append(v)
        allv = torch.stack(vecs).contiguous()
        for (r0, r1), ctx in zip(rows, ctxs):
            ctx.shard_import(allv, 2)
            assert np.array_equal(ctx.get_map(0), whole["q"][:, r0:r1])
    finally:
        for ctx in ctxs:
            ctx.close()


def test_windows_at_stride_one_are_built_from_pixel_records():
    """tile 4, stride 1: cells of one pixel (8-byte records) merged into 4 x 4 windows (R27)."""
    H, W = 40, 52
    st = _stack(H, W)
    g = gpu_run(st, taus=(4.0,), tile=4, stride=1, capacity=1 << 18)
    ref = oracle.run(st.cpu().numpy(), tile=4, tau=4.0, stride=1)
    util.assert_map_close(g["q"], ref.res.q, g["tlisi"], ref.res.tlisi)
    assert g["cands"][4.0][1] == ref.cands.n_found or abs(g["cands"][4.0][1] - ref.cands.n_found) <= 2


# ------------------------------------------------------------------------------------------
# compaction: warps with more candidates than they can keep from the counting pass walk their range again;
# sigma == 0 rows with a negative threshold select every tile (z == 0 > tau, R4 + R6)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("tile,tau", [(4, -0.5), (2, -0.3), (8, -0.5), (32, -3.0)])
def test_low_thresholds_many_candidates_per_warp(tile, tau):
    H, W = 256, 256
    st = _stack(H, W)
    g = gpu_run(st, taus=(tau,), tile=tile, capacity=1 << 20)
    ref = oracle_run(st, tile=tile, tau=tau)
    U, Ty, Tx = g["dims"]
    c, n = g["cands"][tau]
    assert n == len(c) and n > 0
    if tile <= 4:
        assert n > 0.5 * U * Ty * Tx  # more than half of every warp's 128 entries: no warp can keep them all
    lst = [(int(k["x"]), int(k["y"]), int(k["snapshot"]), float(k["score"]), (int(k["y"]) // tile) * Tx + int(k["x"]) // tile,
            int(k["snapshot"])) for k in c]
    util.compare_candidates(lst, ref.z, ref.mu, ref.sigma, tau, Tx, Ty * Tx)


def test_negative_threshold_on_constant_rows_selects_every_tile():
    L, H, W, tile = 5, 64, 96, 32
    one = synth.gaussian_noise_stack(L, tile, tile, seed=11, device=DEV)
    st = one.repeat(1, H // tile, W // tile).contiguous()  # identical tiles: q is constant over every unit, sigma == 0
    with fitrig.Context(H, W, L, tile=tile) as ctx:
        ctx.tlisi(st)
        M, mu, sd = ctx.get_stats()
        assert np.all(sd == 0.0)
        c, n = ctx.detect(-1.0)
        U, Ty, Tx = ctx.map_dims()
        assert n == U * Ty * Tx and np.all(c["score"] == 0.0)
        order = [(int(k["snapshot"]), int(k["y"]) // tile, int(k["x"]) // tile) for k in c]
        assert order == sorted(order) and len(set(order)) == n
        assert ctx.detect(0.0)[1] == 0  # strict: z == 0 is not > 0
    ref = oracle.run(st.cpu().numpy(), tile=tile, tau=-1.0)
    assert ref.cands.n_found == n


# ------------------------------------------------------------------------------------------
# tiles of 4 and 2 pixels (a lane holds whole tiles): every position of a maximum inside a tile, ties included
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("tile", [4, 2])
def test_small_tiles_first_maximum_in_row_major_order(tile):
    L, H, W = 3, 64, 64
    st = torch.zeros((L, H, W), dtype=torch.float32, device=DEV)  # Delta = 0 everywhere ...
    rng = np.random.default_rng(3)
    want = {}
    for ty in range(H // tile):
        for tx in range(W // tile):
            k = int(rng.integers(0, tile * tile))
            y, x = ty * tile + k // tile, tx * tile + k % tile
            st[2, y, x] = 3.0  # ... except here: D_0 = 0, D_1 = 3, Delta = 3
            if rng.random() < 0.5 and k + 1 < tile * tile:  # a second, equal maximum later in row-major order
                k2 = int(rng.integers(k + 1, tile * tile))
                st[2, ty * tile + k2 // tile, tx * tile + k2 % tile] = 3.0
            want[(ty, tx)] = (x, y)
    with fitrig.Context(H, W, L, tile=tile) as ctx:
        ctx.tlisi(st)
        sd, md, sr, ax, ay = ctx.get_raw()
    assert np.all(md == 3.0)
    for (ty, tx), (x, y) in want.items():
        assert (int(ax[0, ty, tx]), int(ay[0, ty, tx])) == (x, y)


# ------------------------------------------------------------------------------------------
# rows that do not start on 16-byte boundaries (W % 4 != 0): cells of 32 pixels ride the fused kernel through a
# tensor map of "super rows" (k = 2 or 4 image rows); shapes whose total row count is not a multiple of k, and
# unaligned base pointers, stay on the generic kernel
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("H,W,L,tile,use_stream", [(100, 250, 8, 32, False), (96, 251, 8, 32, False), (130, 253, 8, 32, False),
                                                   (64, 66, 6, 32, False), (70, 255, 8, 64, False), (160, 250, 8, 32, True),
                                                   (33, 251, 5, 32, False), (257, 1027, 4, 32, False),
                                                   (100, 250, 8, 16, False), (96, 251, 8, 16, False), (130, 253, 8, 8, False),
                                                   (100, 250, 8, 8, True), (70, 254, 6, 4, False), (66, 251, 8, 4, False),
                                                   (64, 250, 6, 2, False), (40, 253, 8, 2, False), (48, 250, 6, 1, False),
                                                   (40, 251, 8, 1, False), (70, 255, 8, 48, False), (64, 250, 6, 12, False)])
def test_rows_off_16_byte_boundaries(H, W, L, tile, use_stream):
    st = _stack(H, W, L)
    taus = (2.0, 3.0)
    kw = dict(strip_rows=64) if use_stream else {}
    g = gpu_run(st, taus=taus, tile=tile, use_stream=use_stream, capacity=1 << 18, **kw)
    ref = oracle_run(st, tile=tile, tau=3.0)
    check_against_oracle(st, g, ref, taus, tile, small_tiles=util.needs_slack(H, W, tile))


def test_rows_off_16_byte_boundaries_fused_and_generic_kernels_agree(monkeypatch):
    H, W, L = 200, 254, 8
    st = _stack(H, W, L)
    a = gpu_run(st, taus=(3.0,))
    monkeypatch.setenv("FITRIG_NO_UNALIGNED_FUSED", "1")
    b = gpu_run(st, taus=(3.0,))
    monkeypatch.delenv("FITRIG_NO_UNALIGNED_FUSED")
    np.testing.assert_allclose(a["q"], b["q"], rtol=2e-6, atol=1e-30)  # (other summation order)
    assert a["M"] == b["M"]
    assert a["cands"][3.0][1] == b["cands"][3.0][1]
    assert np.array_equal(a["raw"][3], b["raw"][3]) and np.array_equal(a["raw"][4], b["raw"][4])  # arg-max pixels


def test_driver_refusing_the_super_row_tensor_map_falls_back_to_the_generic_kernel(monkeypatch):
    """The super-row tensor map has overlapping rows; if a driver refuses to encode it, the call must still succeed on
    the generic kernel (same result as FITRIG_NO_UNALIGNED_FUSED), not return FITRIG_ERR_CUDA."""
    H, W, L = 200, 254, 8
    st = _stack(H, W, L)
    monkeypatch.setenv("FITRIG_NO_UNALIGNED_FUSED", "1")
    b = gpu_run(st, taus=(3.0,))
    monkeypatch.delenv("FITRIG_NO_UNALIGNED_FUSED")
    monkeypatch.setenv("FITRIG_TEST_FAIL_UNALIGNED_ENCODE", "1")
    a = gpu_run(st, taus=(3.0,))
    s = gpu_run(st, taus=(3.0,), use_stream=True, strip_rows=64)
    monkeypatch.delenv("FITRIG_TEST_FAIL_UNALIGNED_ENCODE")
    for g in (a, s):
        assert np.array_equal(g["q"], b["q"]) and g["M"] == b["M"] and np.array_equal(g["cands"][3.0][0], b["cands"][3.0][0])
    ref = oracle_run(st, tile=32, tau=3.0)
    check_against_oracle(st, a, ref, (3.0,), 32)


def test_rows_off_16_byte_boundaries_push():
    H, W, L, tau = 96, 250, 7, 3.0
    st = _stack(H, W, L)
    ref = oracle.run_realtime(st.cpu().numpy(), tile=32, tau=tau)
    with fitrig.Context(H, W, 3) as ctx:
        for i, s in enumerate(list(st) + [None]):
            u, c, n = ctx.push(s, tau)
            if u >= 0:
                util.assert_map_close(ctx.get_map(0)[0], ref[u].res.q[0])
                assert n == ref[u].cands.n_found or abs(n - ref[u].cands.n_found) <= 1


@pytest.mark.parametrize("W,off", [(252, 1), (252, 2), (250, 1), (250, 3), (251, 2)])
def test_unaligned_base_pointers_with_any_width(W, off):
    """The stack starts `off` floats past a 16-byte boundary: the super rows start at the boundary below it."""
    H, L, tau = 100, 8, 3.0
    st = _stack(H, W, L)
    flat = torch.empty(L * H * W + off, dtype=torch.float32, device=DEV)
    view = flat[off:].view(L, H, W)
    view.copy_(st)
    assert view.data_ptr() % 16 == 4 * off
    g = gpu_run(view, taus=(tau,))
    ref = oracle_run(view, tile=32, tau=tau)
    check_against_oracle(view, g, ref, (tau,), 32)
    a = gpu_run(st, taus=(tau,))  # the same pixels from an aligned allocation
    if os.environ.get("FITRIG_NO_UNALIGNED_FUSED") or os.environ.get("FITRIG_FORCE_GENERIC"):
        np.testing.assert_allclose(a["q"], g["q"], rtol=2e-6, atol=1e-30)  # (the generic kernel sums in another order)
    else:
        # the plain fused kernel (aligned, W % 4 == 0) and its super-row variant do the same arithmetic in the same order
        assert np.array_equal(a["q"], g["q"])


# ------------------------------------------------------------------------------------------
# fitrig_choose_accumulate: the stopping rule of snapshot accumulation (reading R30)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,H,W", [(24, 96, 128), (17, 33, 50), (64, 40, 64)])
def test_choose_accumulate_matches_oracle(L, H, W):
    base = synth.gaussian_noise_stack(L, H, W, seed=21, device=DEV)
    drift = torch.arange(L, dtype=torch.float32, device=DEV)[:, None, None] * 0.02
    st = (5.0 + 0.05 * base + drift).contiguous()  # a slow drift under a little noise: contrast grows with g
    snaps = st.cpu().numpy()
    levels = []
    g = 1
    while g <= 32 and L // g >= 3:
        levels.append((g, oracle.accumulation_contrast(snaps, g)))
        g *= 2
    # contrast of every admissible level (an unreachable eps looks at all of them)
    g_dev, d_dev = fitrig.choose_accumulate(st, 1e30)
    assert g_dev == levels[-1][0] and len(d_dev) == len(levels)
    # fp32 accumulation of g <= 32 snapshots and fp32 differences against fp64: (g + 2) 2^-24 relative on every term
    for (g_, d_ref), d in zip(levels, d_dev):
        assert abs(d - d_ref) <= 4e-6 * d_ref, (g_, d, d_ref)
    # thresholds between the levels: the first level that reaches eps; at the oracle's own value of a level: that level
    # (unless the two contrasts differ in the last digits, which the band above allows)
    for i in range(1, len(levels)):
        lo, hi = levels[i - 1][1], levels[i][1]
        if hi > lo * 1.001:
            eps = 0.5 * (lo + hi)
            assert fitrig.choose_accumulate(st, eps)[0] == oracle.choose_accumulate(snaps, eps)[0] == levels[i][0]
    assert fitrig.choose_accumulate(st, 0.0)[0] == 1
    assert fitrig.choose_accumulate(st, 1e30, g_max=2)[0] == min(2, levels[-1][0])


def test_choose_accumulate_degenerate_inputs():
    st = torch.full((12, 16, 16), 2.5, device=DEV)
    g, d = fitrig.choose_accumulate(st, 1e-6)
    assert g == 4 and d == [0.0, 0.0, 0.0]  # identical snapshots: no contrast at any level; 12 // 8 < 3
    assert fitrig.choose_accumulate(torch.zeros((6, 8, 8), device=DEV), 0.5) == (2, [0.0, 0.0])
    with pytest.raises(fitrig.FitrigError):
        fitrig.choose_accumulate(st[:2].contiguous(), 0.1)
    with pytest.raises(fitrig.FitrigError):
        fitrig.choose_accumulate(st, float("nan"))
