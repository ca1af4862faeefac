"""GPU tier: element-by-element parity of the CUDA path (through the C ABI) against the CPU fp64
oracle on the same seeded inputs.  Tolerances:

  * q = 1 - tLISI:  |q_gpu - q_ref| <= 1e-4 * |q_ref| + 1e-30           (util.Q_RTOL)
  * tLISI:          |t_gpu - t_ref| <= 1e-4 * |t_ref|                   (north_star's bound)
  * max Delta:      1e-6 relative (two fp32 subtractions + one, each correctly rounded; the max itself is exact)
  * argmax pixel:   oracle Delta at the reported pixel >= (1 - 1e-5) * oracle max (ties / rounding, R20)
  * candidates:     exact set, except tiles whose oracle z lies within 1e-4*(mu/sigma + |z|) of tau
  * tiles of fewer than 16 pixels (N_T <= 3 and partial edge tiles; util.needs_slack -- ONE rule):
                    the derived first-order fp32 input-rounding bound (util.fp32_slack) is added to the budgets above
  * frequency branch: q to util.EPS_Q_FP32, eta to util.eta_bound (the conditioning of the DC removal), k* and the
                    candidate band from the same bound (util.eta_z_band)
"""
import math

import numpy as np
import pytest
import torch

import oracle
import paper_2509_21754_b200 as fitrig
import synth
from tests import util

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def gpu_run(stack_gpu, taus=(5.0,), capacity=1 << 16, use_stream=False, want_tlisi=True, **params):
    L, H, W = stack_gpu.shape
    out = {}
    with fitrig.Context(H, W, L, **params) as ctx:
        U, Ty, Tx = ctx.map_dims()
        if use_stream:
            host = [stack_gpu[s].cpu().pin_memory() for s in range(L)]
            h_tl = torch.empty((U, Ty, Tx), dtype=torch.float32).pin_memory()
            ctx.stream(host, h_tl)
            torch.cuda.synchronize()
            out["tlisi_out"] = h_tl.numpy().copy()
        else:
            d_tl = torch.empty((U, Ty, Tx), dtype=torch.float32, device=DEV) if want_tlisi else None
            ctx.tlisi(stack_gpu, d_tl)
            torch.cuda.synchronize()
            out["tlisi_out"] = d_tl.cpu().numpy() if want_tlisi else None
        out["cands"] = {}
        for tau in taus:
            c, n = ctx.detect(tau, capacity)
            out["cands"][tau] = (c.copy(), n)
        out["M"], out["mu"], out["sigma"] = ctx.get_stats()
        out["q"] = ctx.get_map(0)
        out["tlisi"] = ctx.get_map(1)
        out["raw"] = ctx.get_raw()
        if params.get("branch", 0) == 1:
            out["eta"] = ctx.get_map(2)
            out["kstar"] = ctx.get_map(3).astype(np.int32)
        out["dims"] = (U, Ty, Tx)
        out["launches"] = ctx.launch_count()
    return out


def oracle_delta_at(stack_np, u, x, y):
    a, b, c = (float(stack_np[u + i][y, x]) for i in range(3))
    return abs(abs(b - a) - abs(c - b))


def check_against_oracle(stack_gpu, g, ref, taus, tile, branch=0, ref_mode=0, C=1e-6, small_tiles=False,
                         sample_argmax=4000, stack_np=None, extra_slack=None):
    """stack_np: the same snapshots on the host ([L,H,W] array or list of [H,W] arrays) when the caller has them."""
    if stack_np is None:
        stack_np = stack_gpu.cpu().numpy()
    res = ref.res
    # --- raw per-tile quantities of Eq. 6 ---
    sd, md, sr, ax, ay = g["raw"]
    q_slack = None
    if small_tiles or extra_slack is not None:
        # tiles of a few pixels: Delta is a cancellation of fp32-rounded differences, so a purely relative bound is
        # not attainable by ANY fp32 evaluation; add the derived first-order rounding bound (util.fp32_slack)
        eS, eM, eR = util.fp32_slack(np.asarray(stack_np), tile, C, ref_mode, extra=extra_slack)
        assert np.all(np.abs(sd - res.sumD) <= 2e-5 * res.sumD + eS)
        assert np.all(np.abs(md - res.maxD) <= 1e-6 * res.maxD + eM)
        assert np.all(np.abs(sr - res.sumR) <= 2e-5 * np.abs(res.sumR) + eR + 2e-5)
        n2m2 = res.q / np.where(res.sumD * res.maxD * res.sumR == 0, 1.0, res.sumD * res.maxD * res.sumR)
        q_slack = ((res.sumD + eS) * (res.maxD + eM) * (np.abs(res.sumR) + eR)
                   - res.sumD * res.maxD * np.abs(res.sumR)) * np.abs(n2m2)
    else:
        np.testing.assert_allclose(sd, res.sumD, rtol=2e-5, atol=1e-30)
        np.testing.assert_allclose(md, res.maxD, rtol=1e-6, atol=1e-30)  # three fp32 roundings vs fp64
        np.testing.assert_allclose(sr, res.sumR, rtol=2e-5, atol=2e-5)
    # --- argmax: unique up to ties / fp32 rounding of Delta (R20) ---
    Wd = stack_np[0].shape[1]
    exact = (ay.astype(np.int64) * Wd + ax) == res.argmax
    idx = np.argwhere(~exact)
    for (u, ty, tx) in idx[:sample_argmax]:
        d = oracle_delta_at(stack_np, u, int(ax[u, ty, tx]), int(ay[u, ty, tx]))
        assert d >= (1 - 1e-5) * res.maxD[u, ty, tx], (u, ty, tx, d, res.maxD[u, ty, tx])
        assert ty * tile <= ay[u, ty, tx] < (ty + 1) * tile and tx * tile <= ax[u, ty, tx] < (tx + 1) * tile
    assert exact.mean() > 0.99
    # --- M, q, tLISI ---
    if extra_slack is None:
        assert g["M"] == np.float32(res.M)
    else:  # the largest ACCUMULATED pixel: g - 1 fp32 additions against the exact sum
        assert abs(g["M"] - res.M) <= 1e-6 * res.M
    util.assert_map_close(g["q"], res.q, g["tlisi"], res.tlisi, slack=q_slack)
    if g["tlisi_out"] is not None:
        assert np.array_equal(g["tlisi_out"], g["tlisi"])
    if branch == 0:
        band = None
        if q_slack is None:
            np.testing.assert_allclose(g["mu"], ref.mu, rtol=1e-5)
            np.testing.assert_allclose(g["sigma"], ref.sigma, rtol=2e-4, atol=1e-30)
        else:  # the slack of q carries over to its mean, its standard deviation and z (first order)
            qs = q_slack.reshape(q_slack.shape[0], -1)
            zr = np.asarray(ref.z, dtype=np.float64).reshape(qs.shape)
            sd = np.where(ref.sigma > 0, ref.sigma, 1.0)
            assert np.all(np.abs(g["mu"] - ref.mu) <= 1e-5 * np.abs(ref.mu) + qs.mean(axis=1))
            assert np.all(np.abs(g["sigma"] - ref.sigma) <= 2e-4 * ref.sigma + qs.max(axis=1) + 1e-30)
            band = (util.Q_RTOL * ((np.abs(ref.mu) / sd)[:, None] + np.abs(zr))
                    + (qs + qs.mean(axis=1, keepdims=True)) / sd[:, None] + np.abs(zr) * qs.max(axis=1, keepdims=True) / sd[:, None])
        for tau in taus:
            c, n = g["cands"][tau]
            assert n == len(c)
            Tx = res.Tx
            lst = [(int(r["x"]), int(r["y"]), int(r["snapshot"]), float(r["score"]),
                    (int(r["y"]) // tile) * Tx + int(r["x"]) // tile, int(r["snapshot"])) for r in c]
            util.compare_candidates(lst, ref.z, ref.mu, ref.sigma, tau, Tx, res.Ty * Tx, band=band)
            for (x, y, u, score, t, _) in lst:  # reported pixel is (one of) the tile's max-Delta pixels
                assert oracle_delta_at(stack_np, u, x, y) >= (1 - 1e-5) * res.maxD[u].flat[t]


def oracle_run(stack_gpu, **kw):
    return oracle.run(stack_gpu.cpu().numpy(), **kw)


# ------------------------------------------------------------------------------------------
# Tiny config (BASELINE.json configs[0]) and its sweeps
# ------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def tiny():
    st, truth = synth.make_stack(synth.CONFIGS["tiny"], device=DEV)
    return st, truth


@pytest.mark.parametrize("ref_mode", [fitrig.REF_ABS, fitrig.REF_LITERAL, fitrig.REF_FLOOR])
def test_tiny_default_tile_all_reference_modes(tiny, ref_mode):
    st, _ = tiny
    taus = (3.0, 4.0, 5.0, 6.0)
    g = gpu_run(st, taus=taus, ref_mode=ref_mode)
    ref = oracle_run(st, tile=32, ref_mode=ref_mode, tau=5.0)
    check_against_oracle(st, g, ref, taus, 32, ref_mode=ref_mode)
    assert g["cands"][6.0][1] == 0  # SURVEY probe: the 8 sigma transient is below 6 sigma with 64 tiles


@pytest.mark.parametrize("tile", [1, 2, 4, 8, 16, 64, 5, 100])
def test_tiny_tile_sweep(tiny, tile):  # 8 and 16 take the fused kernel (sub-tiles of a warp's 32x32 block)
    st, truth = tiny
    taus = (3.0, 4.0, 5.0, 6.0)
    g = gpu_run(st, taus=taus, tile=tile, capacity=1 << 18)
    ref = oracle_run(st, tile=tile, tau=5.0)
    check_against_oracle(st, g, ref, taus, tile, small_tiles=util.needs_slack(256, 256, tile))
    if tile in (4, 8, 16):
        t = truth.transients[0]
        c, n = g["cands"][6.0]
        assert any(int(r["x"]) == t.x and int(r["y"]) == t.y and int(r["snapshot"]) in (0, 2, 4) for r in c)


@pytest.mark.parametrize("tile", [32, 16, 8, 64, 96, 4, 2, 1])
@pytest.mark.parametrize("H,W", [(250, 252), (250, 250), (33, 36), (32, 32), (31, 64), (40, 72), (9, 12)])
def test_partial_edge_tiles_and_odd_shapes(tiny, H, W, tile):
    st = tiny[0][:, :H, :W].contiguous()
    taus = (2.0, 3.0) if (H // tile) * (W // tile) > 12 else (0.5,)
    g = gpu_run(st, taus=taus, tile=tile, capacity=1 << 18)
    ref = oracle_run(st, tile=tile, tau=taus[-1])
    check_against_oracle(st, g, ref, taus, tile, small_tiles=util.needs_slack(H, W, tile))


def test_unaligned_base_pointer_falls_back_to_generic_kernel(tiny):
    flat = torch.empty(8 * 256 * 256 + 1, dtype=torch.float32, device=DEV)
    st = flat[1:].view(8, 256, 256)
    st.copy_(tiny[0])
    assert st.data_ptr() % 16 != 0
    g = gpu_run(st, taus=(4.0,))
    ref = oracle_run(st, tile=32, tau=4.0)
    check_against_oracle(st, g, ref, (4.0,), 32)


def test_m_override_scales_q_but_not_candidates(tiny):
    st, _ = tiny
    g1 = gpu_run(st, taus=(4.0,))
    g2 = gpu_run(st, taus=(4.0,), M_override=123.456)
    assert g2["M"] == np.float32(123.456)
    ref = oracle_run(st, tile=32, tau=4.0, M=float(np.float32(123.456)))
    util.assert_map_close(g2["q"], ref.res.q)
    assert [tuple(r)[:3] for r in g1["cands"][4.0][0]] == [tuple(r)[:3] for r in g2["cands"][4.0][0]]  # P7


@pytest.mark.parametrize("tile", [32, 16, 8, 4, 1])
def test_work_partition_does_not_change_the_map(tiny, monkeypatch, tile):
    """The per-CTA ranges of (box, unit) pairs cut tiles' time series at different places for different box
    widths / grids / ring depths; the per-tile results must not depend on where the cuts fall, on which warp of
    a box owns the tile, or on boxes that hang over the image edge (box width 3 or 5 on an 8-tile row)."""
    st, _ = tiny
    monkeypatch.setenv("FITRIG_BOX_TILES", "1")
    monkeypatch.setenv("FITRIG_GRID", "1")
    a = gpu_run(st, tile=tile)  # one consumer warp walks all 384 pairs: no cut inside any tile
    for box, grid, stages in ((3, 7, 2), (8, 148, 6), (5, 13, 3), (8, 5, 7), (2, 40, 8)):
        monkeypatch.setenv("FITRIG_BOX_TILES", str(box))
        monkeypatch.setenv("FITRIG_GRID", str(grid))
        monkeypatch.setenv("FITRIG_STAGES", str(stages))
        for evict in ("0", "1"):
            monkeypatch.setenv("FITRIG_EVICT_FIRST", evict)
            b = gpu_run(st, tile=tile)
            assert np.array_equal(a["q"], b["q"]) and a["M"] == b["M"]
            for x, y in zip(a["raw"], b["raw"]):
                assert np.array_equal(x, y)


@pytest.mark.parametrize("tile", [32, 16, 8, 64, 128, 4, 2, 1])
def test_fused_and_generic_kernels_agree(tiny, monkeypatch, tile):
    st, _ = tiny
    a = gpu_run(st, tile=tile)
    monkeypatch.setenv("FITRIG_FORCE_GENERIC", "1")
    b = gpu_run(st, tile=tile)
    assert np.array_equal(a["raw"][1], b["raw"][1])  # max Delta exact
    assert np.array_equal(a["raw"][3], b["raw"][3]) and np.array_equal(a["raw"][4], b["raw"][4])
    np.testing.assert_allclose(a["q"], b["q"], rtol=1e-5)


# ------------------------------------------------------------------------------------------
# seeded random sweep over shapes, tile sizes, modes and entry points (every kernel variant, ragged edges)
# ------------------------------------------------------------------------------------------
def _random_cases(n, seed=20250921):
    rng = np.random.default_rng(seed)
    cases = []
    for i in range(n):
        tile = int(rng.choice([32, 32, 16, 8, 64, 96, 5, 4, 12]))
        H = int(rng.integers(max(3, tile // 2), 200))
        W = int(rng.integers(3, 60)) * 4 if rng.random() < 0.8 else int(rng.integers(9, 230))
        g = int(rng.choice([1, 1, 1, 2, 3]))
        L = int(rng.integers(3, 8)) * g + int(rng.integers(0, g))
        cases.append((i, H, W, L, tile, g, int(rng.integers(0, 3)), bool(rng.random() < 0.35), int(rng.integers(0, 2))))
    return cases


@pytest.mark.parametrize("i,H,W,L,tile,g,ref_mode,use_stream,branch", _random_cases(28))
def test_random_shapes_and_modes(i, H, W, L, tile, g, ref_mode, use_stream, branch):
    st = synth.gaussian_noise_stack(L, H, W, seed=1000 + i, device=DEV)
    st[:, H // 2, W // 2] += 25.0 * (torch.arange(L, device=DEV) % 3 == 1)  # something to detect
    if ref_mode == 2:
        st = st + 3.0  # FLOOR: keep the reference mostly above C so that r is not saturated everywhere
    st[0, 0, 0] = 0.0  # an exact zero (reference pixel of no unit) and one that is a reference pixel
    if L // g >= 3:
        st[g:2 * g, min(1, H - 1), min(2, W - 1)] = 0.0
    n_tiles = (-(-H // tile)) * (-(-W // tile))
    tau = 2.0 if n_tiles > 8 else 0.3
    kw = dict(tile=tile, accumulate=g, ref_mode=ref_mode, branch=branch)
    if use_stream:
        q = tile if tile % 32 == 0 else (32 if 32 % tile == 0 else tile)
        kw["strip_rows"] = q * int(1 + i % 2)
    gp = gpu_run(st, taus=(tau,), use_stream=use_stream, **kw)
    ref = oracle_run(st, tile=tile, tau=tau, ref_mode=ref_mode, branch=branch, accumulate_g=g)
    imgs = np.stack(oracle.accumulate(st.cpu().numpy(), g))
    # LITERAL (Eq. 5 as printed): r is signed and unbounded below, so sum r is a cancellation; its derived conditioning
    # bound (util.fp32_slack, ref_mode 1) is part of the budget for q, the statistics and the candidate band
    small = util.needs_slack(H, W, tile) or ref_mode == 1
    extra = util.accumulation_slack(st.cpu().numpy(), g) if g > 1 else (np.zeros_like(imgs[:-2]) if small else None)
    check_against_oracle(None, gp, ref, (tau,) if branch == 0 else (), tile, branch=branch, ref_mode=ref_mode,
                         small_tiles=small, stack_np=imgs, extra_slack=extra)
    if branch == 1 and ref.res.U >= 2 and ref_mode != 1 and not small and g == 1:
        bound = util.eta_bound(ref.res.q, 1, eps_q=util.Q_RTOL)  # (odd tile sizes: only the 1e-4 of the map is claimed)
        assert np.all(np.abs(gp["eta"] - ref.eta) <= bound + 2e-7 * np.abs(ref.eta))


# ------------------------------------------------------------------------------------------
# degenerate and edge cases
# ------------------------------------------------------------------------------------------
def test_identical_snapshots_no_transient_value_and_no_candidates():
    one = synth.gaussian_noise_stack(1, 128, 128, device=DEV)[0]
    st = one.unsqueeze(0).repeat(5, 1, 1).contiguous()
    g = gpu_run(st, taus=(0.0, 3.0))
    assert np.all(g["tlisi"] == 1.0) and np.all(g["q"] == 0.0)  # P1
    assert np.all(g["sigma"] == 0.0)
    assert g["cands"][0.0][1] == 0 and g["cands"][3.0][1] == 0  # R4


def test_minimum_problem_three_snapshots_one_tile():
    st = synth.gaussian_noise_stack(3, 32, 32, device=DEV)
    g = gpu_run(st, taus=(0.5,))
    ref = oracle_run(st, tile=32, tau=0.5)
    check_against_oracle(st, g, ref, (0.5,), 32)
    assert g["dims"] == (1, 1, 1) and g["cands"][0.5][1] == 0  # one tile: sigma = 0


def test_zero_and_negative_reference_pixels_and_steady_sky():
    st = synth.gaussian_noise_stack(5, 64, 96, device=DEV)
    st[1, :8, :8] = 0.0  # x == 0 -> C branch of Eq. 5
    st[2, 10:20, 30:40] = 0.0
    st[:, 40:, :] = st[0:1, 40:, :]  # steady region: Delta = 0, including 0/0-like pixels
    st[:, 50:, 50:] = 0.0
    for mode in (fitrig.REF_ABS, fitrig.REF_LITERAL, fitrig.REF_FLOOR):
        g = gpu_run(st, taus=(1.0,), ref_mode=mode)
        ref = oracle_run(st, tile=32, ref_mode=mode, tau=1.0)
        check_against_oracle(st, g, ref, (1.0,), 32)


def test_large_C_exercises_the_zero_reference_ratio():
    st = synth.gaussian_noise_stack(4, 64, 64, device=DEV) * 0.01
    st[1, ::3, ::5] = 0.0
    g = gpu_run(st, taus=(1.0,), C=0.5)
    ref = oracle_run(st, tile=32, C=0.5, tau=1.0)
    check_against_oracle(st, g, ref, (1.0,), 32)


def test_all_negative_images_floor_M_at_C():
    st = -torch.abs(synth.gaussian_noise_stack(4, 64, 64, device=DEV)) - 1.0
    g = gpu_run(st, taus=(1.0,))
    assert g["M"] == np.float32(1e-6)  # R2
    ref = oracle_run(st, tile=32, tau=1.0)
    util.assert_map_close(g["q"], ref.res.q)


def test_capacity_overflow_reports_total_and_keeps_order(tiny):
    st, _ = tiny
    with fitrig.Context(256, 256, 8, tile=2) as ctx:
        ctx.tlisi(st)
        full, n = ctx.detect(1.0, 1 << 17)
        assert n == len(full) and n > 5000
        part, n2 = ctx.detect(1.0, 10)
        assert n2 == n and len(part) == 10 and np.array_equal(part, full[:10])
        part, n3 = ctx.detect(1.0, 5000)  # longer than the pinned staging chunk
        assert n3 == n and np.array_equal(part, full[:5000])
        none, n4 = ctx.detect(1.0, 0)
        assert n4 == n and len(none) == 0


def test_detect_before_tlisi_is_a_state_error():
    with fitrig.Context(64, 64, 4) as ctx:
        with pytest.raises(fitrig.FitrigError) as e:
            ctx.detect(5.0)
        assert e.value.code == -4
        with pytest.raises(fitrig.FitrigError):
            ctx.get_stats()


def test_repeated_calls_on_one_context_are_reproducible(tiny):
    st, _ = tiny
    with fitrig.Context(256, 256, 8) as ctx:
        ctx.tlisi(st)
        q1 = ctx.get_map(0)
        c1, _ = ctx.detect(3.0)
        st2 = st.flip(0).contiguous()
        ctx.tlisi(st2)
        q2 = ctx.get_map(0)
        ctx.tlisi(st)
        q3 = ctx.get_map(0)
        c3, _ = ctx.detect(3.0)
    assert np.array_equal(q1, q3) and np.array_equal(c1, c3)
    np.testing.assert_allclose(q2, q1[::-1], rtol=1e-5)  # P5: time reversal


# ------------------------------------------------------------------------------------------
# streaming (a9)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("H,W,strip,tile", [(256, 256, 64, 32), (250, 252, 96, 32), (300, 200, 32, 32), (250, 250, 64, 32),
                                            (250, 252, 64, 16), (300, 200, 96, 8), (256, 256, 48, 16), (256, 256, 0, 8),
                                            (300, 200, 128, 64), (250, 252, 96, 96), (250, 252, 64, 4), (120, 100, 32, 1)])
def test_stream_equals_resident_and_oracle(tiny, H, W, strip, tile):
    # strips of 48 rows with 16-pixel tiles do not start on 32-row blocks: those launches take the generic kernel
    base = synth.gaussian_noise_stack(6, 320, 256, seed=7, device=DEV)
    st = base[:, :H, :W].contiguous()
    taus = (2.5,)
    a = gpu_run(st, taus=taus, tile=tile)
    b = gpu_run(st, taus=taus, use_stream=True, strip_rows=strip, tile=tile)
    if strip != 48:
        assert np.array_equal(a["q"], b["q"])
        assert np.array_equal(a["cands"][2.5][0], b["cands"][2.5][0])
    assert a["M"] == b["M"]
    ref = oracle_run(st, tile=tile, tau=2.5)
    check_against_oracle(st, b, ref, taus, tile, small_tiles=util.needs_slack(H, W, tile))


def test_stream_generic_tile(tiny):
    st = tiny[0]
    a = gpu_run(st, taus=(4.0,), tile=5)
    b = gpu_run(st, taus=(4.0,), tile=5, use_stream=True, strip_rows=40)
    assert np.array_equal(a["q"], b["q"]) and np.array_equal(a["cands"][4.0][0], b["cands"][4.0][0])


# ------------------------------------------------------------------------------------------
# image-frequency branch (a10), BASELINE.json configs[4] at reduced size
# ------------------------------------------------------------------------------------------
def _check_frequency(g, ref, taus, tile, harmonics=1):
    """Frequency-branch parity with DERIVED tolerances: q to the fp32 budget EPS_Q_FP32, eta to
    the conditioning bound that budget implies (util.eta_bound), k* wherever the oracle's own spectrum separates the
    two bins by more than that bound (R23), statistics and candidate band from the same bound."""
    util.assert_map_close(g["q"], ref.res.q, rtol=util.EPS_Q_FP32)
    bound = util.eta_bound(ref.res.q, harmonics)
    assert np.all(np.abs(g["eta"] - ref.eta) <= bound + 2e-7 * np.abs(ref.eta)), \
        float((np.abs(g["eta"] - ref.eta) / (bound + 2e-7 * np.abs(ref.eta))).max())
    U = ref.res.q.shape[0]
    K = U // 2
    diff = np.argwhere(g["kstar"] != ref.kstar)
    if len(diff):
        _, _, mag = oracle.spectrum_hsum(ref.res.q, harmonics, want_mag=True)
    for (ty, tx) in diff:  # another bin only where its (harmonic-summed) magnitude is within the bound of the best
        k = int(g["kstar"][ty, tx])
        best_k = max(mag[k - 1:h * k:k, ty, tx].sum() / math.sqrt(h)
                     for h in (1, 2, 4, 8, 16, 32) if h <= harmonics and h * k <= K)
        assert best_k >= ref.eta[ty, tx] - 2.0 * bound[ty, tx] - 4e-7 * ref.eta[ty, tx]
    bmean, bmax = float(bound.mean()), float(bound.max())
    assert abs(g["mu"][0] - ref.mu[0]) <= bmean + 2e-7 * abs(ref.mu[0])
    assert abs(g["sigma"][0] - ref.sigma[0]) <= bmax + 2e-7 * ref.sigma[0]
    Tx = ref.res.Tx
    band = util.eta_z_band(ref.eta, ref.z, ref.sigma[0], bound)
    for tau in taus:
        c, n = g["cands"][tau]
        lst = [(int(r["x"]), int(r["y"]), int(r["snapshot"]), float(r["score"]),
                (int(r["y"]) // tile) * Tx + int(r["x"]) // tile, 0) for r in c]
        util.compare_candidates(lst, ref.z[None], ref.mu, ref.sigma, tau, Tx, ref.res.Ty * Tx, band=band[None])
        for (x, y, k, score, t, _) in lst:
            assert (x % tile, y % tile) == (tile // 2, tile // 2)
            assert k == g["kstar"].flat[t]  # the record carries the library's k* (checked against the oracle above)
    return diff


@pytest.mark.parametrize("channel", [0, 15])
def test_frequency_branch_reduced_config5(channel):
    # reduced size: 1024 tiles instead of 16384, so the transients are drawn at 8 sigma instead of 5 to stay
    # detectable (oracle on this recipe: z = 16.8 and 8.7 at k* = 15); everything else as configs[4]
    cfg = synth.scaled(synth.CONFIGS["imgfreq"], 1024, 1024).replace(n_transients=2, transient_peak=8.0)
    st, truth = synth.make_stack(cfg, device=DEV, channel=channel)
    taus = (4.0, 6.0)
    g = gpu_run(st, taus=taus, branch=fitrig.BRANCH_FREQUENCY)
    ref = oracle_run(st, tile=32, tau=6.0, branch=1)
    _check_frequency(g, ref, taus, 32)
    if channel == 0:  # the periodic transients stand out in eta at the Nyquist bin (on 1 snapshot in 8)
        c, n = g["cands"][6.0]
        tiles = {(int(r["y"]) // 32, int(r["x"]) // 32): int(r["snapshot"]) for r in c}
        for t in truth.transients:
            assert tiles.get((t.y // 32, t.x // 32)) == 15


@pytest.mark.parametrize("harmonics,U", [(2, 30), (4, 30), (8, 62), (32, 21)])
def test_frequency_branch_harmonic_summing(harmonics, U):
    """h = harmonic summing (R26) against oracle.spectrum_hsum; a periodic transient with a short duty
    cycle puts power into several harmonics of its repetition rate."""
    cfg = synth.scaled(synth.CONFIGS["imgfreq"], 512, 512, L=U + 2).replace(n_transients=2, transient_peak=9.0)
    st, truth = synth.make_stack(cfg, device=DEV, channel=0)
    taus = (3.0,)
    g = gpu_run(st, taus=taus, branch=fitrig.BRANCH_FREQUENCY, harmonics=harmonics)
    ref = oracle_run(st, tile=32, tau=3.0, branch=1, harmonics=harmonics)
    _check_frequency(g, ref, taus, 32, harmonics)
    assert g["cands"][3.0][1] > 0


def test_harmonics_argument_is_validated():
    for bad in (3, 64, -1):
        with pytest.raises(fitrig.FitrigError) as e:
            fitrig.Context(64, 64, 8, branch=fitrig.BRANCH_FREQUENCY, harmonics=bad)
        assert e.value.code == fitrig.binding.ERR_INVALID_ARG


def test_frequency_branch_odd_length_series():
    st = synth.gaussian_noise_stack(9, 96, 128, seed=11, device=DEV)  # U = 7
    g = gpu_run(st, taus=(1.0,), branch=fitrig.BRANCH_FREQUENCY)
    ref = oracle_run(st, tile=32, tau=1.0, branch=1)
    _check_frequency(g, ref, (1.0,), 32)


# ------------------------------------------------------------------------------------------
# snapshot accumulation (section 3.3.2, Fig. 16; R25)
# ------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def long_tiny():
    cfg = synth.scaled(synth.CONFIGS["tiny"], 256, 256, L=20)
    return synth.make_stack(cfg, device=DEV)


@pytest.mark.parametrize("g,H,W,tile,use_stream", [(2, 256, 256, 32, False), (3, 250, 252, 32, False), (4, 256, 256, 32, True),
                                                   (5, 256, 256, 32, False), (6, 128, 96, 32, True), (2, 120, 100, 8, False),
                                                   (3, 64, 64, 1, False), (2, 250, 252, 16, False), (5, 256, 256, 8, True),
                                                   (3, 120, 98, 16, False)])
def test_accumulated_snapshots_match_oracle(long_tiny, g, H, W, tile, use_stream):
    st, _ = long_tiny
    st = st[:, :H, :W].contiguous()
    taus = (3.0,) if (H // tile) * (W // tile) >= 40 else (1.0,)
    kw = dict(strip_rows=64) if use_stream and tile == 32 else {}
    gp = gpu_run(st, taus=taus, accumulate=g, tile=tile, use_stream=use_stream, **kw)
    assert gp["dims"][0] == 20 // g - 2  # the incomplete trailing group (20 mod g snapshots) is left out
    ref = oracle_run(st, tile=tile, tau=taus[0], accumulate_g=g)
    acc_np = np.stack(oracle.accumulate(st.cpu().numpy(), g))  # fp64 images: what Delta is measured on
    # fp32 sums of g snapshots carry a rounding of (g-1) 2^-24 sum|x| per pixel into the differences: derived slack
    check_against_oracle(None, gp, ref, taus, tile, stack_np=acc_np,
                         extra_slack=util.accumulation_slack(st.cpu().numpy(), g))


def test_accumulate_one_is_bit_identical_and_frequency_branch_accumulates(long_tiny):
    st, _ = long_tiny
    a, b = gpu_run(st), gpu_run(st, accumulate=1)
    assert np.array_equal(a["q"], b["q"]) and a["M"] == b["M"]
    gq = gpu_run(st, taus=(1.0,), accumulate=2, branch=fitrig.BRANCH_FREQUENCY)
    ref = oracle_run(st, tile=32, tau=1.0, branch=1, accumulate_g=2)
    util.assert_map_close(gq["q"], ref.res.q)
    # accumulated snapshots: the map's budget is 1e-4 plus the accumulation slack (R25); eta inherits it
    bound = util.eta_bound(ref.res.q, 1, eps_q=util.Q_RTOL)
    assert np.all(np.abs(gq["eta"] - ref.eta) <= bound + 2e-7 * np.abs(ref.eta))
    with pytest.raises(fitrig.FitrigError) as e:
        fitrig.Context(64, 64, 8, accumulate=3)  # 8 // 3 = 2 accumulated snapshots: fewer than 3
    assert e.value.code == fitrig.binding.ERR_INVALID_ARG


# ------------------------------------------------------------------------------------------
# overlapping windows (an extension; R27)
# ------------------------------------------------------------------------------------------
def _check_windows(st, g, ref, tile, stride, tau):
    sd, md, sr, ax, ay = g["raw"]
    res = ref.res
    assert g["dims"] == (res.U, res.Ty, res.Tx)
    np.testing.assert_allclose(sd, res.sumD, rtol=2e-5, atol=1e-30)
    np.testing.assert_allclose(md, res.maxD, rtol=1e-6, atol=1e-30)
    np.testing.assert_allclose(sr, res.sumR, rtol=2e-5, atol=2e-5)
    W = st.shape[2]
    exact = (ay.astype(np.int64) * W + ax) == res.argmax
    assert exact.mean() > 0.99
    stack_np = st.cpu().numpy()
    for (u, ty, tx) in np.argwhere(~exact)[:2000]:
        x, y = int(ax[u, ty, tx]), int(ay[u, ty, tx])
        assert oracle_delta_at(stack_np, u, x, y) >= (1 - 1e-5) * res.maxD[u, ty, tx]
        assert ty * stride <= y < ty * stride + tile and tx * stride <= x < tx * stride + tile
    assert g["M"] == np.float32(res.M)
    util.assert_map_close(g["q"], res.q, g["tlisi"], res.tlisi)
    np.testing.assert_allclose(g["mu"], ref.mu, rtol=1e-5)
    np.testing.assert_allclose(g["sigma"], ref.sigma, rtol=2e-4, atol=1e-30)
    c, n = g["cands"][tau]
    Tx = res.Tx
    lst = []
    for r in c:  # the window of a candidate is not recoverable from its peak pixel: find it through the oracle's z order
        lst.append((int(r["x"]), int(r["y"]), int(r["snapshot"]), float(r["score"])))
    sel = [(int(u), int(t)) for u, t in zip(ref.cands.snapshot, ref.cands.tile)]
    band = 1e-4 * (np.abs(ref.mu) / ref.sigma)[:, None, None] + 1e-4 * np.abs(ref.z)
    sure = {(u, t) for (u, t) in sel if ref.z[u].flat[t] > tau + band[u].flat[t]}
    assert len(lst) >= len(sure) and abs(len(lst) - len(sel)) <= int((np.abs(ref.z - tau) <= band).sum())
    if len(lst) == len(sel):
        for (x, y, u, score), (ru, rt) in zip(lst, sel):
            assert u == ru and abs(score - ref.z[ru].flat[rt]) <= band[ru].flat[rt] + 1e-6 * abs(score)
            ty, tx = divmod(rt, Tx)
            assert ty * stride <= y < ty * stride + tile and tx * stride <= x < tx * stride + tile


@pytest.mark.parametrize("H,W,tile,stride,use_stream", [(256, 256, 32, 16, False), (250, 252, 32, 8, False), (256, 256, 64, 32, False),
                                                        (200, 120, 16, 4, False), (96, 64, 32, 32, False), (250, 252, 32, 16, True),
                                                        (130, 100, 64, 16, False), (120, 100, 24, 12, False), (90, 250, 32, 8, False)])
def test_overlapping_windows_match_oracle(tiny, H, W, tile, stride, use_stream):
    st = tiny[0][:, :H, :W].contiguous()
    tau = 3.0
    kw = dict(strip_rows=64) if use_stream else {}
    g = gpu_run(st, taus=(tau,), tile=tile, stride=stride, use_stream=use_stream, capacity=1 << 18, **kw)
    ref = oracle_run(st, tile=tile, tau=tau, stride=stride)
    _check_windows(st, g, ref, tile, stride, tau)


def test_windows_arguments_are_validated():
    for kw in (dict(tile=32, stride=12), dict(tile=32, stride=16, branch=fitrig.BRANCH_FREQUENCY),
               dict(tile=32, stride=16, accumulate=2), dict(tile=32, stride=16, row_offset=32), dict(tile=32, stride=-4)):
        with pytest.raises(fitrig.FitrigError) as e:
            fitrig.Context(128, 128, 8, **kw)
        assert e.value.code == fitrig.binding.ERR_INVALID_ARG


# ------------------------------------------------------------------------------------------
# real-time mode: fitrig_push (PAPER.md:189 running maximum; Fig. 14 timeline), against oracle.run_realtime
# ------------------------------------------------------------------------------------------
def _push_all(ctx, snaps, tau, want_maps=True):
    """Feed every snapshot, then flush; returns {unit: (cands, n, q, M, mu, sigma, tlisi)} in arrival order."""
    U, Ty, Tx = ctx.map_dims()
    got = {}
    d_tl = torch.empty((Ty, Tx), dtype=torch.float32, device=DEV)
    for s in list(snaps) + [None]:
        unit, c, n = ctx.push(s, tau, d_tl)
        if unit >= 0:
            assert unit == len(got)  # units come out in order, one per push
            M, mu, sd = ctx.get_stats()
            got[unit] = (c.copy(), n, ctx.get_map(0)[0] if want_maps else None, M, mu[0], sd[0], d_tl.cpu().numpy())
    unit, c, n = ctx.push(None, tau)  # nothing left
    assert unit == -1 and n == 0
    return got


@pytest.mark.parametrize("H,W,tile,on_device", [(256, 256, 32, False), (250, 252, 32, False), (256, 256, 32, True),
                                                (120, 100, 8, False), (250, 252, 16, False), (120, 102, 8, False),
                                                (120, 100, 4, False), (256, 256, 64, False)])  # 64: merged from 32-pixel cells
def test_push_realtime_matches_oracle(tiny, H, W, tile, on_device):
    st, _ = tiny
    st = st[:, :H, :W].contiguous()
    L, tau = st.shape[0], 3.0
    snaps = [st[s] for s in range(L)] if on_device else [st[s].cpu().pin_memory() for s in range(L)]
    ref = oracle.run_realtime(st.cpu().numpy(), tile=tile, tau=tau)
    with fitrig.Context(H, W, 3, tile=tile) as ctx:
        assert ctx.map_dims()[0] == 1
        first = ctx.push(snaps[0], tau)
        assert first[0] == -1 and first[2] == 0
        ctx.push_reset()
        got = _push_all(ctx, snaps, tau)
        assert sorted(got) == list(range(L - 2))
        stack_np = st.cpu().numpy()
        for n, (c, cnt, q, M, mu, sd, tl) in got.items():
            r = ref[n]
            assert M == np.float32(r.res.M)  # running maximum of x_0 .. x_{n+2}
            util.assert_map_close(q, r.res.q[0], tl, r.res.tlisi[0])
            assert abs(mu - r.mu[0]) <= 1e-5 * abs(r.mu[0]) and abs(sd - r.sigma[0]) <= 2e-4 * r.sigma[0]
            Tx = r.res.Tx
            lst = [(int(k["x"]), int(k["y"]), int(k["snapshot"]), float(k["score"]),
                    (int(k["y"]) // tile) * Tx + int(k["x"]) // tile, 0) for k in c]
            assert all(k[2] == n for k in lst) and cnt == len(c)
            util.compare_candidates(lst, r.z, r.mu, r.sigma, tau, Tx, r.res.Ty * Tx)
            for (x, y, u, score, t, _) in lst:
                assert oracle_delta_at(stack_np, n, x, y) >= (1 - 1e-5) * r.res.maxD[0].flat[t]
        assert sum(v[1] for v in got.values()) > 0
        # a second pass after a reset reproduces the first bit for bit
        ctx.push_reset()
        again = _push_all(ctx, snaps, tau)
        for n in got:
            assert np.array_equal(got[n][2], again[n][2]) and np.array_equal(got[n][0], again[n][0])


def test_push_needs_a_three_snapshot_context():
    with fitrig.Context(64, 64, 5) as ctx:
        with pytest.raises(fitrig.FitrigError) as e:
            ctx.push(torch.zeros(64, 64, device=DEV), 3.0)
        assert e.value.code == fitrig.binding.ERR_INVALID_ARG


# ------------------------------------------------------------------------------------------
# row shards: the shards of one image, run one after another on this GPU (no shard waits
# on another: the exchange vector is simply stacked), must reproduce the whole-image result
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("H,W,world", [(256, 256, 2), (250, 252, 3), (512, 256, 4), (96, 64, 3)])
def test_row_shards_reproduce_the_whole_image(H, W, world):
    from paper_2509_21754_b200 import shard
    cfg = synth.scaled(synth.CONFIGS["tiny"], H, W)
    st, _ = synth.make_stack(cfg, device=DEV)
    L, tau = cfg.L, (3.0 if H * W >= 256 * 250 else 1.0)  # 6 tiles cannot reach z = 3 (P7: max z <= sqrt(n-1))
    whole = gpu_run(st, taus=(tau,))
    rows = shard.row_shards(H, 32, world)
    ctxs, vecs = [], []
    try:
        for (r0, r1) in rows:
            ctx = fitrig.Context(r1 - r0, W, L, row_offset=r0)
            ctxs.append(ctx)
            ctx.tlisi(st[:, r0:r1].contiguous())
            v = torch.empty(2 + 2 * (L - 2), dtype=torch.float64, device=DEV)
            ctx.shard_export(v)
            vecs.append(v)
        allv = torch.stack(vecs).contiguous()  # what the all-gather delivers to every shard
        qs, tls, lists = [], [], []
        for ctx, (r0, r1) in zip(ctxs, rows):
            U, Ty, Tx = ctx.map_dims()
            d_tl = torch.empty((U, Ty, Tx), dtype=torch.float32, device=DEV)
            ctx.shard_import(allv, world, d_tl)
            c, n = ctx.detect(tau)
            M, mu, sd = ctx.get_stats()
            assert M == whole["M"]
            np.testing.assert_allclose(mu, whole["mu"], rtol=1e-6)
            np.testing.assert_allclose(sd, whole["sigma"], rtol=1e-5)
            qs.append(ctx.get_map(0))
            tls.append(d_tl.cpu().numpy())
            lists.append(c.copy())
            assert all(r0 <= int(y) < r1 for y in c["y"])
    finally:
        for ctx in ctxs:
            ctx.close()
    assert np.array_equal(np.concatenate(qs, axis=1), whole["q"])  # same raw sums, same M, same fp64 combine
    assert np.array_equal(np.concatenate(tls, axis=1), whole["tlisi"])
    merged = shard.merge_candidates(lists)
    ref_c, ref_n = whole["cands"][tau]
    # z differs in the last bits (mu, sigma from sums of p instead of the rounded q map): compare outside a 1e-5 band
    keep = lambda c: {(int(r["snapshot"]), int(r["y"]), int(r["x"])) for r in c if abs(float(r["score"]) - tau) > 1e-5 * 20}
    assert keep(merged) == keep(ref_c) and ref_n > 0
    if len(merged) == len(ref_c):
        assert np.array_equal(merged["x"], ref_c["x"]) and np.array_equal(merged["y"], ref_c["y"])
        assert np.array_equal(merged["snapshot"], ref_c["snapshot"])
        np.testing.assert_allclose(merged["score"], ref_c["score"], rtol=1e-4, atol=1e-5)


def test_shard_calls_argument_and_state_errors():
    with fitrig.Context(64, 64, 4) as ctx:
        v = torch.empty(2 + 2 * 2, dtype=torch.float64, device=DEV)
        with pytest.raises(fitrig.FitrigError) as e:
            ctx.shard_export(v)
        assert e.value.code == fitrig.binding.ERR_STATE
    with pytest.raises(fitrig.FitrigError) as e:
        fitrig.Context(64, 64, 4, row_offset=16)  # not a multiple of the tile
    assert e.value.code == fitrig.binding.ERR_INVALID_ARG
    with fitrig.Context(64, 64, 4) as ctx:  # the eta exchange belongs to the frequency branch
        ctx.tlisi(synth.gaussian_noise_stack(4, 64, 64, device=DEV))
        with pytest.raises(fitrig.FitrigError) as e:
            ctx.shard_export_eta(torch.empty(3, dtype=torch.float64, device=DEV))
        assert e.value.code == fitrig.binding.ERR_INVALID_ARG
    with fitrig.Context(64, 64, 4, branch=fitrig.BRANCH_FREQUENCY) as ctx:
        ctx.tlisi(synth.gaussian_noise_stack(4, 64, 64, device=DEV))
        with pytest.raises(fitrig.FitrigError) as e:  # import before export
            ctx.shard_import_eta(torch.empty(3, dtype=torch.float64, device=DEV), 1)
        assert e.value.code == fitrig.binding.ERR_STATE


# ------------------------------------------------------------------------------------------
# full-size configs, in the launch configuration bench.py times
# ------------------------------------------------------------------------------------------
def test_config2_meerkat_full_size_full_oracle():
    cfg = synth.CONFIGS["meerkat"]
    st, truth = synth.make_stack(cfg, device=DEV)
    taus = (3.0, 5.0)
    g = gpu_run(st, taus=taus, want_tlisi=True)
    oracle.set_threads(0)
    ref = oracle_run(st, tile=32, tau=5.0)  # 1.07 GB, a few seconds on the host cores
    check_against_oracle(st, g, ref, taus, 32)
    assert g["cands"][3.0][1] > 0


def _host_snapshots(st):
    """[L,H,W] CUDA tensor -> list of L pinned host tensors (the buffers both the library and the oracle read)."""
    host = []
    for s in range(st.shape[0]):
        h = torch.empty(st.shape[1:], dtype=torch.float32).pin_memory()
        h.copy_(st[s])
        host.append(h)
    torch.cuda.synchronize()
    return host


def test_config3_ska_full_size_full_oracle():
    cfg = synth.CONFIGS["ska_aa2"]
    free, _ = torch.cuda.mem_get_info()
    if free < 12 << 30:
        pytest.skip("needs 12 GB of device memory")
    st, truth = synth.make_stack(cfg, device=DEV)
    taus = (5.0, 6.0, 7.0)
    g = gpu_run(st, taus=taus, want_tlisi=False)
    U, Ty, Tx = g["dims"]
    stack_np = [st[s].cpu().numpy() for s in range(cfg.L)]
    oracle.set_threads(0)
    ref = oracle.run(stack_np, tile=32, tau=5.0)  # 8.6 GB: a few seconds on the host cores
    check_against_oracle(st, g, ref, taus, 32, stack_np=stack_np)
    n5, n6, n7 = (g["cands"][t][1] for t in taus)
    assert n5 >= n6 >= n7 and n5 > 0
    # statistics recomputed from the library's own q map (properties that hold at any size)
    q = g["q"].astype(np.float64).reshape(U, -1)
    np.testing.assert_allclose(g["mu"], q.mean(axis=1), rtol=1e-9)
    np.testing.assert_allclose(g["sigma"], q.std(axis=1), rtol=1e-7)


def test_config4_stream50k_full_size_full_oracle():
    """BASELINE.json configs[3]: 4 x 50000 x 50000 in pinned host memory, streamed in row strips (partial last
    tile row and column of 16 px, R5), against the oracle on the very same host buffers; and the resident path
    on the same data must give the bit-identical map (strips cut the work differently, not the tiles)."""
    import psutil
    cfg = synth.CONFIGS["stream50k"]
    free, _ = torch.cuda.mem_get_info()
    if free < 60 << 30 or psutil.virtual_memory().available < 90 << 30:
        pytest.skip("needs 60 GB of device memory and 90 GB of host memory")
    st, truth = synth.make_stack(cfg, device=DEV)
    host = _host_snapshots(st)
    tau = cfg.tau
    with fitrig.Context(cfg.H, cfg.W, cfg.L) as ctx:
        U, Ty, Tx = ctx.map_dims()
        assert (U, Ty, Tx) == (2, 1563, 1563)
        h_tl = torch.empty((U, Ty, Tx), dtype=torch.float32).pin_memory()
        ctx.stream(host, h_tl)
        torch.cuda.synchronize()
        g = {"tlisi_out": h_tl.numpy().copy(), "cands": {}, "dims": (U, Ty, Tx)}
        c, n = ctx.detect(tau)
        g["cands"][tau] = (c.copy(), n)
        g["M"], g["mu"], g["sigma"] = ctx.get_stats()
        g["q"], g["tlisi"], g["raw"] = ctx.get_map(0), ctx.get_map(1), ctx.get_raw()
        # resident path on the same pixels
        ctx.tlisi(st)
        c2, n2 = ctx.detect(tau)
        assert np.array_equal(ctx.get_map(0), g["q"]) and n2 == n and np.array_equal(c2, c)
    del st
    torch.cuda.empty_cache()
    stack_np = [h.numpy() for h in host]
    oracle.set_threads(0)
    ref = oracle.run(stack_np, tile=32, tau=tau)
    check_against_oracle(None, g, ref, (tau,), 32, stack_np=stack_np)
    # the partial edge tiles (16 px wide / high) carry their own pixel count: compare them explicitly
    util.assert_map_close(g["q"][:, -1, :], ref.res.q[:, -1, :])
    util.assert_map_close(g["q"][:, :, -1], ref.res.q[:, :, -1])


def test_config5_imgfreq_full_size_channel_full_oracle():
    """BASELINE.json configs[4], one of the 16 channels (R19: channels are a batch) at full size, frequency branch."""
    cfg = synth.CONFIGS["imgfreq"]
    channel = 7
    st, truth = synth.make_stack(cfg, device=DEV, channel=channel)
    taus = (4.0, 6.0)
    g = gpu_run(st, taus=taus, branch=fitrig.BRANCH_FREQUENCY, want_tlisi=False)
    stack_np = [st[s].cpu().numpy() for s in range(cfg.L)]
    oracle.set_threads(0)
    ref = oracle.run(stack_np, tile=32, tau=6.0, branch=1)
    assert g["M"] == np.float32(ref.res.M)
    diff = _check_frequency(g, ref, taus, 32)
    assert len(diff) <= 0.001 * ref.kstar.size
