"""Pins for the CPU fp64 oracle -- CPU only.

Each test checks oracle/ against something that is NOT the oracle: hand-worked fixtures
(tests/golden), closed forms derived from Eq. 2-6, invariants the paper states, textbook
DFT values, or brute force on tiny inputs.
"""
import math

import numpy as np
import pytest

import oracle
import synth
from tests import util

RNG = np.random.default_rng(2509)


def _noise_stack(L, H, W, positive=False, scale=1.0):
    a = RNG.standard_normal((L, H, W)).astype(np.float32) * np.float32(scale)
    if positive:
        a = np.abs(a) + np.float32(0.05)
    return a


# ---------------------------------------------------------------- P2 + hand-worked fixtures
def _xy(argmax, W):
    return np.stack([argmax % W, argmax // W], axis=-1)


def test_p2_handworked_2x2_golden():
    g = util.golden("p2_handworked_2x2.json")
    st = np.array(g["snapshots"], dtype=np.float32)
    r = oracle.tlisi(st, tile=g["tile"], C=g["C"], ref_mode=g["ref_mode"])
    e = g["expect"]
    assert r.M == e["M"]
    assert np.array_equal(r.sumD, np.array(e["sumD"]))
    assert np.array_equal(r.maxD, np.array(e["maxD"]))
    assert np.array_equal(r.sumR, np.array(e["sumR"]))
    assert np.array_equal(_xy(r.argmax, 2), np.array(e["argmax_xy"]))
    assert np.array_equal(r.q, np.array(e["q"]))  # 45/1024, exact in binary
    assert np.array_equal(r.tlisi, np.array(e["tlisi"]))  # 0.9560546875


@pytest.mark.parametrize("mode,name", [(oracle.REF_ABS, "ABS"), (oracle.REF_LITERAL, "LITERAL"), (oracle.REF_FLOOR, "FLOOR")])
def test_handworked_2x3_three_reference_readings(mode, name):
    g = util.golden("handworked_2x3_modes.json")
    st = np.array(g["snapshots"], dtype=np.float32)
    r = oracle.tlisi(st, tile=g["tile"], C=g["C"], ref_mode=mode)
    e = g["expect"]
    assert r.M == e["M"]
    assert (r.U, r.Ty, r.Tx) == (2, 1, 2)  # partial tile of width 1 (R5)
    assert np.array_equal(r.sumD, np.array(e["sumD"]))
    assert np.array_equal(r.maxD, np.array(e["maxD"]))
    assert np.array_equal(_xy(r.argmax, 3), np.array(e["argmax_xy"]))
    np.testing.assert_allclose(r.sumR, np.array(e[name]["sumR"]), rtol=1e-15)
    np.testing.assert_allclose(r.q, np.array(e[name]["q"]), rtol=1e-15)
    np.testing.assert_allclose(r.tlisi, 1.0 - np.array(e[name]["q"]), rtol=1e-15)


def test_zscore_and_strict_threshold_golden():
    g = util.golden("zscore_handworked.json")
    v = np.array(g["values"], dtype=np.float64)[None, :]
    mu, sd, z = oracle.zscore(v)
    assert mu[0] == g["expect"]["mu"]
    assert abs(sd[0] ** 2 - g["expect"]["sigma_squared"]) < 1e-14
    np.testing.assert_allclose(z[0] * math.sqrt(10.0), g["expect"]["z_times_sqrt10"], atol=1e-14)
    arg = np.arange(5, dtype=np.int64)[None, :]
    c = oracle.select(z, arg, W=5, tau=1.5)
    assert c.n_found == 1 and list(c.tile) == g["expect"]["selected_at_tau_1.5"]
    c = oracle.select(z, arg, W=5, tau=float(z[0, 4]))  # strict '>' (R6): z == tau is not selected
    assert c.n_found == 0


# ---------------------------------------------------------------- P1
def test_p1_identical_snapshots_give_tlisi_one_and_no_candidates():
    one = _noise_stack(1, 64, 64)[0]
    st = np.stack([one] * 5)
    d = oracle.run(st, tile=16, tau=3.0)
    assert np.all(d.res.tlisi == 1.0) and np.all(d.res.q == 0.0)
    assert np.all(d.sigma == 0.0) and np.all(d.z == 0.0) and d.cands.n_found == 0  # R4


def test_p1_linear_in_time_gives_tlisi_one():
    a = (RNG.integers(-8, 9, (32, 32))).astype(np.float32)
    b = (RNG.integers(-4, 5, (32, 32))).astype(np.float32)
    st = np.stack([a + u * b for u in range(6)]).astype(np.float32)  # small integers: exact in fp32
    r = oracle.tlisi(st, tile=8)
    assert np.all(r.tlisi == 1.0)


# ---------------------------------------------------------------- P3
def test_p3_nonnegative_inputs_keep_every_factor_and_tlisi_in_unit_range():
    st = _noise_stack(6, 48, 40, positive=True, scale=3.0)
    for tile in (1, 4, 16, 32):
        r = oracle.tlisi(st, tile=tile)
        Ty, Tx = r.Ty, r.Tx
        n_t = np.zeros((Ty, Tx))
        for ty in range(Ty):
            for tx in range(Tx):
                n_t[ty, tx] = (min(48, (ty + 1) * tile) - ty * tile) * (min(40, (tx + 1) * tile) - tx * tile)
        assert np.all(r.sumD / n_t / r.M <= 1.0) and np.all(r.maxD / r.M <= 1.0) and np.all(r.sumR / n_t <= 1.0)
        assert np.all(r.tlisi >= 0.0) and np.all(r.tlisi <= 1.0)


# ---------------------------------------------------------------- P4
def test_p4_power_of_two_scaling_is_bit_exact():
    st = _noise_stack(5, 64, 64)
    r1 = oracle.tlisi(st, tile=16, C=1e-6)
    r2 = oracle.tlisi(st * np.float32(8.0), tile=16, C=8e-6)
    assert np.array_equal(r1.q, r2.q) and np.array_equal(r1.argmax, r2.argmax)
    assert np.array_equal(r1.sumR, r2.sumR) and np.array_equal(r1.sumD * 8.0, r2.sumD)


# ---------------------------------------------------------------- P5
def test_p5_time_reversal_maps_unit_u_to_L_minus_3_minus_u():
    st = _noise_stack(7, 32, 48)
    r1 = oracle.tlisi(st, tile=16)
    r2 = oracle.tlisi(st[::-1].copy(), tile=16)
    assert np.array_equal(r1.q, r2.q[::-1])
    assert np.array_equal(r1.argmax, r2.argmax[::-1])


# ---------------------------------------------------------------- P6
def test_p6_circular_shift_by_tile_multiples_permutes_tiles():
    st = _noise_stack(5, 64, 64)
    d1 = oracle.run(st, tile=16, tau=1.0)
    st2 = np.roll(st, shift=(16, 32), axis=(1, 2))
    d2 = oracle.run(st2, tile=16, tau=1.0)
    assert np.array_equal(np.roll(d1.res.q, shift=(1, 2), axis=(1, 2)), d2.res.q)
    np.testing.assert_allclose(d1.mu, d2.mu, rtol=1e-13)
    np.testing.assert_allclose(d1.sigma, d2.sigma, rtol=1e-12)
    np.testing.assert_allclose(np.roll(d1.z, shift=(1, 2), axis=(1, 2)), d2.z, rtol=1e-9, atol=1e-11)
    assert d1.cands.n_found == d2.cands.n_found


# ---------------------------------------------------------------- P7
def test_p7_zscore_invariants_and_independence_of_M():
    st = _noise_stack(6, 128, 128)
    da = oracle.run(st, tile=8, tau=3.0)
    n = da.z.shape[1] * da.z.shape[2]
    for u in range(da.z.shape[0]):
        assert abs(da.z[u].mean()) < 1e-12
        assert abs(da.z[u].std() - 1.0) < 1e-12
        assert da.z[u].max() <= math.sqrt(n - 1) + 1e-9
    db = oracle.run(st, tile=8, tau=3.0, M=123.456)  # M only scales q (Eq. 2), z must not move
    np.testing.assert_allclose(da.z, db.z, rtol=1e-9, atol=1e-11)
    assert list(da.cands.tile) == list(db.cands.tile) and list(da.cands.snapshot) == list(db.cands.snapshot)
    np.testing.assert_allclose(da.res.q * da.res.M ** 2, db.res.q * 123.456 ** 2, rtol=1e-13)


# ---------------------------------------------------------------- P8
@pytest.mark.parametrize("A,b", [(3.0, 4.0), (9.0, 2.0)])  # A/b < 1 and clamped at 1
def test_p8_single_pixel_transient_closed_form(A, b):
    L, H, W, tile, k = 7, 32, 32, 8, 3
    st = np.full((L, H, W), b, dtype=np.float32)
    py, px = 13, 21
    st[k, py, px] += np.float32(A)
    r = oracle.tlisi(st, tile=tile)
    assert r.M == b + A
    expect_q = A * A * min(A / b, 1.0) / ((tile * tile) ** 2 * (b + A) ** 2)
    ty, tx = py // tile, px // tile
    for u in range(L - 2):
        qt = r.q[u].copy()
        if u in (k - 2, k):  # R11: shows in units k-2 and k, cancels in k-1
            assert abs(qt[ty, tx] - expect_q) <= 1e-15 * expect_q
            assert r.sumD[u, ty, tx] == A and r.maxD[u, ty, tx] == A
            assert r.argmax[u, ty, tx] == py * W + px
            qt[ty, tx] = 0.0
        assert np.all(qt == 0.0)
    assert util.expected_active_units((k,), L) == [k - 2, k]


# ---------------------------------------------------------------- P9
def test_p9_tile_one_closed_form_per_pixel():
    st = _noise_stack(4, 16, 20)
    r = oracle.tlisi(st, tile=1)
    x = st.astype(np.float64)
    M = max(x.max(), 1e-6)
    for u in range(2):
        d = np.abs(np.abs(x[u + 1] - x[u]) - np.abs(x[u + 2] - x[u + 1]))
        xh = np.abs(x[u + 1])
        xh[xh == 0] = 1e-6
        np.testing.assert_allclose(r.q[u], d * d * np.minimum(d / xh, 1.0) / M ** 2, rtol=1e-14)
    assert np.array_equal(r.argmax[0], np.arange(16 * 20).reshape(16, 20))


# ---------------------------------------------------------------- P10
@pytest.mark.parametrize("H,W,tile", [(24, 24, 8), (19, 23, 8), (17, 9, 5), (33, 40, 32), (7, 7, 1)])
def test_p10_brute_force_mean_form(H, W, tile):
    st = _noise_stack(5, H, W)
    st[2, H // 2, W // 3] = 0.0  # exercise the x == 0 -> C branch of Eq. 5
    for mode in (oracle.REF_ABS, oracle.REF_LITERAL, oracle.REF_FLOOR):
        r = oracle.tlisi(st, tile=tile, ref_mode=mode)
        q, arg, parts, M = util.brute_force_tlisi(st, tile, ref_mode=mode)
        assert M == r.M
        np.testing.assert_allclose(r.q, q, rtol=1e-13, atol=1e-300)
        assert np.array_equal(r.argmax, arg)
        np.testing.assert_allclose(r.sumD, parts[0], rtol=1e-13)
        assert np.array_equal(r.maxD, parts[1])
        np.testing.assert_allclose(r.sumR, parts[2], rtol=1e-13)


@pytest.mark.parametrize("block_dim", [32, 64, 256])
def test_p10_alg1_index_route_sum_form(block_dim):
    st = _noise_stack(4, 32, 32)
    r = oracle.tlisi(st, tile=8)
    t3 = util.alg1_route_tlisi(st, 8, block_dim)  # Eq. 6 + Eq. 7 route
    np.testing.assert_allclose(r.tlisi, t3, rtol=1e-14)


def test_argmax_takes_first_of_equal_maxima():
    st = np.zeros((3, 4, 4), dtype=np.float32)
    st[2, 1, 2] = 5.0  # in the LAST snapshot of the unit, so only D^(s+1) holds it (R11)
    st[2, 3, 0] = 5.0
    st += 1.0
    r = oracle.tlisi(st, tile=4)
    assert r.argmax[0, 0, 0] == 1 * 4 + 2 and r.maxD[0, 0, 0] == 5.0


# ---------------------------------------------------------------- P11
def test_p11_adding_a_constant_changes_r_and_M_but_not_delta():
    L, H, W, tile, k, A, b, c = 5, 16, 16, 8, 2, 3.0, 4.0, 12.0
    st = np.full((L, H, W), b, dtype=np.float32)
    st[k, 5, 6] += np.float32(A)
    r1 = oracle.tlisi(st, tile=tile)
    r2 = oracle.tlisi(st + np.float32(c), tile=tile)
    assert np.array_equal(r1.sumD, r2.sumD) and np.array_equal(r1.maxD, r2.maxD)
    assert r2.M == r1.M + c
    # the reference of units k-2 and k is the (transient-free) neighbour snapshot: ratio A/b -> A/(b+c)
    assert r1.sumR[k - 2, 0, 0] == A / b and r2.sumR[k - 2, 0, 0] == A / (b + c)
    assert abs(r2.q[k, 0, 0] - A * A * (A / (b + c)) / (64 ** 2 * (b + c + A) ** 2)) < 1e-18


def test_global_max_is_signed_and_floored_at_C():
    st = -np.abs(_noise_stack(3, 8, 8)) - np.float32(1.0)
    assert oracle.global_max(st, C=1e-6) == 1e-6  # R2: signed maximum, then max(., C)
    st[1, 3, 3] = 0.25
    assert oracle.global_max(st) == 0.25
    # M is taken over ALL snapshots (R14), including ones whose only role is the last difference
    st2 = _noise_stack(4, 8, 8)
    st2[3, 0, 0] = 99.0
    assert oracle.tlisi(st2, tile=4).M == 99.0


# ---------------------------------------------------------------- P12
@pytest.mark.parametrize("U,k0", [(30, 4), (30, 15), (16, 3), (7, 2)])
def test_p12_dft_of_a_pure_tone(U, k0):
    A, c = 2.0, 0.7
    n = 6
    q = np.zeros((U, 2, 3))
    u = np.arange(U)
    q[:] = (c + A * np.cos(2 * np.pi * k0 * u / U + 0.3))[:, None, None]
    q[:, 1, 2] = c  # constant series -> eta = 0
    eta, ks = oracle.spectrum(q)
    expect = A * U if (U % 2 == 0 and k0 == U // 2) else A * U / 2
    if U % 2 == 0 and k0 == U // 2:
        expect *= abs(math.cos(0.3))  # at Nyquist only the cosine component survives
    assert abs(eta[0, 0] - expect) < 1e-9 * expect and ks[0, 0] == k0
    assert abs(eta[1, 2]) < 1e-12
    # against the library FFT (special case that reduces to a library routine)
    f = np.abs(np.fft.rfft(q[:, 0, 1] - q[:, 0, 1].mean()))
    assert abs(eta[0, 1] - f[1:U // 2 + 1].max()) < 1e-9


def test_spectrum_matches_numpy_rfft_on_random_series():
    U = 30
    q = np.abs(RNG.standard_normal((U, 4, 5))) * 1e-4
    eta, ks = oracle.spectrum(q)
    f = np.abs(np.fft.rfft(q - q.mean(axis=0, keepdims=True), axis=0))[1:U // 2 + 1]
    np.testing.assert_allclose(eta, f.max(axis=0), rtol=1e-10)
    assert np.array_equal(ks, f.argmax(axis=0) + 1)


def test_branch1_candidate_record_is_tile_centre_and_peak_bin():
    z = np.zeros((3, 3))
    z[2, 1] = 9.0
    ks = np.full((3, 3), 7, dtype=np.int32)
    c = oracle.select_spectrum(z, ks, H=70, W=80, tile=32, tau=6.0)  # last tile row has 6 rows (R18)
    assert c.n_found == 1 and (c.x[0], c.y[0], c.snapshot[0]) == (32 + 16, 64 + 3, 7)


# ---------------------------------------------------------------- P13 + behaviour the paper states
def test_p13_steady_sources_cancel_and_transient_is_recovered_at_its_pixel():
    cfg = synth.CONFIGS["tiny"]
    # noise-free steady sky: differences vanish identically -> tLISI = 1, no candidate
    st0, _ = synth.make_stack(cfg.replace(n_transients=0, transient_mode="none"), noise_sigma=0.0)
    d0 = oracle.run(st0.numpy(), tile=32, tau=3.0)
    assert np.all(d0.res.tlisi == 1.0) and d0.cands.n_found == 0
    # injected transient, strong enough for 64 tiles (SURVEY probe: 8 sigma is not, at N_T=32)
    st, truth = synth.make_stack(cfg.replace(transient_peak=40.0))
    t = truth.transients[0]
    d = oracle.run(st.numpy(), tile=32, tau=5.0)
    units = util.expected_active_units(t.active, cfg.L)
    assert units == [0, 2, 4]  # R11 for snapshots {2, 6}, L = 8
    got = {(int(u), int(x), int(y)) for u, x, y in zip(d.cands.snapshot, d.cands.x, d.cands.y)}
    for u in units:
        assert (u, t.x, t.y) in got
    assert all(u in units for (u, _, _) in got)  # steady sources and noise alone give no candidate at 5 sigma
    # low tLISI when exactly one difference image holds the transient, high otherwise
    ty, tx = t.y // 32, t.x // 32
    assert d.res.tlisi[units, ty, tx].max() < d.res.tlisi[[1, 3, 5], ty, tx].min()


def test_tiny_config_small_tiles_localise_the_8_sigma_transient():
    st, truth = synth.make_stack(synth.CONFIGS["tiny"])
    t = truth.transients[0]
    d = oracle.run(st.numpy(), tile=4, tau=4.5)  # this seed: z = 9.3, 11.9, 5.0 in units 0, 2, 4
    hits = [(int(u), int(x), int(y)) for u, x, y in zip(d.cands.snapshot, d.cands.x, d.cands.y)
            if abs(int(x) - t.x) <= 2 and abs(int(y) - t.y) <= 2]
    assert {h[0] for h in hits} >= {0, 2, 4}


def test_candidates_are_ordered_and_capacity_is_honoured():
    z = RNG.standard_normal((3, 4, 5))
    arg = np.arange(60, dtype=np.int64).reshape(3, 4, 5)
    c = oracle.select(z, arg, W=10, tau=0.0)
    keys = list(zip(c.snapshot.tolist(), c.tile.tolist()))
    assert keys == sorted(keys) and c.n_found == int((z > 0).sum())
    c2 = oracle.select(z, arg, W=10, tau=0.0, capacity=3)
    assert c2.n_found == c.n_found and len(c2.x) == 3 and list(c2.tile) == list(c.tile[:3])


def test_bad_arguments():
    with pytest.raises(ValueError):
        oracle.tlisi(_noise_stack(2, 8, 8), tile=4)  # R10: L < 3


# ------------------------------------------------------------------------------------------
# real-time form (R24): running maximum M_n, one unit per new snapshot
# ------------------------------------------------------------------------------------------
def test_realtime_running_maximum_closed_form_and_batch_equivalence():
    L, H, W = 7, 32, 48
    rng = np.random.default_rng(5)
    st = rng.normal(size=(L, H, W)).astype(np.float32)
    st = np.clip(st, -0.9, 0.9)
    peaks = [1.0, 4.0, 2.0, 3.0, 8.0, 5.0, 6.0]  # largest pixel of snapshot s
    for s, p in enumerate(peaks):
        st[s, 3 + s, 5] = p
    rt = oracle.run_realtime(st, tile=16, tau=1.0)
    batch = oracle.run(st, tile=16, tau=1.0)
    assert [r.res.M for r in rt] == [4.0, 4.0, 8.0, 8.0, 8.0]  # max of peaks[0 .. n+2], written out by hand
    assert rt[-1].res.M == batch.res.M
    for n, r in enumerate(rt):
        # q scales with 1/M^2 only (Eq. 2): q_n M_n^2 == q_batch M^2; z, hence the selection, is M-free (P7)
        np.testing.assert_allclose(r.res.q[0] * r.res.M ** 2, batch.res.q[n] * batch.res.M ** 2, rtol=1e-13)
        np.testing.assert_allclose(r.z[0], batch.z[n], rtol=1e-9, atol=1e-12)
        assert np.array_equal(r.res.argmax[0], batch.res.argmax[n])
        assert set(r.cands.snapshot.tolist()) <= {n}
    got = sorted((int(u), int(t)) for r in rt for u, t in zip(r.cands.snapshot, r.cands.tile))
    exp = sorted((int(u), int(t)) for u, t in zip(batch.cands.snapshot, batch.cands.tile))
    assert got == exp and len(exp) > 0


def test_realtime_single_pixel_transient_closed_form():
    # P8 with the running maximum: background b, one pixel +A in snapshot k only.  Unit k-2 (the transient is its
    # third snapshot) already sees M = b + A; units before it see M = b and have q = 0.
    L, H, W, tile, b, A, k = 8, 16, 16, 8, 4.0, 3.0, 4
    st = np.full((L, H, W), b, dtype=np.float32)
    st[k, 9, 2] += A
    rt = oracle.run_realtime(st, tile=tile, tau=0.5)
    n_t = tile * tile
    q_expected = A * A * min(A / b, 1.0) / (n_t ** 2 * (b + A) ** 2)
    for n, r in enumerate(rt):
        assert r.res.M == (b if n < k - 2 else b + A)
        q = r.res.q[0]
        if n in (k - 2, k):
            assert abs(q[1, 0] - q_expected) <= 1e-15 and np.count_nonzero(q) == 1
        else:
            assert not q.any()


# ------------------------------------------------------------------------------------------
# snapshot accumulation (section 3.3.2, Fig. 16; R25)
# ------------------------------------------------------------------------------------------
def test_accumulate_handworked_golden_and_incomplete_group_is_left_out():
    g = util.golden("accumulate_handworked_2x2.json")
    raw = np.array(g["raw"], dtype=np.float32)
    acc = oracle.accumulate(raw, g["g"])
    assert len(acc) == 3 and all(np.array_equal(a, np.array(e)) for a, e in zip(acc, g["accumulated"]))
    for stack in (raw, raw[:6]):  # the seventh snapshot completes no group
        r = oracle.tlisi(stack, tile=g["tile"], accumulate_g=g["g"])
        assert (r.U, r.Ty, r.Tx) == (1, 1, 1) and r.M == g["M"]
        assert r.sumD[0, 0, 0] == g["sumD"] and r.maxD[0, 0, 0] == g["maxD"] and r.sumR[0, 0, 0] == g["sumR"]
        assert r.q[0, 0, 0] == g["q"] and r.tlisi[0, 0, 0] == g["tlisi"]
        assert (int(r.argmax[0, 0, 0]) % 2, int(r.argmax[0, 0, 0]) // 2) == tuple(g["argmax_xy"])  # y*W + x, W = 2


def test_accumulate_one_is_the_identity_and_small_integers_match_the_presummed_stack():
    st = _noise_stack(9, 40, 56)
    a, b = oracle.run(st, tile=8, tau=2.0), oracle.run(st, tile=8, tau=2.0, accumulate_g=1)
    assert np.array_equal(a.res.q, b.res.q) and np.array_equal(a.z, b.z)
    # integer-valued pixels: fp32 sums are exact, so the fp32 route on the pre-summed stack is the same computation
    rng = np.random.default_rng(3)
    ints = rng.integers(-50, 50, size=(12, 24, 24)).astype(np.float32)
    pre = ints.reshape(4, 3, 24, 24).sum(axis=1).astype(np.float32)
    x, y = oracle.run(ints, tile=8, tau=1.0, accumulate_g=3), oracle.run(pre, tile=8, tau=1.0)
    assert x.res.M == y.res.M and np.array_equal(x.res.q, y.res.q) and np.array_equal(x.res.argmax, y.res.argmax)
    assert np.array_equal(x.cands.tile, y.cands.tile)
    with pytest.raises(ValueError):
        oracle.run(ints[:8], tile=8, accumulate_g=3)  # only two complete groups: fewer than 3 snapshots


@pytest.mark.parametrize("g", [2, 4])
def test_accumulate_single_pixel_transient_closed_form(g):
    # P8 on accumulated snapshots: background b in every raw snapshot, +A at one pixel of raw snapshot k only.
    # A_j = g*b everywhere, + A in group j* = k // g: units j*-2 and j* see Delta = A at that pixel against a
    # reference of g*b, and M = g*b + A.
    L, H, W, tile, b, A = 8 * g, 16, 16, 8, 2.0, 3.0
    k = 4 * g + 1
    st = np.full((L, H, W), b, dtype=np.float32)
    st[k, 3, 12] += A
    r = oracle.tlisi(st, tile=tile, accumulate_g=g)
    js = k // g
    assert r.U == 8 - 2 and r.M == g * b + A
    expected = A * A * min(A / (g * b), 1.0) / ((tile * tile) ** 2 * (g * b + A) ** 2)
    for u in range(r.U):
        if u in (js - 2, js):
            assert abs(r.q[u, 0, 1] - expected) <= 1e-15 and np.count_nonzero(r.q[u]) == 1
        else:
            assert not r.q[u].any()


# ------------------------------------------------------------------------------------------
# harmonic summing as the spectral refinement h of Eq. 10 (R26)
# ------------------------------------------------------------------------------------------
def test_harmonic_sum_one_harmonic_is_the_maximum_magnitude():
    rng = np.random.default_rng(8)
    q = rng.random((30, 5, 7))
    e1, k1 = oracle.spectrum(q)
    eh, kh = oracle.spectrum_hsum(q, 1)
    assert np.array_equal(e1, eh) and np.array_equal(k1, kh)


@pytest.mark.parametrize("U,k0,amps", [(64, 3, (2.0, 1.0, 0.0, 0.5)), (30, 2, (1.0, 1.0, 0.0, 1.0)), (48, 5, (3.0, 0.0, 0.0, 0.0))])
def test_harmonic_sum_closed_form_comb(U, k0, amps):
    # q_u = c + sum_j A_j cos(2 pi j k0 u / U), j = 1..4, all j*k0 below Nyquist: m_{j k0} = A_j U / 2 exactly,
    # every other bin is 0, so s_h(k0) = (U/2) (A_1 + .. + A_h) / sqrt(h) and eta is the largest of h = 1, 2, 4
    u = np.arange(U)
    series = 0.7 + sum(A * np.cos(2 * np.pi * (j + 1) * k0 * u / U) for j, A in enumerate(amps))
    q = series.reshape(U, 1, 1)
    eta, ks, mag = oracle.spectrum_hsum(q, 4, want_mag=True)
    for j, A in enumerate(amps):
        assert abs(mag[(j + 1) * k0 - 1, 0, 0] - A * U / 2) <= 1e-9 * U
    cand = [(U / 2) * sum(amps[:h]) / np.sqrt(h) for h in (1, 2, 4)]
    assert abs(eta[0, 0] - max(cand)) <= 1e-9 * U and ks[0, 0] == k0
    # with one harmonic only the strongest single line counts
    e1, k1 = oracle.spectrum_hsum(q, 1)
    jbest = int(np.argmax(amps))
    assert abs(e1[0, 0] - amps[jbest] * U / 2) <= 1e-9 * U and k1[0, 0] == (jbest + 1) * k0


def test_harmonic_sum_brute_force_against_numpy_rfft():
    rng = np.random.default_rng(21)
    U, H = 40, 8
    q = rng.random((U, 3, 4))
    eta, ks = oracle.spectrum_hsum(q, H)
    m = np.abs(np.fft.rfft(q - q.mean(axis=0), axis=0))  # bins 0..U/2
    K = U // 2
    for idx in np.ndindex(3, 4):
        best, kb = -1.0, 0
        for k in range(1, K + 1):
            h = 1
            while h <= H and h * k <= K:
                s = m[(slice(k, h * k + 1, k),) + idx].sum() / np.sqrt(h)
                if s > best * (1 + 1e-12):
                    best, kb = s, k
                h *= 2
        assert abs(eta[idx] - best) <= 1e-10 * best and ks[idx] == kb


# ------------------------------------------------------------------------------------------
# overlapping windows (an extension; R27)
# ------------------------------------------------------------------------------------------
def test_windows_with_full_stride_are_the_tiles_and_aligned_windows_are_tile_values():
    st = _noise_stack(6, 80, 112)
    a, b = oracle.tlisi(st, tile=16), oracle.tlisi_windows(st, 16, 16)
    assert np.array_equal(a.q, b.q) and np.array_equal(a.argmax, b.argmax)
    w = oracle.tlisi_windows(st, 16, 4, M=a.M)
    assert w.q.shape == (4, 80 // 4 - 3, 112 // 4 - 3)
    # the windows that start on a tile boundary ARE the tiles
    assert np.array_equal(w.q[:, ::4, ::4], a.q) and np.array_equal(w.argmax[:, ::4, ::4], a.argmax)


@pytest.mark.parametrize("H,W,tile,stride", [(37, 50, 8, 4), (33, 20, 16, 8), (10, 70, 16, 4), (64, 64, 32, 16)])
def test_windows_brute_force(H, W, tile, stride):
    st = _noise_stack(5, H, W)
    r = oracle.tlisi_windows(st, tile, stride)
    x = st.astype(np.float64)
    M = max(x.max(), 1e-6)
    cy, cx = -(-H // stride), -(-W // stride)
    Ty, Tx = max(1, cy - tile // stride + 1), max(1, cx - tile // stride + 1)
    assert r.q.shape == (3, Ty, Tx)
    for u in range(3):
        delta = np.abs(np.abs(x[u + 1] - x[u]) - np.abs(x[u + 2] - x[u + 1]))
        ref = np.abs(x[u + 1])
        rr = np.minimum(delta / np.where(ref == 0, 1e-6, ref), 1.0)
        for ty in range(Ty):
            for tx in range(Tx):
                d = delta[ty * stride:ty * stride + tile, tx * stride:tx * stride + tile]
                q = d.mean() * d.max() * rr[ty * stride:ty * stride + tile, tx * stride:tx * stride + tile].mean() / M ** 2
                assert abs(r.q[u, ty, tx] - q) <= 1e-13 * q
                iy, ix = np.unravel_index(np.argmax(d), d.shape)  # first maximum in row-major order
                assert r.argmax[u, ty, tx] == (ty * stride + iy) * W + tx * stride + ix
