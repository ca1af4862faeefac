"""Pins of the oracle's accumulation rule (reading R30: "combined progressively until there is enough
difference between adjacent accumulated snapshots").  CPU only.  The rule is a reading (the paper defines neither the
measure nor the threshold), so the pins fix what mathematics fixes about the measure as defined -- closed forms,
invariances, a brute force in plain python -- and the progressive search."""
import math

import numpy as np
import pytest

import oracle


def _ramp(L, H, W, a, b):
    """x_s = a + b s in every pixel."""
    return [np.full((H, W), a + b * s, dtype=np.float32) for s in range(L)]


def test_identical_snapshots_have_no_contrast_and_take_the_largest_admissible_group():
    st = [np.full((8, 8), 3.0, dtype=np.float32)] * 24
    for g in (1, 2, 4, 8):
        assert oracle.accumulation_contrast(st, g) == 0.0
    g, levels = oracle.choose_accumulate(st, 1e-3, g_max=32)
    assert g == 8 and [lv[0] for lv in levels] == [1, 2, 4, 8]  # 24 // 16 < 3: g = 16 is not admissible
    assert oracle.choose_accumulate(st, 1e-3, g_max=2)[0] == 2


@pytest.mark.parametrize("g", [1, 2, 4])
def test_linear_drift_closed_form(g):
    """x_s = a + b s (a, b > 0): A_j = g a + b (g^2 j + g (g - 1) / 2), so |A_{j+1} - A_j| = b g^2 everywhere and
    mean |A_j| = g a + b (g^2 (J - 1) / 2 + g (g - 1) / 2)."""
    L, a, b = 32, 4.0, 0.125
    J = L // g
    want = b * g * g / (g * a + b * (g * g * (J - 1) / 2 + g * (g - 1) / 2))
    assert oracle.accumulation_contrast(_ramp(L, 4, 6, a, b), g) == pytest.approx(want, rel=1e-12)


def test_alternating_signal_cancels_under_pairwise_accumulation():
    """x_s = c + (-1)^s e: adjacent snapshots differ by 2 e, adjacent PAIR sums are identical."""
    c, e = 5.0, 0.5
    st = [np.full((4, 4), c + (e if s % 2 == 0 else -e), dtype=np.float32) for s in range(16)]
    assert oracle.accumulation_contrast(st, 1) == pytest.approx(2 * e / c, rel=1e-12)
    assert oracle.accumulation_contrast(st, 2) == 0.0
    assert oracle.choose_accumulate(st, 0.1)[0] == 1        # 0.2 >= 0.1 at once
    g, levels = oracle.choose_accumulate(st, 0.3)            # never reached: the largest admissible level
    assert g == 4 and [lv[0] for lv in levels] == [1, 2, 4]


def test_progressive_search_stops_at_the_first_level_that_reaches_eps():
    L, a, b = 48, 10.0, 0.01
    st = _ramp(L, 4, 4, a, b)
    d = {g: oracle.accumulation_contrast(st, g) for g in (1, 2, 4, 8, 16)}
    assert d[1] < d[2] < d[4] < d[8] < d[16]  # a slow drift becomes visible as snapshots are combined
    for g_want in (2, 4, 8):
        eps = 0.5 * (d[g_want // 2] + d[g_want])
        g, levels = oracle.choose_accumulate(st, eps)
        assert g == g_want and levels[-1] == (g_want, d[g_want]) and len(levels) == int(math.log2(g_want)) + 1
    assert oracle.choose_accumulate(st, d[1])[0] == 1  # ">=": reaching eps exactly is enough


def test_brute_force_and_scale_invariance():
    rng = np.random.default_rng(7)
    L, H, W, g = 13, 5, 7, 3
    st = [rng.normal(2.0, 1.0, (H, W)).astype(np.float32) for _ in range(L)]
    J = L // g
    A = [[[sum(float(st[g * j + i][y, x]) for i in range(g)) for x in range(W)] for y in range(H)] for j in range(J)]
    num = sum(abs(A[j + 1][y][x] - A[j][y][x]) for j in range(J - 1) for y in range(H) for x in range(W)) / ((J - 1) * H * W)
    den = sum(abs(A[j][y][x]) for j in range(J) for y in range(H) for x in range(W)) / (J * H * W)
    assert oracle.accumulation_contrast(st, g) == pytest.approx(num / den, rel=1e-12)
    # a power-of-two scale changes nothing (every operation is exact under it); the trailing L mod g snapshots are left out (R25)
    assert oracle.accumulation_contrast([4.0 * x for x in st], g) == oracle.accumulation_contrast(st, g)
    assert oracle.accumulation_contrast(st[:J * g], g) == oracle.accumulation_contrast(st, g)
    # a transient in one snapshot raises the contrast; an all-zero stack has none
    st2 = [x.copy() for x in st]
    st2[4][2, 3] += 50.0
    assert oracle.accumulation_contrast(st2, g) > oracle.accumulation_contrast(st, g)
    assert oracle.accumulation_contrast([np.zeros((H, W), np.float32)] * 6, 1) == 0.0


def test_bad_arguments():
    st = _ramp(5, 2, 2, 1.0, 1.0)
    with pytest.raises(ValueError):
        oracle.accumulation_contrast(st, 4)  # one accumulated snapshot only
    with pytest.raises(ValueError):
        oracle.choose_accumulate(st[:2], 0.1)
    assert oracle.choose_accumulate(st, 1e9)[0] == 1  # 5 // 2 < 3: only g = 1 is admissible
